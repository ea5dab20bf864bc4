"""Seeded synthetic workloads (BASELINE.json configs C1..C5; recipe in DESIGN.md §4).

This module is the ONLY code shared by the CPU oracle's tests and the CUDA path's
tests/bench.  It holds none of the method's arithmetic: it draws smooth-field-plus-noise
Q/K/V tensors with the shapes of the paper's workloads (n = 75,600 and
118,800 tokens; l.65: 128-d head features, spatio-temporally smooth) and names the
hyper-parameters of each config.  Nothing here imports `oracle/` or the CUDA binding.

Every (config seed, head) draws from its own `numpy.random.default_rng([seed, head, step])`
stream, so one head can be generated without the others (the oracle checks sampled heads at
the full-size configs).
"""
from __future__ import annotations

import dataclasses
import math
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import torch


@dataclasses.dataclass(frozen=True)
class Workload:
    """Problem statement of one attention call (Alg. 2 inputs l.349)."""
    name: str
    B: int
    heads: int
    D: int
    dtype: str                 # "f32" | "bf16"
    T: int
    H: int
    W: int
    cell: tuple                # (k_t, k_h, k_w) for both Q and K
    win: tuple                 # (w_t, w_h, w_w)
    iters: int
    tile: tuple                # (tau_q, tau_k)
    top_p: float
    merge_rounds: int
    seed: int
    noise: float = 0.3
    logit_std: float = 2.0     # target std of q.k/sqrt(D) (0 = no rescale)

    @property
    def n(self) -> int:
        return self.T * self.H * self.W

    @property
    def grid(self) -> tuple:
        return tuple(-(-d // k) for d, k in zip((self.T, self.H, self.W), self.cell))

    @property
    def n_clusters(self) -> int:
        g = self.grid
        return g[0] * g[1] * g[2]

    def torch_dtype(self):
        return torch.float32 if self.dtype == "f32" else torch.bfloat16


# BASELINE.json configs[0..4]; R = 3 merge rounds is PAPER.md l.322.
C1 = Workload("C1-tiny", 1, 2, 64, "f32", 4, 8, 8, (2, 4, 4), (3, 3, 3), 3, (64, 64), 0.9, 3, seed=0)
C2 = Workload("C2-mid", 1, 8, 128, "bf16", 9, 24, 32, (3, 4, 4), (3, 3, 3), 3, (128, 128), 0.9, 3, seed=1)
C3 = Workload("C3-wan", 1, 40, 128, "bf16", 21, 45, 80, (3, 5, 8), (3, 3, 3), 3, (128, 128), 0.9, 3, seed=2)
C4 = Workload("C4-hunyuan", 1, 24, 128, "bf16", 33, 45, 80, (3, 5, 8), (3, 3, 3), 3, (128, 128), 0.9, 3, seed=3)
C5 = dataclasses.replace(C4, name="C5-hybrid", seed=4)
CONFIGS = {"C1": C1, "C2": C2, "C3": C3, "C4": C4, "C5": C5}


def _field(rng: np.random.Generator, wl: Workload) -> np.ndarray:
    """Smooth field F[t,h,w,:] = sum of 8 3-D sinusoids, frequencies U[0,0.25] cycles per
    clustering cell per axis, random phases, N(0,1) amplitude vectors (BASELINE.json C1)."""
    M = 8
    f = rng.uniform(0.0, 0.25, size=(M, 3))
    phi = rng.uniform(0.0, 2.0 * math.pi, size=M)
    A = rng.standard_normal((M, wl.D))
    t = np.arange(wl.T, dtype=np.float64)[:, None, None] / wl.cell[0]
    h = np.arange(wl.H, dtype=np.float64)[None, :, None] / wl.cell[1]
    w = np.arange(wl.W, dtype=np.float64)[None, None, :] / wl.cell[2]
    F = np.zeros((wl.n, wl.D), dtype=np.float32)
    for m in range(M):
        ph = 2.0 * math.pi * (f[m, 0] * t + f[m, 1] * h + f[m, 2] * w) + phi[m]
        F += np.sin(ph).reshape(-1, 1).astype(np.float32) * A[m].astype(np.float32)[None, :]
    return F


def _draw_head(wl: Workload, head: int, step: int = 0) -> np.ndarray:
    """One head's (Q, K, V) in fp32, shape [3, n, D]: shared field F, per-tensor random
    D x D projection (variance preserving) plus `noise` * N(0,1), then Q and K scaled so
    that q.k/sqrt(D) has std ~ logit_std over a fixed sample of 8192 token pairs."""
    rng = np.random.default_rng([wl.seed, head, step])
    F = _field(rng, wl)
    out = np.empty((3, wl.n, wl.D), dtype=np.float32)
    for i in range(3):
        P = (rng.standard_normal((wl.D, wl.D)) / math.sqrt(wl.D)).astype(np.float32)
        eps = rng.standard_normal((wl.n, wl.D), dtype=np.float32)
        out[i] = F @ P + np.float32(wl.noise) * eps
    if wl.logit_std > 0:
        ia = rng.integers(0, wl.n, size=8192)
        ib = rng.integers(0, wl.n, size=8192)
        lg = np.einsum("ij,ij->i", out[0][ia].astype(np.float64), out[1][ib].astype(np.float64))
        sd = float(np.std(lg / math.sqrt(wl.D)))
        s = np.float32(math.sqrt(wl.logit_std / max(sd, 1e-12)))
        out[0] *= s
        out[1] *= s
    return out


def make_head(wl: Workload, head: int, step: int = 0) -> torch.Tensor:
    """[3, n, D] tensor (Q, K, V of one head) in the workload's I/O dtype.  Values are
    generated in fp32 and rounded ONCE (RNE) to bf16 when dtype == 'bf16'; that tensor is
    the input of both the oracle and the CUDA path."""
    x = torch.from_numpy(_draw_head(wl, head, step))
    return x.to(wl.torch_dtype())


def make_qkv(wl: Workload, heads=None, step: int = 0, threads: int = 8):
    """(Q, K, V), each [B=1, len(heads), n, D] CPU tensors in the I/O dtype."""
    assert wl.B == 1
    heads = list(range(wl.heads)) if heads is None else list(heads)
    out = torch.empty((3, 1, len(heads), wl.n, wl.D), dtype=wl.torch_dtype())

    def job(i):
        out[:, 0, i] = make_head(wl, heads[i], step)

    with ThreadPoolExecutor(max_workers=max(1, min(threads, len(heads)))) as ex:
        list(ex.map(job, range(len(heads))))
    return out[0], out[1], out[2]


def hybrid_next(wl: Workload, prev: torch.Tensor, head: int, step: int, rms0: torch.Tensor) -> torch.Tensor:
    """C5 dynamics: X_s = 0.98 X_{s-1} + 0.2 fresh_s, fresh_s a new generator draw
    normalised to the RMS of X_0 per tensor (BASELINE.json configs[4]).  `prev` and the
    result are [3, n, D] in the I/O dtype; arithmetic in fp32, rounded once."""
    fresh = torch.from_numpy(_draw_head(wl, head, step))
    rms = fresh.pow(2).mean(dim=(1, 2), keepdim=True).sqrt()
    fresh = fresh * (rms0.view(3, 1, 1) / rms)
    return (0.98 * prev.float() + 0.2 * fresh).to(wl.torch_dtype())


def to_f64(x: torch.Tensor) -> np.ndarray:
    """Exact widening of an fp32/bf16 tensor to a float64 numpy array (oracle input)."""
    return x.detach().cpu().to(torch.float64).numpy()
