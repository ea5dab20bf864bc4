"""Thin ctypes binding of libhva.so (include/hva.h).  Argument marshalling only: every step of
the path runs in the CUDA kernels behind the C ABI.  PyTorch is used for device memory and the
current stream.  There is no CPU fallback: importing works without a GPU (symbols load), any
compute call without a CUDA device raises."""
from __future__ import annotations

import ctypes as C
import math
import os

import torch

from .inputs import Workload

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhva.so")

HVA_F32, HVA_BF16 = 0, 1
HVA_ANCHOR, HVA_INTERMEDIATE, HVA_DENSE = 0, 1, 2
HVA_FLAG_CLUSTER_SIMT, HVA_FLAG_ATTN_SIMT, HVA_FLAG_MASK_BLOCKSORT, HVA_FLAG_MERGE_SIMT, HVA_FLAG_Q_UNPERMUTED = 1, 2, 4, 8, 16

EXPORTS = ["hva_strerror", "hva_version", "hva_num_clusters", "hva_workspace_bytes", "hva_state_bytes", "hva_state_describe", "hva_workspace_describe",
           "hva_cluster_workspace_bytes", "hva_cluster_update_workspace_bytes", "hva_merge_workspace_bytes", "hva_plan_workspace_bytes",
           "hva_plan_describe", "hva_cluster", "hva_cluster_ex", "hva_cluster_qk", "hva_select_subset", "hva_cluster_update", "hva_cluster_update_ex",
           "hva_build_mask", "hva_build_mask_ex", "hva_merge", "hva_merge_ex", "hva_build_plan", "hva_build_plan_static",
           "hva_build_plan_static_limit", "hva_permute", "hva_unpermute",
           "hva_sparse_attention", "hva_forward", "hva_forward_host"]


class hva_shape(C.Structure):
    _fields_ = [(k, C.c_int32) for k in ("B", "heads", "T", "H", "W", "D", "dtype")]


class hva_config(C.Structure):
    _fields_ = [("cell_q", C.c_int32 * 3), ("cell_k", C.c_int32 * 3), ("win_q", C.c_int32 * 3), ("win_k", C.c_int32 * 3),
                ("iters", C.c_int32), ("tile_q", C.c_int32), ("tile_k", C.c_int32), ("top_p", C.c_float),
                ("min_kc", C.c_float), ("merge_rounds", C.c_int32), ("max_q_tiles", C.c_int32), ("seed", C.c_uint32),
                ("subset_frac", C.c_float), ("hybrid_refresh_all", C.c_int32), ("softmax_scale", C.c_float),
                ("flags", C.c_uint32)]


class hva_stats(C.Structure):
    _fields_ = [("n_groups", C.c_int32), ("q_tiles", C.c_int32), ("q_rows_valid", C.c_int64),
                ("q_rows_padded", C.c_int64), ("k_cols_valid", C.c_int64), ("k_cols_padded", C.c_int64),
                ("tiles_executed", C.c_int64), ("pairs_valid", C.c_int64)]


class hva_plan_layout(C.Structure):
    _fields_ = [(k, C.c_size_t) for k in ("perm_q", "inv_perm_q", "perm_k", "koff", "n_groups", "gid", "goff", "kappa",
                                          "run_cnt", "runs", "run_stride", "work_cnt", "work", "work_cap", "stats", "total")]


class hva_state_layout(C.Structure):
    _fields_ = [(k, C.c_size_t * 2) for k in ("assign", "mu", "sums", "sizes", "subset")] + \
               [("n_clusters", C.c_int32 * 2), ("m", C.c_int32), ("total", C.c_size_t)]


class hva_workspace_layout(C.Structure):
    _fields_ = [(k, C.c_size_t) for k in ("lowe", "mask", "group_of", "n_groups", "group_mask", "plan", "plan_bytes", "qp", "kp",
                                          "vp", "scratch", "state", "total")]


_lib = None


def lib():
    """Loads libhva.so (raises if it has not been built: `python -m paper_2607_03012_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} missing: build it with `python paper_2607_03012_b200/build.py`")
        L = C.CDLL(LIB_PATH)
        L.hva_strerror.restype = C.c_char_p
        L.hva_workspace_bytes.restype = C.c_size_t
        L.hva_state_bytes.restype = C.c_size_t
        L.hva_cluster_workspace_bytes.restype = C.c_size_t
        L.hva_cluster_update_workspace_bytes.restype = C.c_size_t
        L.hva_merge_workspace_bytes.restype = C.c_size_t
        L.hva_plan_workspace_bytes.restype = C.c_size_t
        L.hva_build_plan_static_limit.restype = C.c_size_t
        _lib = L
    return _lib


class HvaError(RuntimeError):
    pass


def _check(rc):
    if rc != 0:
        raise HvaError(f"hva error {rc}: {lib().hva_strerror(rc).decode()}")


def _p(t):
    if t is None:
        return C.c_void_p(0)
    assert t.is_contiguous()
    return C.c_void_p(t.data_ptr())


def _stream():
    if not torch.cuda.is_available():
        raise HvaError("no CUDA device: the hva path has no CPU fallback")
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _i3(v):
    return (C.c_int32 * 3)(*[int(x) for x in v])


def make_shape(wl_or_dims, heads=None, dtype=None) -> hva_shape:
    if isinstance(wl_or_dims, Workload):
        w = wl_or_dims
        return hva_shape(w.B, w.heads if heads is None else heads, w.T, w.H, w.W, w.D,
                         HVA_F32 if w.dtype == "f32" else HVA_BF16)
    B, h, T, H, W, D = wl_or_dims
    return hva_shape(B, h, T, H, W, D, HVA_F32 if dtype in ("f32", torch.float32) else HVA_BF16)


def make_config(wl: Workload, top_p=None, merge_rounds=None, subset_frac=0.0, refresh_all=0, min_kc=0.0,
                max_q_tiles=0, flags=0) -> hva_config:
    c = hva_config()
    c.cell_q = _i3(wl.cell); c.cell_k = _i3(wl.cell); c.win_q = _i3(wl.win); c.win_k = _i3(wl.win)
    c.iters = wl.iters; c.tile_q, c.tile_k = wl.tile
    c.top_p = wl.top_p if top_p is None else top_p
    c.min_kc = min_kc
    c.merge_rounds = wl.merge_rounds if merge_rounds is None else merge_rounds
    c.max_q_tiles = max_q_tiles; c.seed = wl.seed; c.subset_frac = subset_frac
    c.hybrid_refresh_all = refresh_all; c.softmax_scale = 0.0; c.flags = flags
    return c


def _ws(nbytes, device="cuda"):
    return torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device)


def hva_num_clusters(shape, cell):
    return lib().hva_num_clusters(C.byref(shape), _i3(cell))


def hva_workspace_bytes(shape, cfg):
    return lib().hva_workspace_bytes(C.byref(shape), C.byref(cfg))


def hva_state_bytes(shape, cfg):
    return lib().hva_state_bytes(C.byref(shape), C.byref(cfg))


def hva_plan_describe(BH, n, Nq, Nk, tile_q) -> hva_plan_layout:
    L = hva_plan_layout()
    _check(lib().hva_plan_describe(BH, n, Nq, Nk, tile_q, C.byref(L)))
    return L


def hva_cluster(shape, cell, win, iters, X, mu_init=None, want_sums=True, want_lowe=True, flags=0, probe=None):
    """-> dict(assign [BH,n] i32, mu [BH,Nc,D] f32, sizes [BH,Nc] i32, sums, lowe).  flags / probe: hva_cluster_ex."""
    BH, n, D = shape.B * shape.heads, shape.T * shape.H * shape.W, shape.D
    Nc = hva_num_clusters(shape, cell)
    K = [-(-d // k) for d, k in zip((shape.T, shape.H, shape.W), cell)]
    nwin = math.prod(min(w, k) for w, k in zip(win, K))
    dev = X.device
    out = dict(assign=torch.empty((BH, n), dtype=torch.int32, device=dev),
               mu=torch.empty((BH, Nc, D), dtype=torch.float32, device=dev),
               sizes=torch.empty((BH, Nc), dtype=torch.int32, device=dev),
               sums=torch.empty((BH, Nc, D), dtype=torch.float32, device=dev) if want_sums else None,
               lowe=torch.empty((BH, n), dtype=torch.float32, device=dev) if want_lowe else None)
    ws = _ws(lib().hva_cluster_workspace_bytes(C.byref(shape), _i3(cell), _i3(win)), dev)
    if flags or probe is not None:
        _check(lib().hva_cluster_ex(C.byref(shape), _i3(cell), _i3(win), int(iters), _p(X), _p(mu_init), _p(out["assign"]),
                                    _p(out["mu"]), _p(out["sizes"]), _p(out["sums"]), _p(out["lowe"]), C.c_uint32(flags),
                                    _p(probe), _p(ws), C.c_size_t(ws.numel()), _stream()))
    else:
        _check(lib().hva_cluster(C.byref(shape), _i3(cell), _i3(win), int(iters), _p(X), _p(mu_init), _p(out["assign"]),
                                 _p(out["mu"]), _p(out["sizes"]), _p(out["sums"]), _p(out["lowe"]), _p(ws),
                                 C.c_size_t(ws.numel()), _stream()))
    return out


def hva_cluster_qk(shape, cfg, Q, K, want_sums=True, bufs=None):
    """Q and K clustered by one call on two streams (hva.h) -> (dict_q, dict_k) as hva_cluster (no lowe).  `bufs`: the tuple a
    previous call returned as its third value, to reuse outputs and scratch."""
    BH, n, D = shape.B * shape.heads, shape.T * shape.H * shape.W, shape.D
    dev = Q.device
    if bufs is None:
        outs = []
        for cell, win in ((list(cfg.cell_q), list(cfg.win_q)), (list(cfg.cell_k), list(cfg.win_k))):
            Nc = hva_num_clusters(shape, cell)
            outs.append(dict(assign=torch.empty((BH, n), dtype=torch.int32, device=dev),
                             mu=torch.empty((BH, Nc, D), dtype=torch.float32, device=dev),
                             sizes=torch.empty((BH, Nc), dtype=torch.int32, device=dev),
                             sums=torch.empty((BH, Nc, D), dtype=torch.float32, device=dev) if want_sums else None, lowe=None,
                             ws=_ws(lib().hva_cluster_workspace_bytes(C.byref(shape), _i3(cell), _i3(win)), dev)))
        bufs = tuple(outs)
    q, k = bufs
    _check(lib().hva_cluster_qk(C.byref(shape), C.byref(cfg), _p(Q), _p(K), _p(q["assign"]), _p(q["mu"]), _p(q["sizes"]), _p(q["sums"]),
                                _p(k["assign"]), _p(k["mu"]), _p(k["sizes"]), _p(k["sums"]), _p(q["ws"]), C.c_size_t(q["ws"].numel()),
                                _p(k["ws"]), C.c_size_t(k["ws"].numel()), _stream()))
    return q, k, bufs


def hva_select_subset(lowe, m):
    BH, n = lowe.shape
    subset = torch.empty((BH, m), dtype=torch.int32, device=lowe.device)
    _check(lib().hva_select_subset(BH, n, _p(lowe), int(m), _p(subset), C.c_void_p(0), C.c_size_t(0), _stream()))
    return subset


def hva_cluster_update(shape, X, subset, assign, mu, sums, sizes, refresh_all=0, flags=0):
    """In place on assign / mu / sums / sizes."""
    BH, m = subset.shape
    ws = _ws(lib().hva_cluster_update_workspace_bytes(C.byref(shape), int(mu.shape[1]), int(m)), X.device)
    _check(lib().hva_cluster_update_ex(C.byref(shape), mu.shape[1], _p(X), _p(subset), int(m), int(refresh_all), _p(assign),
                                       _p(mu), _p(sums), _p(sizes), C.c_uint32(flags), _p(ws), C.c_size_t(ws.numel()), _stream()))


def hva_build_mask(mu_q, mu_k, sizes_k, scale, top_p, min_kc=0.0, flags=0):
    BH, Nq, D = mu_q.shape
    Nk = mu_k.shape[1]
    mask = torch.empty((BH, Nq, Nk), dtype=torch.uint8, device=mu_q.device)
    _check(lib().hva_build_mask_ex(BH, Nq, Nk, D, _p(mu_q), _p(mu_k), _p(sizes_k), C.c_float(scale), C.c_float(top_p),
                                   C.c_float(min_kc), _p(mask), C.c_uint32(flags), C.c_void_p(0), C.c_size_t(0), _stream()))
    return mask


def hva_merge(sizes_q, sizes_k, mask, tile_q, tile_k, rounds, seed=0, max_q_tiles=0, flags=0):
    BH, Nq, Nk = mask.shape
    dev = mask.device
    group_of = torch.empty((BH, Nq), dtype=torch.int32, device=dev)
    n_groups = torch.empty((BH,), dtype=torch.int32, device=dev)
    gmask = torch.empty((BH, Nq, Nk), dtype=torch.uint8, device=dev)
    ws = _ws(lib().hva_merge_workspace_bytes(BH, Nq, Nk), dev)
    _check(lib().hva_merge_ex(BH, Nq, Nk, _p(sizes_q), _p(sizes_k), _p(mask), int(tile_q), int(tile_k), int(rounds),
                              int(max_q_tiles), C.c_uint32(seed), _p(group_of), _p(n_groups), _p(gmask), C.c_uint32(flags), _p(ws),
                              C.c_size_t(ws.numel()), _stream()))
    return group_of, n_groups, gmask


class Plan:
    """Opaque device plan buffer + typed views of its arrays."""

    def __init__(self, buf, L, BH, n, Nq, Nk):
        self.buf, self.L, self.BH, self.n, self.Nq, self.Nk = buf, L, BH, n, Nq, Nk

    def _view(self, off, shape, dtype=torch.int32):
        nb = int(math.prod(shape)) * torch.empty((), dtype=dtype).element_size()
        return self.buf[off:off + nb].view(dtype).view(*shape)

    def __getattr__(self, k):
        L, BH, n, Nq, Nk = self.L, self.BH, self.n, self.Nq, self.Nk
        shapes = dict(perm_q=(BH, n), inv_perm_q=(BH, n), perm_k=(BH, n), koff=(BH, Nk + 1), n_groups=(BH,),
                      gid=(BH, Nq), goff=(BH, Nq + 1), kappa=(BH, Nq), run_cnt=(BH, Nq),
                      runs=(BH, Nq, L.run_stride), work_cnt=(BH,), work=(BH, L.work_cap))
        if k in shapes:
            return self._view(getattr(L, k), shapes[k])
        if k == "stats":
            return self._view(L.stats, (BH, 7), torch.int64)   # hva_stats = 2 x int32 + 6 x int64 = 7 words
        raise AttributeError(k)

    def stats_dicts(self):
        raw = self.stats.cpu().numpy()
        out = []
        for r in raw:
            out.append(dict(n_groups=int(r[0] & 0xffffffff), q_tiles=int(r[0] >> 32), q_rows_valid=int(r[1]),
                            q_rows_padded=int(r[2]), k_cols_valid=int(r[3]), k_cols_padded=int(r[4]),
                            tiles_executed=int(r[5]), pairs_valid=int(r[6])))
        return out


def hva_build_plan(n, assign_q, assign_k, sizes_q, sizes_k, group_of, n_groups, gmask, tile_q, tile_k) -> Plan:
    BH, Nq, Nk = gmask.shape
    dev = gmask.device
    L = hva_plan_describe(BH, n, Nq, Nk, tile_q)
    buf = torch.zeros(L.total, dtype=torch.uint8, device=dev)
    ws = _ws(lib().hva_plan_workspace_bytes(BH, n, Nq, Nk), dev)
    _check(lib().hva_build_plan(BH, n, Nq, Nk, _p(assign_q), _p(assign_k), _p(sizes_q), _p(sizes_k), _p(group_of),
                                _p(n_groups), _p(gmask), int(tile_q), int(tile_k), _p(buf), C.c_size_t(L.total), _p(ws),
                                C.c_size_t(ws.numel()), _stream()))
    return Plan(buf, L, BH, n, Nq, Nk)


def hva_build_plan_static(n, assign_q, assign_k, sizes_q, sizes_k, group_of, n_groups, gmask, tile_q, tile_k, out=None) -> Plan:
    """hva_build_plan with the library's built-in scratch array (hva.h: no allocation inside the call; HVA_ELIMIT beyond
    hva_build_plan_static_limit()).  `out`: a caller-owned uint8 plan buffer of hva_plan_describe().total bytes (allocated here if
    omitted -- the C entry point itself allocates nothing)."""
    BH, Nq, Nk = gmask.shape
    L = hva_plan_describe(BH, n, Nq, Nk, tile_q)
    buf = torch.zeros(L.total, dtype=torch.uint8, device=gmask.device) if out is None else out
    assert buf.numel() >= L.total and buf.dtype == torch.uint8
    _check(lib().hva_build_plan_static(BH, n, Nq, Nk, _p(assign_q), _p(assign_k), _p(sizes_q), _p(sizes_k), _p(group_of),
                                       _p(n_groups), _p(gmask), int(tile_q), int(tile_k), _p(buf), C.c_size_t(L.total), _stream()))
    return Plan(buf, L, BH, n, Nq, Nk)


def hva_permute(shape, X, perm, out=None):
    Y = torch.empty_like(X) if out is None else out
    _check(lib().hva_permute(C.byref(shape), _p(X), _p(perm), _p(Y), _stream()))
    return Y


def hva_unpermute(shape, Xp, perm, out=None):
    Y = torch.empty_like(Xp) if out is None else out
    _check(lib().hva_unpermute(C.byref(shape), _p(Xp), _p(perm), _p(Y), _stream()))
    return Y


def hva_sparse_attention(shape, cfg, Qp, Kp, Vp, plan: Plan, unpermute=True, out=None):
    O = torch.empty_like(Qp) if out is None else out
    _check(lib().hva_sparse_attention(C.byref(shape), C.byref(cfg), _p(Qp), _p(Kp), _p(Vp), _p(plan.buf),
                                      C.c_size_t(plan.L.total), plan.Nq, plan.Nk, _p(O), int(bool(unpermute)),
                                      C.c_void_p(0), C.c_size_t(0), _stream()))
    return O


class Forward:
    """Owns the workspace / state / stats buffers of hva_forward for one (shape, config)."""

    def __init__(self, shape, cfg, device="cuda", with_state=False):
        self.shape, self.cfg = shape, cfg
        self.BH = shape.B * shape.heads
        sb = hva_state_bytes(shape, cfg)
        wb = hva_workspace_bytes(shape, cfg)
        if wb == 0:
            raise HvaError("invalid shape/config")
        self.state = _ws(sb, device) if with_state else None
        self.ws = _ws(wb - (sb if with_state else 0) + 1024, device)
        self.stats = torch.zeros((self.BH, 7), dtype=torch.int64, device=device)

    def __call__(self, Q, K, V, O=None, step_kind=HVA_ANCHOR):
        O = torch.empty_like(Q) if O is None else O
        _check(lib().hva_forward(C.byref(self.shape), C.byref(self.cfg), _p(Q), _p(K), _p(V), _p(O), int(step_kind),
                                 _p(self.state), _p(self.stats), _p(self.ws), C.c_size_t(self.ws.numel()), _stream()))
        return O

    def host(self, hQ, hK, hV, hO, dev_qkvo, step_kind=HVA_ANCHOR):
        _check(lib().hva_forward_host(C.byref(self.shape), C.byref(self.cfg), _p(hQ), _p(hK), _p(hV), _p(hO),
                                      int(step_kind), _p(self.state), _p(dev_qkvo), _p(self.ws),
                                      C.c_size_t(self.ws.numel()), _stream()))
        return hO

    def state_views(self):
        """Typed views of the hybrid cache, located by hva_state_describe()."""
        assert self.state is not None
        s = self.shape
        BH, n, D = self.BH, s.T * s.H * s.W, s.D
        L = hva_state_layout()
        _check(lib().hva_state_describe(C.byref(s), C.byref(self.cfg), C.byref(L)))
        out = {}
        for i, t in enumerate("qk"):
            Nc = L.n_clusters[i]
            for name, shp, dt in (("assign", (BH, n), torch.int32), ("mu", (BH, Nc, D), torch.float32),
                                  ("sums", (BH, Nc, D), torch.float32), ("sizes", (BH, Nc), torch.int32),
                                  ("subset", (BH, max(L.m, 1)), torch.int32)):
                o = getattr(L, name)[i]
                nb = int(math.prod(shp)) * 4
                out[f"{name}_{t}"] = self.state[o:o + nb].view(dt).view(*shp)
        return out

    def ws_views(self):
        """Typed views of the intermediate results the last sparse call left in the workspace (hva_workspace_describe):
        mask, group_of, n_groups, group_mask and the plan."""
        s = self.shape
        BH, n = self.BH, s.T * s.H * s.W
        W = hva_workspace_layout()
        _check(lib().hva_workspace_describe(C.byref(s), C.byref(self.cfg), C.byref(W)))
        Nq, Nk = hva_num_clusters(s, list(self.cfg.cell_q)), hva_num_clusters(s, list(self.cfg.cell_k))
        v = lambda off, shp, dt: self.ws[off:off + int(math.prod(shp)) * torch.empty((), dtype=dt).element_size()].view(dt).view(*shp)
        L = hva_plan_describe(BH, n, max(Nq, 1), max(Nk, 1), self.cfg.tile_q)
        assert L.total == W.plan_bytes
        return dict(mask=v(W.mask, (BH, Nq, Nk), torch.uint8), group_of=v(W.group_of, (BH, Nq), torch.int32),
                    n_groups=v(W.n_groups, (BH,), torch.int32), group_mask=v(W.group_mask, (BH, Nq, Nk), torch.uint8),
                    plan=Plan(self.ws[W.plan:W.plan + W.plan_bytes], L, BH, n, Nq, Nk))

    def stats_dicts(self):
        out = []
        for r in self.stats.cpu().numpy():
            out.append(dict(n_groups=int(r[0] & 0xffffffff), q_tiles=int(r[0] >> 32), q_rows_valid=int(r[1]),
                            q_rows_padded=int(r[2]), k_cols_valid=int(r[3]), k_cols_padded=int(r[4]),
                            tiles_executed=int(r[5]), pairs_valid=int(r[6])))
        return out


hva_forward = Forward
