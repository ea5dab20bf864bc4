#!/usr/bin/env python
"""bench.py -- one "step" = one hva_forward call (anchor step: clustering of Q and K, mask, merge, plan,
permutation, block-sparse attention, inverse permutation) over one batch of synthetic input.

Default workload = BASELINE.json configs[3] (C4, HunyuanVideo shape: 24 heads x 118,800 tokens x 128, bf16),
the configuration the metric is quoted on.  Prints ONE JSON line.
  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4] [--impl ours|reference]
N > 1 (torchrun): every rank runs the same-size call on its own heads' worth of data (head sharding, no
collective; "weak" scaling); value = max-over-ranks ms per step / N.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
from paper_2607_03012_b200 import inputs, sharding  # noqa: E402

# dram__bytes_read.sum + dram__bytes_write.sum of one hva_attn_tc_kernel launch at C4 (top-p 0.9, merging on), from the `ncu --set full`
# capture summarised in profiles/r1f_ncu_full.md (11.72 GB + 0.78 GB); algorithmic minimum 2.9 GB (Q', K', V' once + O)
ATTN_DRAM_BYTES_C4 = 12.49e9

METRIC = "sparse-attn ms/call + clustering ms/step at 118,800-token HunyuanVideo shape"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], tf_burst=d["bf16_tflops"], tf_sust=d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                    src="measured")
    return dict(hbm=6650.0, tf_burst=1590.0, tf_sust=1400.0, src="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, idx):
        self.idx, self.rows, self.proc = idx, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.idx}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i].lower().startswith("active")})
        pw = [float(r[2]) for r in self.rows if len(r) >= 7 and r[2].replace(".", "").isdigit()]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": reasons}


def ev_time(fn, reps):
    """ms per call of fn over `reps` back-to-back calls, CUDA events on the current stream."""
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    a.record()
    for _ in range(reps):
        fn()
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b) / reps


def oracle_sample(wl, head=0, attn_rows=32, merge_rounds=None):
    """The CPU oracle, as it stands, on a bounded sample of the workload: one head's clustering (Q and K), mask,
    merge, plan, and `attn_rows` attention rows.  Returns (seconds by stage, extrapolated ms per full call)."""
    import oracle
    x = inputs.make_head(wl, head)
    Q, K, V = [inputs.to_f64(t) for t in x]
    lat = (wl.T, wl.H, wl.W)
    t = {}
    t0 = time.perf_counter(); cq = oracle.local_window_kmeans(Q, lat, wl.cell, wl.win, wl.iters)
    ck = oracle.local_window_kmeans(K, lat, wl.cell, wl.win, wl.iters); t["cluster"] = time.perf_counter() - t0
    scale = float(np.float32(1 / math.sqrt(wl.D)))
    t0 = time.perf_counter(); M = oracle.build_mask(cq["mu"], ck["mu"], ck["sizes"], scale, float(np.float32(wl.top_p)))
    t["mask"] = time.perf_counter() - t0
    R = wl.merge_rounds if merge_rounds is None else merge_rounds
    t0 = time.perf_counter(); gof, gids, chi = oracle.merge_clusters(cq["sizes"], ck["sizes"], M, wl.tile[0], wl.tile[1], R, seed=wl.seed, bh=head)
    t["merge"] = time.perf_counter() - t0
    t0 = time.perf_counter(); oracle.build_plan(cq["assign"], ck["assign"], gof, len(cq["sizes"]), len(ck["sizes"]))
    t["plan"] = time.perf_counter() - t0
    rows = np.sort(np.random.default_rng(0).choice(wl.n, attn_rows, replace=False))
    t0 = time.perf_counter(); oracle.masked_attention_rows(Q, K, V, rows, cq["assign"], ck["assign"], gof, gids, chi, scale)
    t["attn_rows"] = time.perf_counter() - t0
    per_head = t["cluster"] + t["mask"] + t["merge"] + t["plan"] + t["attn_rows"] * (wl.n / attn_rows)
    return t, per_head * wl.heads * 1e3


def oracle_threads():
    """Threads the oracle actually uses: it is single-process numpy, so its BLAS pool (else 1)."""
    try:
        from threadpoolctl import threadpool_info
        return max([int(i.get("num_threads", 1)) for i in threadpool_info()] or [1])
    except Exception:
        return 1


def workload_config(wl, cell_q, cell_k, win, min_kc, top_p, merge_rounds, custom=False):
    """The `config` object of the JSON line: the same keys for both arms."""
    in_gb = 3 * wl.B * wl.heads * wl.n * wl.D * (2 if wl.dtype == "bf16" else 4) / 1e9
    return {"workload": wl.name + ("+custom-grids" if custom else ""), "B": wl.B, "heads": wl.heads, "n": wl.n, "D": wl.D,
            "cell_q": list(cell_q), "cell_k": list(cell_k), "win": list(win), "min_kc": min_kc, "iters": wl.iters,
            "top_p": top_p, "merge_rounds": merge_rounds, "tile": wl.tile,
            "l2": "inputs (%.2g GB) %s L2" % (in_gb, "larger than" if in_gb > 0.3 else "NOT larger than"),
            "parallelism": "head-sharded replicas, no collective"}


def run_reference(args, wl):
    """--impl reference: the oracle timed on the host cores, each step a bounded sample, extrapolated to ms/call."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    vals = []
    for i in range(args.warmup + args.steps):
        t, ms = oracle_sample(wl, head=i % wl.heads, attn_rows=16, merge_rounds=1 if wl.n > 50000 else None)
        if i >= args.warmup:
            vals.append(ms)
    v = float(np.mean(vals))
    cores = oracle_threads()
    sample = ("per step: one head of %s through oracle clustering (Q,K), mask, 1 merge round, plan and 16 attention rows; "
              "extrapolated x heads and x n/16 rows" % wl.name)
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": "ms", "n_gpus": args.gpus, "steps": args.steps,
                      "warmup": args.warmup, "ms_per_step": v, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
                      "dtype": "f64", "data": "synthetic",
                      "config": workload_config(wl, wl.cell, wl.cell, wl.win, 0.0, float(np.float32(wl.top_p)), wl.merge_rounds),
                      "cpu_baseline": {"value": v, "unit": "ms", "cores": cores, "kind": "oracle", "sample": sample},
                      "e2e": {"value": v, "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C4")
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--top-p", type=float, default=None)
    ap.add_argument("--merge-rounds", type=int, default=None)
    ap.add_argument("--report", default=None, choices=[None, "sweep", "hybrid", "selfbase", "assign-phases"],
                    help="extra reports of BASELINE.json configs[3] / configs[4] instead of the bench line: 'sweep' = top-p x merging "
                         "with CTA tile occupancy, 'hybrid' = the 50-step anchor / subset sequence (use --config C5), 'selfbase' = "
                         "on-box self-baselines: the dense (HVA_DENSE) call next to the sparse one, clustering over window sizes")
    ap.add_argument("--seq-steps", type=int, default=50)
    ap.add_argument("--cell-q", default=None, help="k_t,k_h,k_w of the Q grid (default: the workload's); e.g. the paper's 11,5,5")
    ap.add_argument("--cell-k", default=None, help="k_t,k_h,k_w of the K grid; e.g. the paper's 11,3,3")
    ap.add_argument("--win", default=None, help="w_t,w_h,w_w of both windows; e.g. the paper's 3,8,8")
    ap.add_argument("--min-kc", type=float, default=0.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-stages", action="store_true")
    args = ap.parse_args()
    wl = inputs.CONFIGS[args.config]
    if args.impl == "reference":
        return run_reference(args, wl)

    from paper_2607_03012_b200 import binding as b
    b.lib()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hva path has no CPU fallback")
    if args.report == "sweep":
        return report_sweep(b, wl, args)
    if args.report == "hybrid":
        return report_hybrid(b, wl, args)
    if args.report == "selfbase":
        return report_selfbase(b, wl, args)
    if args.report == "assign-phases":
        return report_assign_phases(b, wl, args)
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl")
    pk = peaks()

    # ---- inputs: generated on the host, resident in HBM before the timed region
    import dataclasses
    wl_r = dataclasses.replace(wl, seed=wl.seed + 1000 * rank) if rank else wl
    hQ, hK, hV = [t.contiguous().pin_memory() for t in inputs.make_qkv(wl_r)]
    Q, K, V = hQ.cuda(), hK.cuda(), hV.cuda()
    shape = b.make_shape(wl)
    cfg = b.make_config(wl, top_p=args.top_p, merge_rounds=args.merge_rounds, min_kc=args.min_kc)
    i3 = type(cfg.cell_q)
    tri = lambda t: i3(*[int(x) for x in t.split(",")])
    if args.cell_q: cfg.cell_q = tri(args.cell_q)
    if args.cell_k: cfg.cell_k = tri(args.cell_k)
    if args.win: cfg.win_q = cfg.win_k = tri(args.win)
    custom = bool(args.cell_q or args.cell_k or args.win or args.min_kc)
    fwd = b.Forward(shape, cfg)
    O = torch.empty_like(Q)
    step = lambda: fwd(Q, K, V, O)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clk = ClockSampler(local)
    clk.start()
    ms = ev_time(step, args.steps)
    clocks = clk.stop()
    if world > 1:
        ms = sharding.max_over_ranks(ms, device="cuda")
        dist.barrier()
    stats = fwd.stats_dicts()

    # ---- end to end through the C ABI with HOST buffers (H2D of Q,K,V and D2H of O inside the timed region)
    hO = torch.empty_like(hQ).pin_memory()
    dev4 = torch.empty((4,) + tuple(Q.shape), dtype=Q.dtype, device="cuda")
    fwd.host(hQ, hK, hV, hO, dev4)
    t0 = time.perf_counter()
    for _ in range(max(1, min(args.steps, 3))):
        fwd.host(hQ, hK, hV, hO, dev4)
    e2e_ms = (time.perf_counter() - t0) * 1e3 / max(1, min(args.steps, 3))
    nbytes = Q.numel() * Q.element_size()
    del dev4

    out = {"metric": METRIC, "value": sharding.whole_job_value(ms, world), "unit": "ms", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
           "ms_per_step": ms, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
           "dtype": "bf16" if wl.dtype == "bf16" else "f32", "data": "synthetic",
           "config": workload_config(wl, list(cfg.cell_q), list(cfg.cell_k), list(cfg.win_q), float(cfg.min_kc), float(cfg.top_p),
                                     int(cfg.merge_rounds), custom),
           "clocks": clocks,
           "e2e": {"value": e2e_ms / world, "unit": "ms", "h2d_bytes_per_step": 3 * nbytes, "d2h_bytes_per_step": nbytes},
           "gpu_launches": args.steps * (2 * (2 + 2 * wl.iters) + 1 + (3 + 3 * int(cfg.merge_rounds) + (1 if int(cfg.merge_rounds) > 0 else 0)) + 7 + 3 + 1)}

    # ---- per-stage times and rooflines (rank 0)
    if rank == 0 and not args.no_stages:
        out.update(stage_report(b, wl, shape, cfg, Q, K, V, stats, pk))
    if rank == 0 and not args.no_cpu_baseline and not custom:
        t, cpu_ms = oracle_sample(wl, attn_rows=32, merge_rounds=1 if wl.n > 50000 else None)
        out["cpu_baseline"] = {"value": cpu_ms, "unit": "ms", "cores": oracle_threads(), "kind": "oracle",
                               "sample": "one head of %s: oracle clustering Q,K %.1fs, mask %.2fs, merge(1 round) %.1fs, plan %.2fs, "
                                         "32 attention rows %.2fs; extrapolated x%d heads, x n/32 rows" % (
                                             wl.name, t["cluster"], t["mask"], t["merge"], t["plan"], t["attn_rows"], wl.heads)}
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def occupancy(wl, stats):
    BH, n = wl.B * wl.heads, wl.n
    tq, tk = wl.tile
    tiles = sum(s["tiles_executed"] for s in stats)
    pairs = sum(s["pairs_valid"] for s in stats)
    padded = tiles * tq * tk
    return {"groups": sum(s["n_groups"] for s in stats), "theoretical_density": pairs / (BH * float(n) * n),
            "cta_density": padded / (BH * float(n) * n), "cta_tile_occupancy": pairs / padded,
            "q_rows_valid_over_padded": sum(s["q_rows_valid"] for s in stats) / sum(s["q_rows_padded"] for s in stats),
            "k_cols_valid_over_padded": sum(s["k_cols_valid"] for s in stats) / sum(s["k_cols_padded"] for s in stats),
            "tiles_executed": tiles}


def report_sweep(b, wl, args):
    """BASELINE.json configs[3]: top-p in {0.8, 0.9, 0.95} x merging {off, on}: ms per call and per attention launch, executed
    and dense-equivalent TFLOP/s, CTA tile occupancy (valid / padded pairs, rows, columns; Eq. 7 l.111, Fig. 5c l.225)."""
    Q, K, V = [t.cuda().contiguous() for t in inputs.make_qkv(wl)]
    shape = b.make_shape(wl)
    O = torch.empty_like(Q)
    BH, n, D = wl.B * wl.heads, wl.n, wl.D
    for top_p in (0.8, 0.9, 0.95):
        for rounds in (0, wl.merge_rounds):
            cfg = b.make_config(wl, top_p=top_p, merge_rounds=rounds)
            fwd = b.Forward(shape, cfg)
            for _ in range(2):
                fwd(Q, K, V, O)
            ms = ev_time(lambda: fwd(Q, K, V, O), max(args.steps, 3))
            occ = occupancy(wl, fwd.stats_dicts())
            exec_flop = 4.0 * D * wl.tile[0] * wl.tile[1] * occ["tiles_executed"]
            print(json.dumps({"report": "sweep", "workload": wl.name, "top_p": top_p, "merge_rounds": rounds, "ms_per_call": round(ms, 3),
                              "executed_tflop": round(exec_flop / 1e12, 2), "dense_equiv_tflops_call": round(4.0 * BH * n * n * D / (ms * 1e-3) / 1e12, 1),
                              "occupancy": {k: (round(v, 4) if isinstance(v, float) else v) for k, v in occ.items()}}))
            del fwd


def report_selfbase(b, wl, args):
    """(a) the dense tcgen05 FlashAttention call (HVA_DENSE: what warm-up steps / layers run,
    l.324) next to the sparse call on the same inputs and box -> an on-box speed-up figure (the paper's own: Table 1 / l.11,
    other hardware); (b) hva_cluster of one tensor over window sizes (our analogue of Fig. 4b, l.85)."""
    Q, K, V = [t.cuda().contiguous() for t in inputs.make_qkv(wl)]
    shape = b.make_shape(wl)
    O = torch.empty_like(Q)
    BH, n, D = wl.B * wl.heads, wl.n, wl.D
    reps = max(args.steps, 3)
    fwd = b.Forward(shape, b.make_config(wl, top_p=args.top_p, merge_rounds=args.merge_rounds, min_kc=args.min_kc))
    for _ in range(2):
        fwd(Q, K, V, O)
    ms_sparse = ev_time(lambda: fwd(Q, K, V, O), reps)
    fwd(Q, K, V, O, step_kind=b.HVA_DENSE)
    ms_dense = ev_time(lambda: fwd(Q, K, V, O, step_kind=b.HVA_DENSE), reps)
    dense_flop = 4.0 * BH * float(n) * n * D
    print(json.dumps({"report": "selfbase", "workload": wl.name, "top_p": float(fwd.cfg.top_p), "merge_rounds": int(fwd.cfg.merge_rounds),
                      "sparse_ms_per_call": round(ms_sparse, 3), "dense_ms_per_call": round(ms_dense, 3),
                      "dense_tflops": round(dense_flop / (ms_dense * 1e-3) / 1e12, 1), "speedup_over_dense": round(ms_dense / ms_sparse, 3)}))
    del fwd
    K3 = [-(-d // k) for d, k in zip((wl.T, wl.H, wl.W), wl.cell)]
    for win in ((1, 1, 1), (3, 3, 3), (3, 5, 5), (5, 5, 5), (3, 8, 8)):
        nwin = 1
        for w_, k_ in zip(win, K3):
            nwin *= min(w_, k_)
        run = lambda: b.hva_cluster(shape, wl.cell, win, wl.iters, K, want_sums=False, want_lowe=False)
        out = run()
        ms = ev_time(run, reps)
        # k-means objective per token (fp64 on the device, from the labels and centroids the call returned)
        J = 0.0
        for h in range(BH):
            x = K.view(BH, n, D)[h].double()
            J += float(((x - out["mu"][h].double()[out["assign"][h].long()]) ** 2).sum())
        gb = wl.iters * BH * n * D * K.element_size() + BH * n * 4
        print(json.dumps({"report": "selfbase-window", "workload": wl.name, "tensor": "K", "win": list(win), "candidates": nwin,
                          "iters": wl.iters, "ms": round(ms, 3), "algorithmic_GBps": round(gb / (ms * 1e-3) / 1e9, 1),
                          "objective_per_token": round(J / (BH * n), 5)}))
        del out


def report_assign_phases(b, wl, args):
    """Per-phase clock64 breakdown of hva_assign_tc_kernel.  Diagnostic, not a bench number: needs the library built with
    `HVA_NVCC_FLAGS=-DHVA_ASSIGN_TIMING python paper_2607_03012_b200/build.py --force` (thread 0 of every CTA adds its clocks per
    phase to the probe buffer of hva_cluster_ex); the product build leaves those entries at zero and this report says so."""
    heads = list(range(min(8, wl.heads)))
    _, K, _ = inputs.make_qkv(wl, heads=heads)
    X = K.cuda().contiguous()
    shape = b.make_shape(wl, heads=len(heads))
    roles = {"scan_group0": ["loop", "table_wait", "tile_wait_xsq", "mma1_wait", "scan_refine_store", "onehot_tile_wait", "onehot_fence_arrive"],
             "epilogue": ["loop", "table_wait", "sums_wait", "stores"],
             "loader": ["draw_issue", "slot_wait", "header", "centroid_buf_wait", "boxes", "draw_wait"],
             "mma1": ["loop", "header_wait", "tables", "tile_wait", "issue"],
             "mma2": ["loop", "table_wait", "onehot_wait", "issue"]}
    cells = 1
    for d, k in zip((wl.T, wl.H, wl.W), wl.cell):
        cells *= -(-d // k)
    for lowe, iters in ((False, 1), (True, 1), (False, wl.iters)):
        b.hva_cluster(shape, wl.cell, wl.win, iters, X, want_lowe=lowe, want_sums=False)
        probe = torch.zeros(64, dtype=torch.float32, device="cuda")
        b.hva_cluster(shape, wl.cell, wl.win, iters, X, want_lowe=lowe, want_sums=False, probe=probe)
        torch.cuda.synchronize()
        pr = probe.cpu().numpy()
        ntiles = cells * len(heads) * iters
        out = {"report": "assign-phases", "workload": wl.name, "heads": len(heads), "iters": iters, "lowe_ratio": lowe,
               "timing_build": bool(pr[16:56].sum() > 0), "unit": "clk per tile of the CTA (scan_group0 handles every third tile)"}
        for r, (role, names) in enumerate(roles.items()):
            out[role] = {n: int(round(float(pr[16 + 8 * r + k]) / ntiles)) for k, n in enumerate(names)}
            out[role]["sum"] = int(sum(out[role].values()))
        print(json.dumps(out))


def report_hybrid(b, wl, args):
    """BASELINE.json configs[4]: X_s = 0.98 X_{s-1} + 0.2 fresh_s for Q, K, V; full clustering at anchor steps (every 10th), subset
    update (l.101-103) in between.  Per step: ms of the whole call and of its clustering part, label agreement with a cold-start
    full re-clustering of X_s (ours, and the frozen anchor labels for comparison), relative k-means objective."""
    import math as _m
    heads = list(range(wl.heads))
    shape = b.make_shape(wl)
    cfg = b.make_config(wl, subset_frac=0.15)
    fwd = b.Forward(shape, cfg, with_state=True)
    cur = [inputs.make_head(wl, h, 0) for h in heads]                      # per head [3, n, D]
    rms0 = [c.float().pow(2).mean(dim=(1, 2)).sqrt() for c in cur]
    from concurrent.futures import ThreadPoolExecutor
    O = None
    frozen = None
    rows = []
    for s in range(args.seq_steps):
        if s > 0:
            with ThreadPoolExecutor(max_workers=min(16, os.cpu_count() or 8)) as ex:
                cur = list(ex.map(lambda h: inputs.hybrid_next(wl, cur[h], h, s, rms0[h]), heads))
        X = torch.stack(cur, dim=1).unsqueeze(1).cuda()                    # [3, 1, heads, n, D]
        Q, K, V = X[0].contiguous(), X[1].contiguous(), X[2].contiguous()
        O = torch.empty_like(Q) if O is None else O
        kind = b.HVA_ANCHOR if s % 10 == 0 else b.HVA_INTERMEDIATE
        a, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); a.record()
        fwd(Q, K, V, O, step_kind=kind)
        e.record(); torch.cuda.synchronize()
        ms = a.elapsed_time(e)
        st = {k: v.clone() for k, v in fwd.state_views().items()}
        # clustering part of the step, timed on copies of the cache
        if kind == b.HVA_ANCHOR:
            def clus():
                for X_, t in ((Q, "q"), (K, "k")):
                    r = b.hva_cluster(shape, wl.cell, wl.win, wl.iters, X_, want_lowe=True)
                    b.hva_select_subset(r["lowe"], st["subset_" + t].shape[1])
            frozen = {t: st["assign_" + t].clone() for t in "qk"}
        else:
            prev = prev_state
            def clus():
                for X_, t in ((Q, "q"), (K, "k")):
                    c2 = {k: prev[k + "_" + t].clone() for k in ("assign", "mu", "sums", "sizes")}
                    b.hva_cluster_update(shape, X_, prev["subset_" + t], c2["assign"], c2["mu"], c2["sums"], c2["sizes"])
        clus()
        ms_cl = ev_time(clus, 1)
        prev_state = st
        agree, agree_frozen, obj = {}, {}, {}
        for X_, t in ((Q, "q"), (K, "k")):
            full = b.hva_cluster(shape, wl.cell, wl.win, wl.iters, X_, want_lowe=False, want_sums=False)
            agree[t] = float((st["assign_" + t] == full["assign"]).float().mean())
            agree_frozen[t] = float((frozen[t] == full["assign"]).float().mean())
            Xf = X_[0].float()
            def J(lab, mu):
                idx = lab.long().unsqueeze(-1).expand(-1, -1, wl.D)
                return float((Xf - torch.gather(mu, 1, idx)).pow(2).sum())
            obj[t] = J(st["assign_" + t], st["mu_" + t]) / J(full["assign"], full["mu"])
        row = {"report": "hybrid", "step": s, "kind": "anchor" if kind == b.HVA_ANCHOR else "subset", "ms_call": round(ms, 3),
               "ms_clustering": round(ms_cl, 3), "agree_q": round(agree["q"], 4), "agree_k": round(agree["k"], 4),
               "agree_frozen_q": round(agree_frozen["q"], 4), "agree_frozen_k": round(agree_frozen["k"], 4),
               "rel_objective_q": round(obj["q"], 4), "rel_objective_k": round(obj["k"], 4)}
        rows.append(row)
        print(json.dumps(row), flush=True)
    anc = [r for r in rows if r["kind"] == "anchor"]; sub = [r for r in rows if r["kind"] == "subset"]
    mean = lambda xs, k: round(sum(x[k] for x in xs) / max(len(xs), 1), 4)
    print(json.dumps({"report": "hybrid-summary", "workload": wl.name, "steps": len(rows), "subset_frac": 0.15,
                      "anchor": {k: mean(anc, k) for k in ("ms_call", "ms_clustering")},
                      "subset": {k: mean(sub, k) for k in ("ms_call", "ms_clustering", "agree_q", "agree_k", "agree_frozen_q",
                                                           "agree_frozen_k", "rel_objective_q", "rel_objective_k")}}))


def stage_report(b, wl, shape, cfg, Q, K, V, stats, pk):
    BH, n, D = wl.B * wl.heads, wl.n, wl.D
    es = Q.element_size()
    reps = 3
    st = {}
    cell_q, cell_k, win_q, win_k = list(cfg.cell_q), list(cfg.cell_k), list(cfg.win_q), list(cfg.win_k)
    cq = b.hva_cluster(shape, cell_q, win_q, wl.iters, Q, want_lowe=False)
    ck = b.hva_cluster(shape, cell_k, win_k, wl.iters, K, want_lowe=False)
    st["cluster_qk"] = ev_time(lambda: (b.hva_cluster(shape, cell_q, win_q, wl.iters, Q, want_lowe=False),
                                        b.hva_cluster(shape, cell_k, win_k, wl.iters, K, want_lowe=False)), reps)
    scale = 1.0 / math.sqrt(D)
    M = b.hva_build_mask(cq["mu"], ck["mu"], ck["sizes"], scale, float(cfg.top_p), float(cfg.min_kc))
    st["mask"] = ev_time(lambda: b.hva_build_mask(cq["mu"], ck["mu"], ck["sizes"], scale, float(cfg.top_p), float(cfg.min_kc)), reps)
    mg = lambda: b.hva_merge(cq["sizes"], ck["sizes"], M, wl.tile[0], wl.tile[1], int(cfg.merge_rounds), seed=wl.seed)
    gof, ng, gm = mg()
    st["merge"] = ev_time(mg, reps)
    pl = lambda: b.hva_build_plan(n, cq["assign"], ck["assign"], cq["sizes"], ck["sizes"], gof, ng, gm, wl.tile[0], wl.tile[1])
    plan = pl()
    st["plan"] = ev_time(pl, reps)
    Qp, Kp, Vp = b.hva_permute(shape, Q, plan.perm_q), b.hva_permute(shape, K, plan.perm_k), b.hva_permute(shape, V, plan.perm_k)
    st["permute_qkv"] = ev_time(lambda: (b.hva_permute(shape, Q, plan.perm_q, out=Qp), b.hva_permute(shape, K, plan.perm_k, out=Kp),
                                         b.hva_permute(shape, V, plan.perm_k, out=Vp)), reps)
    Oo = torch.empty_like(Q)
    at = lambda: b.hva_sparse_attention(shape, cfg, Qp, Kp, Vp, plan, unpermute=True, out=Oo)
    at()
    st["attention"] = ev_time(at, reps)
    tiles = sum(s["tiles_executed"] for s in stats)
    tq, tk = wl.tile
    exec_flop = 4.0 * D * tq * tk * tiles                    # QK^T + PV on every executed (padded) tile
    dense_flop = 4.0 * BH * float(n) * n * D
    t_att = st["attention"] * 1e-3
    ach = exec_flop / t_att / 1e12
    pairs = sum(s["pairs_valid"] for s in stats)
    padded = tiles * tq * tk
    cl_bytes = 2 * wl.iters * BH * n * D * es + 2 * BH * n * 4      # X read once per iteration (Q and K) + labels
    pm_bytes = 3 * 2 * BH * n * D * es + 3 * BH * n * 4
    rep = {
        "stages_ms": {k: round(v, 4) for k, v in st.items()},
        "roofline": {"bound": "tensor", "kernel": "hva_attn_tc_kernel", "achieved": ach, "peak": pk["tf_sust"], "unit": "TFLOP/s",
                     "frac": ach / pk["tf_sust"], "frac_of_burst": ach / pk["tf_burst"], "peak_source": pk["src"] + " (sustained)",
                     "traffic": ATTN_DRAM_BYTES_C4 if (wl.name == "C4-hunyuan" and abs(float(cfg.top_p) - 0.9) < 1e-6 and int(cfg.merge_rounds) == 3) else None,
                     "executed_tflop": exec_flop / 1e12, "dense_equiv_tflops": dense_flop / t_att / 1e12},
        "roofline_cluster": {"bound": "hbm", "kernel": "hva_assign_tc_kernel+hva_finalize_kernel", "achieved": cl_bytes / (st["cluster_qk"] * 1e-3) / 1e9,
                             "peak": pk["hbm"], "unit": "GB/s", "frac": cl_bytes / (st["cluster_qk"] * 1e-3) / 1e9 / pk["hbm"],
                             "algorithmic_bytes": cl_bytes},
        "roofline_permute": {"bound": "hbm", "kernel": "hva_permute_kernel", "achieved": pm_bytes / (st["permute_qkv"] * 1e-3) / 1e9,
                             "peak": pk["hbm"], "unit": "GB/s", "frac": pm_bytes / (st["permute_qkv"] * 1e-3) / 1e9 / pk["hbm"]},
        "occupancy": occupancy(wl, stats),
    }
    return rep


if __name__ == "__main__":
    main()
