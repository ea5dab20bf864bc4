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

# roofline.traffic: dram__bytes_read.sum + dram__bytes_write.sum of one hva_attn_tc_kernel launch at C4 (top-p 0.9, merging on), read
# from the committed `ncu --set full` export named here (profiles/*.md beside it gives the command); algorithmic minimum 2.9 GB
NCU_FULL_CSV = os.path.join("profiles", "r2_ncu_full_raw.csv")


def attn_dram_bytes():
    """(bytes per launch, source file) from the committed ncu raw export, or (None, None)."""
    path = os.path.join(ROOT, NCU_FULL_CSV)
    if not os.path.exists(path):
        return None, None
    import csv
    rows = list(csv.reader(open(path)))
    hdr = next((r for r in rows if "Kernel Name" in r), None)
    if hdr is None:
        return None, None
    try:
        kn, rd, wr = hdr.index("Kernel Name"), hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum")
    except ValueError:
        return None, None
    units = rows[rows.index(hdr) + 1]
    mult = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    for r in rows[rows.index(hdr) + 2:]:
        if len(r) > max(rd, wr) and "hva_attn_tc_kernel" in r[kn]:
            f = lambda i: float(r[i].replace(",", "")) * mult.get(units[i], 1.0)
            return f(rd) + f(wr), NCU_FULL_CSV
    return None, None

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


def oracle_sample(wl, head=0, attn_rows=256):
    """The CPU oracle, as it stands, on a bounded sample of the workload: ONE head in full through clustering (Q and K), mask,
    merge (all R rounds), plan, and `attn_rows` attention rows chosen to cover merged groups, groups of several q-tiles and ragged
    last tiles.  Returns (seconds by stage, ms per full call: the per-head stages x heads, the attention rows
    x n / attn_rows x heads -- both extrapolations are labelled by the caller)."""
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
    t0 = time.perf_counter(); gof, gids, chi = oracle.merge_clusters(cq["sizes"], ck["sizes"], M, wl.tile[0], wl.tile[1], wl.merge_rounds, seed=wl.seed, bh=head)
    t["merge"] = time.perf_counter() - t0
    t0 = time.perf_counter(); po = oracle.build_plan(cq["assign"], ck["assign"], gof, len(cq["sizes"]), len(ck["sizes"]))
    t["plan"] = time.perf_counter() - t0
    # rows: a third from groups of more than one q-tile (first and last row of the group included), a third from merged groups,
    # the rest uniform
    rng = np.random.default_rng(0)
    rows_g = np.diff(po["goff"])
    members = np.bincount(np.searchsorted(np.asarray(gids), gof[cq["sizes"] > 0]), minlength=len(gids))
    pick = []
    for sel in (np.nonzero(rows_g > wl.tile[0])[0], np.nonzero(members > 1)[0]):
        for k in sel[: max(1, attn_rows // 12)]:
            seg = po["perm_q"][po["goff"][k]:po["goff"][k + 1]]
            pick += [seg[0], seg[-1]] + list(rng.choice(seg, min(2, len(seg)), replace=False))
    pick = np.unique(np.array(pick, dtype=np.int64))[: 2 * attn_rows // 3]
    rest = rng.choice(wl.n, attn_rows, replace=False)
    rows = np.unique(np.concatenate([pick, rest]))[:attn_rows]
    t0 = time.perf_counter(); oracle.masked_attention_rows(Q, K, V, rows, cq["assign"], ck["assign"], gof, gids, chi, scale)
    t["attn_rows"] = time.perf_counter() - t0
    t["n_rows"] = len(rows)
    per_head = t["cluster"] + t["mask"] + t["merge"] + t["plan"] + t["attn_rows"] * (wl.n / len(rows))
    return t, per_head * wl.heads * 1e3


def oracle_sample_text(wl, t):
    return ("one head of %s in full through the oracle: clustering Q,K %.1f s, mask %.2f s, merge (%d rounds) %.1f s, plan %.2f s "
            "[measured; x %d heads extrapolated]; attention %d rows (merged, multi-tile and ragged groups included) %.2f s "
            "[measured; x n/%d rows x %d heads extrapolated]" % (wl.name, t["cluster"], t["mask"], wl.merge_rounds, t["merge"], t["plan"],
                                                                 wl.heads, t["n_rows"], t["attn_rows"], t["n_rows"], wl.heads))


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
        t, ms = oracle_sample(wl, head=i % wl.heads, attn_rows=64 if wl.n > 50000 else 256)
        if i >= args.warmup:
            vals.append(ms)
    v = float(np.mean(vals))
    cores = oracle_threads()
    sample = "per step: " + oracle_sample_text(wl, t)
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
    ap.add_argument("--hybrid-heads", type=int, default=24, help="--report hybrid: heads of the call to run (the sequence stays on the device)")
    ap.add_argument("--verbose", action="store_true", help="--report hybrid: one JSON line per step besides the summaries")
    ap.add_argument("--cell-q", default=None, help="k_t,k_h,k_w of the Q grid (default: the workload's); e.g. the paper's 11,5,5")
    ap.add_argument("--cell-k", default=None, help="k_t,k_h,k_w of the K grid; e.g. the paper's 11,3,3")
    ap.add_argument("--win", default=None, help="w_t,w_h,w_w of both windows; e.g. the paper's 3,8,8")
    ap.add_argument("--min-kc", type=float, default=0.0)
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: 'weak' = every rank runs one full-size call (value = max ms / N); 'strong' = ONE call whose heads are "
                         "sharded round-robin over the ranks (sharding.shard_heads; no collective), value = max ms over ranks")
    ap.add_argument("--no-paper-setting", action="store_true", help="skip the secondary measurement at the paper's own hyper-parameters")
    ap.add_argument("--no-graph", action="store_true", help="launch the step eagerly instead of replaying a CUDA graph of hva_forward")
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
    import dataclasses
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl")
    pk = peaks()

    # ---- inputs: generated on the host, resident in HBM before the timed region
    strong = args.scaling == "strong" and world > 1
    if strong:      # one call, heads sharded over the ranks: every rank generates and runs only its own heads of the SAME call
        my_heads = sharding.shard_heads(wl.heads, rank, world)
        hQ, hK, hV = [t.contiguous().pin_memory() for t in inputs.make_qkv(wl, my_heads)]
        wl_full, wl = wl, dataclasses.replace(wl, heads=len(my_heads))
    else:
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

    # clustering timed ALONE, before the long step heats the GPU into its power cap (the kernel is SM-side bound, so its time follows
    # the SM clock: ~1.9 GHz here, ~1.45 GHz inside the step); the in-step figure is taken by stage_report() after the timed region
    cl_alone = None
    if rank == 0 and not args.no_stages:
        cw = cluster_qk_call(b, shape, cfg, Q, K)
        cw()
        cl_alone = ev_time(cw, 10)
    use_graph = not args.no_graph
    if use_graph:       # hva_forward is stream-ordered with no host synchronisation: the step is captured once and replayed
        for _ in range(2):
            step()
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        cap = torch.cuda.Stream()
        with torch.cuda.stream(cap):
            fwd(Q, K, V, O)
            torch.cuda.synchronize()
            with torch.cuda.graph(graph, stream=cap):
                fwd(Q, K, V, O)
        torch.cuda.synchronize()
        step = graph.replay
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

    out = {"metric": METRIC, "value": ms if strong else sharding.whole_job_value(ms, world), "unit": "ms", "n_gpus": world, "steps": args.steps,
           "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": False, "scaling": "strong" if strong else "weak", "vs_baseline": None,
           "dtype": "bf16" if wl.dtype == "bf16" else "f32", "data": "synthetic",
           "config": workload_config(wl_full if strong else wl, list(cfg.cell_q), list(cfg.cell_k), list(cfg.win_q), float(cfg.min_kc),
                                     float(cfg.top_p), int(cfg.merge_rounds), custom),
           "clocks": clocks,
           "e2e": {"value": e2e_ms if strong else e2e_ms / world, "unit": "ms", "h2d_bytes_per_step": 3 * nbytes, "d2h_bytes_per_step": nbytes},
           # kernels of one hva_forward: per tensor init (writes the bf16 split too) + iters x (assign, finalize); mask; merge init (+ nterms) + R x (sides, overlap,
           # propose, apply) + rank + out; plan: key half (koff, hist, scan, scatter; side stream) + query half (groups, work, hist, scan, scatter); one K, V gather (Q is gathered inside the attention kernel); attention
           "gpu_launches": args.steps * (2 * (1 + 2 * wl.iters) + 1 + (3 + 4 * int(cfg.merge_rounds) + (1 if int(cfg.merge_rounds) > 0 else 0)) + 9 + 1 + 1)}

    # ---- per-stage times and rooflines (rank 0)
    if rank == 0 and not args.no_stages:
        out.update(stage_report(b, wl, shape, cfg, Q, K, V, stats, pk, cl_alone))
    out["config"]["launch"] = "CUDA graph replay of one hva_forward" if use_graph else "eager"
    if rank == 0 and world == 1 and not custom and not args.no_paper_setting and wl.name == "C4-hunyuan":
        out["paper_setting"] = paper_setting(b, wl, shape, Q, K, V, O)
    if rank == 0 and not args.no_cpu_baseline and not custom:
        t, cpu_ms = oracle_sample(wl, attn_rows=256)
        out["cpu_baseline"] = {"value": cpu_ms, "unit": "ms", "cores": oracle_threads(), "kind": "oracle", "sample": oracle_sample_text(wl, t)}
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def paper_setting(b, wl, shape, Q, K, V, O):
    """Secondary number: the same call at the paper's own HunyuanVideo hyper-parameters (Table 2 l.338 / SURVEY App. A; 10 iterations
    l.215) instead of BASELINE.json configs[3]'s: Q grid (11,5,5) -> 432 clusters, K grid (11,3,3) -> 1215, (3,8,8) windows = 192
    candidates per token, top-p 0.9, min-kc 0.15, R = 3.  The JSON line's `value` stays on the config BASELINE.json names."""
    cfg = b.make_config(wl, min_kc=0.15)
    i3 = type(cfg.cell_q)
    cfg.cell_q, cfg.cell_k, cfg.win_q, cfg.win_k, cfg.iters = i3(11, 5, 5), i3(11, 3, 3), i3(3, 8, 8), i3(3, 8, 8), 10
    fwd = b.Forward(shape, cfg)
    for _ in range(2):
        fwd(Q, K, V, O)
    ms = ev_time(lambda: fwd(Q, K, V, O), 3)
    assert int(cfg.iters) == 10
    clq = cluster_qk_call(b, shape, cfg, Q, K)
    clq()
    cl = ev_time(clq, 3)
    occ = occupancy(wl, fwd.stats_dicts())
    return {"config": {"cell_q": [11, 5, 5], "cell_k": [11, 3, 3], "win": [3, 8, 8], "iters": 10, "top_p": float(cfg.top_p), "min_kc": 0.15,
                       "merge_rounds": int(cfg.merge_rounds), "N_q": 432, "N_k": 1215},
            "ms_per_call": ms, "clustering_qk_ms": cl, "groups": occ["groups"], "theoretical_density": occ["theoretical_density"],
            "cta_density": occ["cta_density"]}


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
    """BASELINE.json configs[4]: X_s = 0.98 X_{s-1} + 0.2 fresh_s for Q, K, V; full clustering at anchor steps, subset update (l.101-103)
    in between.  The input sequence is generated once (first `--hybrid-heads` heads, `--seq-steps` steps, resident on the device) and
    replayed for every variant: reading R-H3 / R-H3' (hybrid_refresh_all), anchors every 10 steps (BASELINE.json) / every 2 (the paper,
    l.322), subset fraction 0.05 / 0.15 / 0.30.  Per step: ms of the whole call and of its clustering part; label agreement with a
    cold-start full re-clustering of X_s (ours, and the frozen anchor labels for comparison); k-means objective of (labels, centroids)
    relative to the full re-clustering's, for the hybrid state and for the frozen anchor state."""
    from concurrent.futures import ThreadPoolExecutor
    heads = list(range(min(args.hybrid_heads, wl.heads)))
    nh = len(heads)
    shape = b.make_shape(wl, heads=nh)
    cur = [inputs.make_head(wl, h, 0) for h in heads]                      # per head [3, n, D]
    rms0 = [c.float().pow(2).mean(dim=(1, 2)).sqrt() for c in cur]
    seq = []
    for s in range(args.seq_steps):
        if s > 0:
            with ThreadPoolExecutor(max_workers=min(16, os.cpu_count() or 8)) as ex:
                cur = list(ex.map(lambda h: inputs.hybrid_next(wl, cur[h], heads[h], s, rms0[h]), range(nh)))
        X = torch.stack(cur, dim=1).unsqueeze(1).cuda()                    # [3, 1, heads, n, D]
        seq.append((X[0].contiguous(), X[1].contiguous(), X[2].contiguous()))
    full = []                                                              # cold-start full re-clustering of every step (the yardstick)
    for Q, K, V in seq:
        fq = b.hva_cluster(shape, wl.cell, wl.win, wl.iters, Q, want_lowe=False, want_sums=False)
        fk = b.hva_cluster(shape, wl.cell, wl.win, wl.iters, K, want_lowe=False, want_sums=False)
        full.append({"q": (fq["assign"], fq["mu"]), "k": (fk["assign"], fk["mu"])})

    def J(X, lab, mu):
        idx = lab.long().unsqueeze(-1).expand(-1, -1, wl.D)
        return float((X[0].float() - torch.gather(mu, 1, idx)).pow(2).sum())

    variants = [(0, 10, 0.15), (1, 10, 0.15), (0, 2, 0.15), (1, 2, 0.15), (0, 10, 0.05), (0, 10, 0.30)]
    O = torch.empty_like(seq[0][0])
    for refresh, every, frac in variants:
        cfg = b.make_config(wl, subset_frac=frac, refresh_all=refresh)
        fwd = b.Forward(shape, cfg, with_state=True)
        rows, frozen, prev_state = [], None, None
        for s, (Q, K, V) in enumerate(seq):
            kind = b.HVA_ANCHOR if s % every == 0 else b.HVA_INTERMEDIATE
            a, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize(); a.record()
            fwd(Q, K, V, O, step_kind=kind)
            e.record(); torch.cuda.synchronize()
            ms = a.elapsed_time(e)
            st = {k: v.clone() for k, v in fwd.state_views().items()}
            if kind == b.HVA_ANCHOR:          # clustering part of the step, timed on copies of the cache
                def clus():
                    for X_, t in ((Q, "q"), (K, "k")):
                        r = b.hva_cluster(shape, wl.cell, wl.win, wl.iters, X_, want_lowe=True)
                        b.hva_select_subset(r["lowe"], st["subset_" + t].shape[1])
                frozen = {t: (st["assign_" + t].clone(), st["mu_" + t].clone()) for t in "qk"}
            else:
                prev = prev_state
                def clus():
                    for X_, t in ((Q, "q"), (K, "k")):
                        c2 = {k: prev[k + "_" + t].clone() for k in ("assign", "mu", "sums", "sizes")}
                        b.hva_cluster_update(shape, X_, prev["subset_" + t], c2["assign"], c2["mu"], c2["sums"], c2["sizes"], refresh)
            clus()
            ms_cl = ev_time(clus, 1)
            prev_state = st
            row = {"report": "hybrid", "refresh_all": refresh, "anchor_every": every, "subset_frac": frac, "step": s,
                   "kind": "anchor" if kind == b.HVA_ANCHOR else "subset", "ms_call": round(ms, 3), "ms_clustering": round(ms_cl, 3)}
            for X_, t in ((Q, "q"), (K, "k")):
                fl, fm = full[s][t]
                jf = J(X_, fl, fm)
                row["agree_" + t] = round(float((st["assign_" + t] == fl).float().mean()), 4)
                row["agree_frozen_" + t] = round(float((frozen[t][0] == fl).float().mean()), 4)
                row["rel_objective_" + t] = round(J(X_, st["assign_" + t], st["mu_" + t]) / jf, 4)
                row["rel_objective_frozen_" + t] = round(J(X_, frozen[t][0], frozen[t][1]) / jf, 4)
            rows.append(row)
            if args.verbose:
                print(json.dumps(row), flush=True)
        anc = [r for r in rows if r["kind"] == "anchor"]; sub = [r for r in rows if r["kind"] == "subset"]
        mean = lambda xs, k: round(sum(x[k] for x in xs) / max(len(xs), 1), 4)
        keys = ("ms_call", "ms_clustering", "agree_q", "agree_k", "agree_frozen_q", "agree_frozen_k", "rel_objective_q", "rel_objective_k",
                "rel_objective_frozen_q", "rel_objective_frozen_k")
        print(json.dumps({"report": "hybrid-summary", "workload": wl.name, "heads": nh, "steps": len(rows), "refresh_all": refresh,
                          "anchor_every": every, "subset_frac": frac, "anchor": {k: mean(anc, k) for k in ("ms_call", "ms_clustering")},
                          "subset": {k: mean(sub, k) for k in keys},
                          "last_subset_step_before_anchor": {k: mean([r for r in sub if (r["step"] + 1) % every == 0], k) for k in keys}}), flush=True)
        del fwd


def cluster_qk_call(b, shape, cfg, Q, K):
    """The clustering stage as hva_forward runs it (hva_cluster_qk: Q and K on two streams, cfg.iters passes each), with outputs and
    scratch allocated once."""
    _, _, bufs = b.hva_cluster_qk(shape, cfg, Q, K)
    return lambda: b.hva_cluster_qk(shape, cfg, Q, K, bufs=bufs)


def stage_report(b, wl, shape, cfg, Q, K, V, stats, pk, cl_alone=None):
    BH, n, D = wl.B * wl.heads, wl.n, wl.D
    es = Q.element_size()
    reps = 3
    st = {}
    cell_q, cell_k, win_q, win_k = list(cfg.cell_q), list(cfg.cell_k), list(cfg.win_q), list(cfg.win_k)
    cq = b.hva_cluster(shape, cell_q, win_q, wl.iters, Q, want_lowe=False)
    ck = b.hva_cluster(shape, cell_k, win_k, wl.iters, K, want_lowe=False)
    st["cluster_qk"] = ev_time(cluster_qk_call(b, shape, cfg, Q, K), 10)
    if cl_alone is not None:
        st["cluster_qk_alone"] = cl_alone
    scale = 1.0 / math.sqrt(D)
    M = b.hva_build_mask(cq["mu"], ck["mu"], ck["sizes"], scale, float(cfg.top_p), float(cfg.min_kc))
    st["mask"] = ev_time(lambda: b.hva_build_mask(cq["mu"], ck["mu"], ck["sizes"], scale, float(cfg.top_p), float(cfg.min_kc)), reps)
    mg = lambda: b.hva_merge(cq["sizes"], ck["sizes"], M, wl.tile[0], wl.tile[1], int(cfg.merge_rounds), seed=wl.seed)
    gof, ng, gm = mg()
    st["merge"] = ev_time(mg, reps)
    pl = lambda: b.hva_build_plan(n, cq["assign"], ck["assign"], cq["sizes"], ck["sizes"], gof, ng, gm, wl.tile[0], wl.tile[1])
    plan = pl()
    st["plan"] = ev_time(pl, reps)
    # as hva_forward runs it: K' and V' are materialised, the Q rows are gathered inside the attention kernel (HVA_FLAG_Q_UNPERMUTED)
    Kp, Vp = b.hva_permute(shape, K, plan.perm_k), b.hva_permute(shape, V, plan.perm_k)
    st["permute_kv"] = ev_time(lambda: (b.hva_permute(shape, K, plan.perm_k, out=Kp), b.hva_permute(shape, V, plan.perm_k, out=Vp)), reps)
    Oo = torch.empty_like(Q)
    fused = wl.dtype == "bf16" and D == 128 and tuple(wl.tile) == (128, 128)
    cfg_a = cfg
    if fused:
        import copy
        cfg_a = copy.copy(cfg); cfg_a.flags = int(cfg.flags) | b.HVA_FLAG_Q_UNPERMUTED
    Qa = Q if fused else b.hva_permute(shape, Q, plan.perm_q)
    at = lambda: b.hva_sparse_attention(shape, cfg_a, Qa, Kp, Vp, plan, unpermute=True, out=Oo)
    at()
    st["attention"] = ev_time(at, reps)
    tiles = sum(s["tiles_executed"] for s in stats)
    tq, tk = wl.tile
    exec_flop = 4.0 * D * tq * tk * tiles                    # QK^T + PV on every executed (padded) tile
    dense_flop = 4.0 * BH * float(n) * n * D
    t_att = st["attention"] * 1e-3
    ach = exec_flop / t_att / 1e12
    default_cfg = (wl.name == "C4-hunyuan" and abs(float(cfg.top_p) - 0.9) < 1e-6 and int(cfg.merge_rounds) == 3 and
                   list(cfg.cell_q) == list(wl.cell) and list(cfg.cell_k) == list(wl.cell) and list(cfg.win_q) == list(wl.win))
    pairs = sum(s["pairs_valid"] for s in stats)
    padded = tiles * tq * tk
    cl_bytes = 2 * wl.iters * BH * n * D * es + 2 * BH * n * 4      # X read once per iteration (Q and K) + labels
    pm_bytes = 2 * 2 * BH * n * D * es + 2 * BH * n * 4
    rep = {
        "stages_ms": {k: round(v, 4) for k, v in st.items()},
        "roofline": {"bound": "tensor", "kernel": "hva_attn_tc_kernel", "achieved": ach, "peak": pk["tf_sust"], "unit": "TFLOP/s",
                     "frac": ach / pk["tf_sust"], "frac_of_burst": ach / pk["tf_burst"], "peak_source": pk["src"] + " (sustained)",
                     "traffic": attn_dram_bytes()[0] if default_cfg else None, "traffic_source": attn_dram_bytes()[1] if default_cfg else None,
                     "executed_tflop": exec_flop / 1e12, "dense_equiv_tflops": dense_flop / t_att / 1e12},
        "roofline_cluster": {"bound": "hbm", "kernel": "hva_assign_tc_kernel+hva_finalize_kernel", "achieved": cl_bytes / (st["cluster_qk"] * 1e-3) / 1e9,
                             "peak": pk["hbm"], "unit": "GB/s", "frac": cl_bytes / (st["cluster_qk"] * 1e-3) / 1e9 / pk["hbm"],
                             "timed": "inside the step (right after the timed region, GPU at its power-capped clock)",
                             "frac_timed_alone": (cl_bytes / (cl_alone * 1e-3) / 1e9 / pk["hbm"]) if cl_alone else None,
                             "algorithmic_bytes": cl_bytes},
        "roofline_permute": {"bound": "hbm", "kernel": "hva_gather_kv_kernel", "achieved": pm_bytes / (st["permute_kv"] * 1e-3) / 1e9,
                             "peak": pk["hbm"], "unit": "GB/s", "frac": pm_bytes / (st["permute_kv"] * 1e-3) / 1e9 / pk["hbm"]},
        "occupancy": occupancy(wl, stats),
    }
    return rep


if __name__ == "__main__":
    main()
