"""GPU parity: the CUDA path (through the C ABI of libhva.so) against the fp64 oracle, stage by stage with
teacher forcing and end to end.  Tolerances are BASELINE.json's north_star:
labels / masks / merge plans / permutations bit-exact (tokens whose best and second-best squared distances
differ by < 1e-5 relative may take the runner-up); attention max abs <= 2e-2 and rel-L2 <= 1e-2 for bf16,
rel-L2 <= 1e-4 for fp32, against the oracle with the same mask."""
import dataclasses
import math

import numpy as np
import pytest
import torch

import oracle
from paper_2607_03012_b200 import inputs

pytestmark = pytest.mark.gpu

GAP = 1e-5


def _b():
    from paper_2607_03012_b200 import binding
    binding.lib()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device (no CPU fallback exists)"
    return binding


def _heads(wl, heads, f64_idx=None):
    """[3][1, len(heads), n, D] device tensors + per-head fp64 copies (only for f64_idx if given)."""
    Q, K, V = inputs.make_qkv(wl, heads)
    dev = [t.cuda().contiguous() for t in (Q, K, V)]
    keep = range(len(heads)) if f64_idx is None else f64_idx
    f64 = [[inputs.to_f64(t[0, i]) if i in keep else None for i in range(len(heads))] for t in (Q, K, V)]
    return dev, f64


def _lat(wl):
    return (wl.T, wl.H, wl.W)


def check_labels(lab_gpu, X, orc, mu_used):
    """Bit-exact except near ties: a differing token must have oracle gap < 1e-5 and hold the runner-up."""
    lab_o = orc["assign"]
    diff = np.nonzero(lab_gpu != lab_o)[0]
    for l in diff:
        gap = (orc["d2sq"][l] - orc["d1sq"][l]) / max(orc["d1sq"][l], 1e-300)
        d_g = float(((X[l] - mu_used[lab_gpu[l]]) ** 2).sum())
        assert gap < GAP, f"token {l}: labels differ with gap {gap:.3e}"
        assert abs(d_g - orc["d2sq"][l]) <= 1e-9 * max(1.0, orc["d2sq"][l]), f"token {l}: not the runner-up"
    return diff


def _mu_tol(X):
    # Centroid sums are fixed-order fp32 sums of <= ~300 exactly representable terms; the mean divides the accumulated rounding by
    # the count.  Observed on B200 at every config (tests/test_gpu_full_size.py prints it): <= 0.75 * 2^-24 * max|x|.  The bound used
    # here leaves a factor ~5: 4 * 2^-24 * max|x|  (2.4e-7 relative to the largest feature; SURVEY 8(c) asks for 1e-5).
    return 4 * 2.0 ** -24 * float(np.abs(X).max())


def run_cluster_parity(wl, heads, which):
    b = _b()
    dev, f64 = _heads(wl, heads)
    Xd, Xs = dev[which], f64[which]
    shape = b.make_shape(wl, heads=len(heads))
    Nc = wl.n_clusters
    # --- teacher-forced, one iteration at a time (GPU iteration i starts from the oracle's mu^(i-1))
    mu_prev32 = None
    for it in range(wl.iters):
        orcs = []
        for hi in range(len(heads)):
            mi = None if mu_prev32 is None else mu_prev32[hi].astype(np.float64)
            orcs.append(oracle.local_window_kmeans(Xs[hi], _lat(wl), wl.cell, wl.win, 1, mu_init=mi))
        g = b.hva_cluster(shape, wl.cell, wl.win, 1, Xd,
                          mu_init=None if mu_prev32 is None else torch.from_numpy(mu_prev32).cuda())
        torch.cuda.synchronize()
        lab = g["assign"].cpu().numpy()
        for hi, orc in enumerate(orcs):
            mu_used = oracle.cluster.init_centroids(Xs[hi], _lat(wl), wl.cell) if mu_prev32 is None else mu_prev32[hi].astype(np.float64)
            diff = check_labels(lab[hi], Xs[hi], orc, mu_used)
            sz = g["sizes"][hi].cpu().numpy()
            assert sz.sum() == wl.n
            touched = set(lab[hi][diff]) | set(orc["assign"][diff])
            keep = np.array([u not in touched for u in range(Nc)])
            assert np.array_equal(sz[keep], orc["sizes"][keep])
            mg = g["mu"][hi].cpu().numpy().astype(np.float64)
            assert np.abs(mg[keep] - orc["mu"][keep]).max() <= _mu_tol(Xs[hi])
            sg = g["sums"][hi].cpu().numpy().astype(np.float64)
            assert np.abs(sg[keep] - orc["sums"][keep]).max() <= _mu_tol(Xs[hi]) * max(1, orc["sizes"].max())
            rho = oracle.lowe_ratio(orc["d1sq"], orc["d2sq"])
            same = lab[hi] == orc["assign"]
            assert np.abs(g["lowe"][hi].cpu().numpy()[same] - rho[same]).max() <= 2e-5
        mu_prev32 = np.stack([o["mu"] for o in orcs]).astype(np.float32)
    # --- free running N_iter iterations: exact unless a near tie flipped upstream
    g = b.hva_cluster(shape, wl.cell, wl.win, wl.iters, Xd)
    g2 = b.hva_cluster(shape, wl.cell, wl.win, wl.iters, Xd)
    torch.cuda.synchronize()
    for k in ("assign", "mu", "sizes", "sums", "lowe"):                 # deterministic: same bits twice
        assert torch.equal(g[k], g2[k]), k
    flips = 0
    for hi in range(len(heads)):
        orc = oracle.local_window_kmeans(Xs[hi], _lat(wl), wl.cell, wl.win, wl.iters)
        lab = g["assign"][hi].cpu().numpy()
        nd = int((lab != orc["assign"]).sum())
        flips += nd
        if nd == 0:
            assert np.array_equal(g["sizes"][hi].cpu().numpy(), orc["sizes"])
            assert np.abs(g["mu"][hi].cpu().numpy() - orc["mu"]).max() <= 4 * _mu_tol(Xs[hi])
    return flips


@pytest.mark.parametrize("which", [0, 1])
def test_cluster_c1(which):
    assert run_cluster_parity(inputs.C1, [0, 1], which) == 0


@pytest.mark.parametrize("which", [0, 1])
def test_cluster_c2(which):
    flips = run_cluster_parity(inputs.C2, [0, 3, 7], which)
    assert flips <= 3          # free-running flips can only come from exempt near ties (checked per iteration)


def test_cluster_non_dividing_lattice_and_wide_window():
    # non-dividing cells (R-C4), even window (R-C3), window wider than the grid on one axis, D=64 bf16, f32 D=128
    for dt, D, cell, win in (("bf16", 64, (2, 3, 4), (3, 4, 3)), ("f32", 128, (3, 2, 5), (5, 3, 2))):
        wl = dataclasses.replace(inputs.C1, name="edge", heads=2, D=D, dtype=dt, T=5, H=7, W=9, cell=cell, win=win, seed=11)
        assert run_cluster_parity(wl, [0, 1], 0) == 0


def test_cluster_tensor_pipe_edge_shapes():
    # tcgen05 assignment path (bf16, D=128): non-dividing lattice with zero-filled TMA rows (R-C4), even window (R-C3),
    # windows of 12 / 48 / 75 candidates (one and several 32-column TMEM chunks), cell of exactly 128 tokens
    # ... and cells of more than 128 tokens, split along t into several CTA tiles (the paper's (11,5,5) Q cells: 275 tokens)
    for T, H, W, cell, win in ((5, 7, 9, (2, 3, 4), (3, 4, 3)), (6, 13, 21, (2, 3, 5), (3, 4, 4)), (8, 16, 16, (2, 8, 8), (3, 2, 2)),
                               (10, 11, 12, (2, 2, 2), (3, 5, 5)), (23, 10, 10, (11, 5, 5), (3, 8, 8)), (9, 16, 8, (4, 8, 8), (3, 3, 3))):
        wl = dataclasses.replace(inputs.C2, name="edge-tc", heads=2, T=T, H=H, W=W, cell=cell, win=win, seed=12)
        assert run_cluster_parity(wl, [0, 1], 1) <= 1


@pytest.mark.parametrize("wl", [inputs.C2, dataclasses.replace(inputs.C2, name="edge-tc2", T=7, H=22, W=30, cell=(3, 4, 4), seed=13)])
def test_cluster_tensor_pipe_equals_direct_form(wl):
    """The tensor-pipe score only filters: after one pass labels, sizes and rho are those of the fp32 direct-form kernel
    bit for bit, with and without the Lowe ratio (the filter-decided fast path); the centroid sums come from the MMA's
    fp32 accumulation instead of a sequential fp32 loop and agree within the summation tolerance; the observed filter
    error stays far inside the margin the kernel assumes (2 * kEpsDot = 2^-14)."""
    b = _b()
    heads = [0, 5]
    (Qd, Kd, _), _ = _heads(wl, heads, f64_idx=[])
    shape = b.make_shape(wl, heads=len(heads))
    for X in (Qd, Kd):
        tol = _mu_tol(X.float().cpu().numpy())
        for lowe in (False, True):
            for iters in (1, wl.iters):
                ref = b.hva_cluster(shape, wl.cell, wl.win, iters, X, want_lowe=lowe, flags=b.HVA_FLAG_CLUSTER_SIMT)
                probe = torch.zeros(32, dtype=torch.float32, device="cuda")
                got = b.hva_cluster(shape, wl.cell, wl.win, iters, X, want_lowe=lowe, probe=probe)      # instrumented instantiation
                plain = b.hva_cluster(shape, wl.cell, wl.win, iters, X, want_lowe=lowe)                 # product instantiation
                torch.cuda.synchronize()
                for k in ("assign", "sizes", "mu", "sums") + (("lowe",) if lowe else ()):
                    assert torch.equal(plain[k], got[k]), k
                if iters == 1:
                    for k in ("assign", "sizes") + (("lowe",) if lowe else ()):
                        assert torch.equal(ref[k], got[k]), k
                    assert float((ref["mu"] - got["mu"]).abs().max()) <= tol
                    assert float((ref["sums"] - got["sums"]).abs().max()) <= tol * int(ref["sizes"].max())
                else:   # later passes start from centroids that differ in the last bits: only near ties may flip
                    assert float((ref["assign"] != got["assign"]).float().mean()) <= 1e-4
                assert 0 < float(probe[0].item()) < 2.0 ** -14 / 8, float(probe[0].item())


def test_tensor_pipe_exact_ties_take_the_first_minimum():
    """Degenerate inputs for the filter-and-refine kernels: few distinct token values, so most centroids coincide and every
    candidate of a token ties EXACTLY.  All of them are contenders (the many-contender path of both kernels: in-window exact
    refine, and the warp-cooperative exact scan of the subset step); the result must be the first minimum in ascending
    centroid id, as in the oracle (R-C1)."""
    b = _b()
    wl = dataclasses.replace(inputs.C2, name="ties", heads=2, T=6, H=8, W=16, cell=(2, 4, 4), seed=21)
    rng = np.random.default_rng(21)
    vals = torch.from_numpy(rng.standard_normal((3, wl.D)).astype(np.float32)).to(torch.bfloat16)      # three distinct rows
    pick = torch.from_numpy(rng.integers(0, 3, size=(1, 2, wl.n)))
    X = vals[pick].contiguous()                                                                         # [1, 2, n, D]
    Xd = X.cuda()
    shape = b.make_shape(wl, heads=2)
    g = b.hva_cluster(shape, wl.cell, wl.win, 2, Xd)
    torch.cuda.synchronize()
    Nc = wl.n_clusters
    for hi in range(2):
        x64 = inputs.to_f64(X[0, hi])
        orc = oracle.local_window_kmeans(x64, _lat(wl), wl.cell, wl.win, 2)
        assert np.array_equal(g["assign"][hi].cpu().numpy(), orc["assign"])
        assert np.array_equal(g["sizes"][hi].cpu().numpy(), orc["sizes"])
    # subset step: every token, all N_c candidates, centroids that coincide exactly
    sub = torch.arange(wl.n, dtype=torch.int32).repeat(2, 1).cuda()
    mu32 = g["mu"].clone(); mu32[:, 1::2] = mu32[:, 0::2][:, : mu32[:, 1::2].shape[1]]                  # duplicate centroids pairwise
    assign, mu, sums, sizes = g["assign"].clone(), mu32.clone(), g["sums"].clone(), g["sizes"].clone()
    b.hva_cluster_update(shape, Xd, sub, assign, mu, sums, sizes, 1)
    torch.cuda.synchronize()
    for hi in range(2):
        x64 = inputs.to_f64(X[0, hi])
        a, *_ = oracle.subset_update(x64, g["assign"][hi].cpu().numpy().astype(np.int64), mu32[hi].cpu().numpy().astype(np.float64),
                                     g["sums"][hi].cpu().numpy().astype(np.float64), g["sizes"][hi].cpu().numpy().astype(np.int64),
                                     np.arange(wl.n), refresh_all=True)
        assert np.array_equal(assign[hi].cpu().numpy(), a)


def _oracle_stage_inputs(wl, heads, f64):
    """Oracle clustering of Q and K per head (the 'teacher' for the downstream stages)."""
    out = []
    for hi in range(len(heads)):
        cq = oracle.local_window_kmeans(f64[0][hi], _lat(wl), wl.cell, wl.win, wl.iters)
        ck = oracle.local_window_kmeans(f64[1][hi], _lat(wl), wl.cell, wl.win, wl.iters)
        out.append((cq, ck))
    return out


def run_downstream_parity(wl, heads, top_p, rounds, rows_per_head=None, seed_rows=0, max_q_tiles=0):
    """mask -> merge -> plan -> permute -> attention, each fed the ORACLE's upstream results."""
    b = _b()
    dev, f64 = _heads(wl, heads)
    shape = b.make_shape(wl, heads=len(heads))
    cfg = b.make_config(wl, top_p=top_p, merge_rounds=rounds, max_q_tiles=max_q_tiles)
    cl = _oracle_stage_inputs(wl, heads, f64)
    scale32 = float(np.float32(1.0 / math.sqrt(wl.D)))
    p32 = float(np.float32(top_p))
    i32 = lambda a: torch.from_numpy(np.ascontiguousarray(a).astype(np.int32)).cuda()
    mu_q32 = np.stack([c[0]["mu"] for c in cl]).astype(np.float32)
    mu_k32 = np.stack([c[1]["mu"] for c in cl]).astype(np.float32)
    sizes_q = np.stack([c[0]["sizes"] for c in cl]); sizes_k = np.stack([c[1]["sizes"] for c in cl])
    # S5 mask
    Mg = b.hva_build_mask(torch.from_numpy(mu_q32).cuda(), torch.from_numpy(mu_k32).cuda(), i32(sizes_k), scale32, p32).cpu().numpy()
    Mo = []
    for hi in range(len(heads)):
        M, margin = oracle.build_mask(mu_q32[hi].astype(np.float64), mu_k32[hi].astype(np.float64), sizes_k[hi], scale32, p32,
                                      return_margin=True)
        bad = np.nonzero((M != Mg[hi]).any(axis=1))[0]
        assert all(margin[r] < 1e-9 for r in bad), f"mask rows differ away from the threshold: {bad[:5]}"
        Mo.append(M)
    Mo = np.stack(Mo)
    # S6 merge (fed the oracle's mask)
    gof_g, ng_g, gm_g = b.hva_merge(i32(sizes_q), i32(sizes_k), torch.from_numpy(Mo).cuda(), wl.tile[0], wl.tile[1], rounds,
                                    seed=wl.seed, max_q_tiles=max_q_tiles)
    merged = []
    for hi in range(len(heads)):
        gof, gids, chi = oracle.merge_clusters(sizes_q[hi], sizes_k[hi], Mo[hi], wl.tile[0], wl.tile[1], rounds, seed=wl.seed,
                                               bh=hi, max_q_tiles=max_q_tiles)
        assert np.array_equal(gof_g[hi].cpu().numpy(), gof)
        assert int(ng_g[hi]) == len(gids)
        gm = gm_g[hi].cpu().numpy()
        assert np.array_equal(gm[:len(gids)], chi) and not gm[len(gids):].any()
        merged.append((gof, gids, chi))
    # S7 plan (fed the oracle's labels and groups)
    aq = np.stack([c[0]["assign"] for c in cl]); ak = np.stack([c[1]["assign"] for c in cl])
    plan = b.hva_build_plan(wl.n, i32(aq), i32(ak), i32(sizes_q), i32(sizes_k), gof_g, ng_g, gm_g, wl.tile[0], wl.tile[1])
    torch.cuda.synchronize()
    stats = plan.stats_dicts()
    for hi in range(len(heads)):
        po = oracle.build_plan(aq[hi], ak[hi], merged[hi][0], wl.n_clusters, wl.n_clusters)
        assert np.array_equal(plan.perm_q[hi].cpu().numpy(), po["perm_q"])
        assert np.array_equal(plan.inv_perm_q[hi].cpu().numpy(), po["inv_perm_q"])
        assert np.array_equal(plan.perm_k[hi].cpu().numpy(), po["perm_k"])
        assert np.array_equal(plan.koff[hi].cpu().numpy(), po["koff"])
        ng = len(po["gids"])
        assert np.array_equal(plan.gid[hi].cpu().numpy()[:ng], po["gids"])
        assert np.array_equal(plan.goff[hi].cpu().numpy()[:ng + 1], po["goff"])
        kap = (merged[hi][2].astype(np.int64) * sizes_k[hi][None, :]).sum(1)
        assert np.array_equal(plan.kappa[hi].cpu().numpy()[:ng], kap)
        rows = np.diff(po["goff"])
        st = stats[hi]                                                  # occupancy terms of Eq. 7-8
        assert st["n_groups"] == ng and st["q_rows_valid"] == wl.n and st["k_cols_valid"] == kap.sum()
        assert st["pairs_valid"] == int((rows * kap).sum())
        assert st["tiles_executed"] == int((-(-rows // wl.tile[0]) * -(-kap // wl.tile[1])).sum())
    # S8 permute / S10 unpermute: byte copies
    Qp = b.hva_permute(shape, dev[0], plan.perm_q); Kp = b.hva_permute(shape, dev[1], plan.perm_k)
    Vp = b.hva_permute(shape, dev[2], plan.perm_k)
    for hi in range(len(heads)):
        assert torch.equal(Qp[0, hi], dev[0][0, hi][plan.perm_q[hi].long()])
        assert torch.equal(Kp[0, hi], dev[1][0, hi][plan.perm_k[hi].long()])
    assert torch.equal(b.hva_unpermute(shape, Qp, plan.perm_q), dev[0])
    # S9 + S10 attention with the oracle's plan
    O = b.hva_sparse_attention(shape, cfg, Qp, Kp, Vp, plan, unpermute=True)
    Operm = b.hva_sparse_attention(shape, cfg, Qp, Kp, Vp, plan, unpermute=False)
    torch.cuda.synchronize()
    assert torch.equal(b.hva_unpermute(shape, Operm, plan.perm_q), O)
    if wl.dtype == "bf16" and wl.D == 128:             # Eq. 1 fused into the load: the kernel gathers the rows of the UNPERMUTED Q (TMA gather4)
        cfg_g = b.make_config(wl, top_p=top_p, merge_rounds=rounds, max_q_tiles=max_q_tiles, flags=b.HVA_FLAG_Q_UNPERMUTED)
        assert torch.equal(b.hva_sparse_attention(shape, cfg_g, dev[0], Kp, Vp, plan, unpermute=True), O)
    check_attention(wl, heads, f64, O, [(c[0]["assign"], c[1]["assign"]) for c in cl], merged, rows_per_head, seed_rows)
    return plan, stats


def check_attention(wl, heads, f64, O, labels, merged, rows_per_head=None, seed_rows=0):
    scale32 = float(np.float32(1.0 / math.sqrt(wl.D)))
    rng = np.random.default_rng(seed_rows)
    for hi in range(len(heads)):
        rows = np.arange(wl.n) if rows_per_head is None else np.sort(rng.choice(wl.n, rows_per_head, replace=False))
        gof, gids, chi = merged[hi]
        ref = oracle.masked_attention_rows(f64[0][hi], f64[1][hi], f64[2][hi], rows, labels[hi][0], labels[hi][1], gof, gids,
                                           chi, scale32)
        got = O[0, hi].float().cpu().numpy().astype(np.float64)[rows]
        rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
        mx = np.abs(got - ref).max()
        if wl.dtype == "bf16":
            assert mx <= 2e-2 and rel <= 1e-2, (hi, mx, rel)
        else:
            assert rel <= 1e-4, (hi, mx, rel)


def test_downstream_c1_fp32():
    run_downstream_parity(inputs.C1, [0, 1], 0.9, 3)


def test_downstream_c1_merge_off_and_dense_top_p():
    run_downstream_parity(inputs.C1, [0, 1], 0.9, 0)
    run_downstream_parity(inputs.C1, [0], 1.0, 3)          # top_p = 1: every key cluster, full attention


def test_downstream_c2_bf16_tcgen05():
    plan, stats = run_downstream_parity(inputs.C2, [0, 5], 0.9, 3, rows_per_head=768)
    assert stats[0]["n_groups"] < inputs.C2.n_clusters     # merging did merge


def test_downstream_c2_variants():
    run_downstream_parity(inputs.C2, [1], 0.8, 0, rows_per_head=512)      # merge off: many ragged single-cluster groups
    run_downstream_parity(inputs.C2, [2], 0.95, 3, rows_per_head=512, max_q_tiles=1)
    run_downstream_parity(inputs.C2, [3], 1.0, 1, rows_per_head=256)      # dense through the sparse machinery


def test_attention_tc_matches_simt_kernel():
    """The two attention kernels (tcgen05 / CUDA-core) agree on the same bf16 inputs and plan."""
    b = _b()
    wl = inputs.C2
    dev, f64 = _heads(wl, [4])
    fwd = b.Forward(b.make_shape(wl, heads=1), b.make_config(wl))
    O1 = fwd(*dev).clone()
    fwd2 = b.Forward(b.make_shape(wl, heads=1), b.make_config(wl, flags=b.HVA_FLAG_ATTN_SIMT))
    O2 = fwd2(*dev).clone()
    torch.cuda.synchronize()
    d = (O1.float() - O2.float()).abs()
    assert (d <= 2e-2 + 2.0 ** -7 * O2.float().abs()).all()          # both are bf16-rounded: allow 2 output ulps
    assert (d.norm() / O2.float().norm()).item() <= 5e-3
    assert torch.equal(fwd2(*dev), O2)                       # deterministic
    assert torch.equal(fwd(*dev), O1)


def _forward_vs_oracle(wl, heads, top_p=None, rounds=None, rows_per_head=None, check_heads=None):
    """hva_forward from Q, K, V only.  Labels are checked against the free-running oracle; mask / merge / attention
    are checked against the oracle re-run from the GPU's own clustering result (labels, fp32 centroids, sizes), so a
    near-tie flip upstream cannot masquerade as a downstream error."""
    b = _b()
    dev, f64 = _heads(wl, heads, check_heads)
    top_p = wl.top_p if top_p is None else top_p
    rounds = wl.merge_rounds if rounds is None else rounds
    fwd = b.Forward(b.make_shape(wl, heads=len(heads)), b.make_config(wl, top_p=top_p, merge_rounds=rounds), with_state=True)
    O = fwd(*dev)
    torch.cuda.synchronize()
    sv = fwd.state_views()
    scale32 = float(np.float32(1.0 / math.sqrt(wl.D)))
    labels, merged, flips = [], [], 0
    st = fwd.stats_dicts()
    check_heads = range(len(heads)) if check_heads is None else check_heads
    for hi in check_heads:
        aq, ak = sv["assign_q"][hi].cpu().numpy().astype(np.int64), sv["assign_k"][hi].cpu().numpy().astype(np.int64)
        for which, lab in ((0, aq), (1, ak)):
            orc = oracle.local_window_kmeans(f64[which][hi], _lat(wl), wl.cell, wl.win, wl.iters)
            flips += int((lab != orc["assign"]).sum())
        sq, sk = np.bincount(aq, minlength=wl.n_clusters), np.bincount(ak, minlength=wl.n_clusters)
        assert np.array_equal(sq, sv["sizes_q"][hi].cpu().numpy()) and np.array_equal(sk, sv["sizes_k"][hi].cpu().numpy())
        M = oracle.build_mask(sv["mu_q"][hi].cpu().numpy().astype(np.float64), sv["mu_k"][hi].cpu().numpy().astype(np.float64),
                              sk, scale32, float(np.float32(top_p)))
        gof, gids, chi = oracle.merge_clusters(sq, sk, M, wl.tile[0], wl.tile[1], rounds, seed=wl.seed, bh=hi)
        assert st[hi]["n_groups"] == len(gids)
        kap = (chi.astype(np.int64) * sk[None, :]).sum(1)
        assert st[hi]["k_cols_valid"] == int(kap.sum())
        labels.append((aq, ak)); merged.append((gof, gids, chi))
    sel = list(check_heads)
    check_attention(wl, [heads[i] for i in sel], [[f[i] for i in sel] for f in f64], O[:, sel], labels, merged, rows_per_head)
    return fwd, dev, O, flips


def test_forward_c1_end_to_end():
    fwd, dev, O, flips = _forward_vs_oracle(inputs.C1, [0, 1])
    assert flips == 0
    assert torch.equal(fwd(*dev), O)


def test_forward_c2_end_to_end():
    """All 8 heads of C2 through hva_forward, every head chain-checked (GPU iteration i against one oracle iteration from the GPU's
    own previous centroids, R-C10) and every downstream array compared bit for bit (tests/test_gpu_full_size.py helpers)."""
    from test_gpu_full_size import forward_full_check
    for hi in range(8):
        forward_full_check("C2", check_head=hi, rows_per_head=128)


def test_forward_host_matches_device_call():
    """hva_forward_host (HOST buffers; with >= 8 heads it runs in chunks of heads with the copies overlapped on two copy
    streams) returns the bits of hva_forward on device tensors."""
    b = _b()
    for wl, heads in ((inputs.C2, list(range(8))), (inputs.C2, [0, 3, 5])):
        Q, K, V = inputs.make_qkv(wl, heads)
        shape = b.make_shape(wl, heads=len(heads))
        fwd = b.Forward(shape, b.make_config(wl))
        O_dev = fwd(Q.cuda(), K.cuda(), V.cuda()).cpu()
        hQ, hK, hV = [t.contiguous().pin_memory() for t in (Q, K, V)]
        hO = torch.empty_like(hQ).pin_memory()
        dev4 = torch.empty((4,) + tuple(Q.shape), dtype=Q.dtype, device="cuda")
        fwd.host(hQ, hK, hV, hO, dev4)
        assert torch.equal(hO, O_dev)


def test_forward_dense_step_is_full_attention():
    b = _b()
    for wl in (inputs.C1, inputs.C2):
        dev, f64 = _heads(wl, [0])
        fwd = b.Forward(b.make_shape(wl, heads=1), b.make_config(wl))
        O = fwd(*dev, step_kind=b.HVA_DENSE)
        torch.cuda.synchronize()
        rows = np.arange(wl.n) if wl.n <= 512 else np.arange(0, wl.n, 13)
        ones = np.ones((1, 1), np.uint8)
        z = np.zeros(wl.n, np.int64)
        ref = oracle.masked_attention_rows(f64[0][0], f64[1][0], f64[2][0], rows, z, z, np.zeros(1, np.int64), [0], ones,
                                           float(np.float32(1 / math.sqrt(wl.D))))
        got = O[0, 0].float().cpu().numpy().astype(np.float64)[rows]
        rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
        assert rel <= (1e-4 if wl.dtype == "f32" else 1e-2) and (wl.dtype == "f32" or np.abs(got - ref).max() <= 2e-2)


# ----------------------------------------------------------------------------- hybrid (S3, S4)
@pytest.mark.parametrize("wl,heads", [(inputs.C1, [0, 1]), (inputs.C2, [0, 6])])
def test_subset_select_and_update(wl, heads):
    b = _b()
    dev, f64 = _heads(wl, heads)
    shape = b.make_shape(wl, heads=len(heads))
    n, Nc = wl.n, wl.n_clusters
    m = int(math.floor(0.15 * n + 0.5))
    for which in (0, 1):
        orcs = [oracle.local_window_kmeans(f64[which][hi], _lat(wl), wl.cell, wl.win, wl.iters) for hi in range(len(heads))]
        rho32 = np.stack([oracle.lowe_ratio(o["d1sq"], o["d2sq"]) for o in orcs]).astype(np.float32)
        rho32[0, : n // 7] = rho32[0, n // 7]                          # a block of exact ties
        sub_g = b.hva_select_subset(torch.from_numpy(rho32).cuda(), m).cpu().numpy()
        sub_o = np.stack([oracle.select_subset(rho32[hi].astype(np.float64), 0.15) for hi in range(len(heads))])
        assert np.array_equal(sub_g, sub_o)                            # exact on identical fp32 rho (S3)
        # S4: new features, cached oracle state rounded to fp32
        rng = np.random.default_rng(5 + which)
        X2 = (dev[which].float() + 0.25 * torch.from_numpy(rng.standard_normal(dev[which].shape).astype(np.float32)).cuda()).to(dev[which].dtype)
        for refresh in (0, 1):
            assign = torch.from_numpy(np.stack([o["assign"] for o in orcs]).astype(np.int32)).cuda()
            mu32 = np.stack([o["mu"] for o in orcs]).astype(np.float32)
            z32 = np.stack([o["sums"] for o in orcs]).astype(np.float32)
            mu, sums = torch.from_numpy(mu32).cuda(), torch.from_numpy(z32).cuda()
            sizes = torch.from_numpy(np.stack([o["sizes"] for o in orcs]).astype(np.int32)).cuda()
            b.hva_cluster_update(shape, X2, torch.from_numpy(sub_o.astype(np.int32)).cuda(), assign, mu, sums, sizes, refresh)
            torch.cuda.synchronize()
            for hi in range(len(heads)):
                x2 = inputs.to_f64(X2[0, hi])
                a, mo, zo, no, d1, d2 = oracle.subset_update(x2, orcs[hi]["assign"], mu32[hi].astype(np.float64),
                                                             z32[hi].astype(np.float64), orcs[hi]["sizes"], sub_o[hi],
                                                             refresh_all=bool(refresh))
                ag = assign[hi].cpu().numpy()
                diff = np.nonzero(ag != a)[0]
                pos = {int(t): k for k, t in enumerate(sub_o[hi])}
                for l in diff:                                          # near-tie rule over all N_c candidates
                    k = pos[int(l)]
                    assert (d2[k] - d1[k]) / max(d1[k], 1e-300) < GAP
                if len(diff) == 0:
                    assert np.array_equal(sizes[hi].cpu().numpy(), no)
                    tol = _mu_tol(x2) * (4 if not refresh else 1)
                    assert np.abs(mu[hi].cpu().numpy() - mo).max() <= tol + 1e-6 * np.abs(mo).max()
                    assert np.abs(sums[hi].cpu().numpy() - zo).max() <= (tol + 1e-6) * max(1, no.max())
                rest = np.setdiff1d(np.arange(n), sub_o[hi])
                assert np.array_equal(ag[rest], orcs[hi]["assign"][rest])   # non-subset labels untouched


@pytest.mark.parametrize("refresh", [0, 1])
def test_hybrid_forward_sequence_c2(refresh):
    """anchor -> intermediate -> intermediate through hva_forward (step_kind), against the oracle at every step: the subset cached
    at the anchor equals oracle.select_subset on the GPU's own rho; each intermediate step equals oracle.subset_update (R-H3 /
    R-H3') applied to the GPU's previous state under the gap rule; mask / merge / plan / attention of every step are checked
    against the oracle re-run from the GPU's state."""
    from test_gpu_full_size import check_downstream
    b = _b()
    wl = inputs.C2
    heads = [0, 1]
    dev, f64 = _heads(wl, heads)
    shape = b.make_shape(wl, heads=2)
    cfg = b.make_config(wl, subset_frac=0.15, refresh_all=refresh)
    fwd = b.Forward(shape, cfg, with_state=True)
    O0 = fwd(*dev, step_kind=b.HVA_ANCHOR).clone()
    plain = b.Forward(shape, b.make_config(wl))(*dev)
    assert torch.equal(O0, plain)                                      # the hybrid cache does not change an anchor step
    sv = {k: v.clone() for k, v in fwd.state_views().items()}
    for t, X in (("q", dev[0]), ("k", dev[1])):                        # S3 inside hva_forward
        r = b.hva_cluster(shape, wl.cell, wl.win, wl.iters, X, want_lowe=True)
        assert torch.equal(r["assign"], sv["assign_" + t])
        for hi in range(2):
            sub_o = oracle.select_subset(r["lowe"][hi].cpu().numpy().astype(np.float64), 0.15)
            assert np.array_equal(sv["subset_" + t][hi].cpu().numpy(), sub_o)
    g = torch.Generator(device="cuda").manual_seed(0)
    cur = [t.clone() for t in dev]
    for step in range(2):
        cur = [(0.98 * t.float() + 0.2 * torch.randn(t.shape, device="cuda", generator=g)).to(t.dtype) for t in cur]
        O = fwd(*cur, step_kind=b.HVA_INTERMEDIATE).clone()
        torch.cuda.synchronize()
        new = {k: v.clone() for k, v in fwd.state_views().items()}
        c64 = [[inputs.to_f64(t[0, hi]) for hi in range(2)] for t in cur]
        for ti, t in enumerate("qk"):
            for hi in range(2):
                X1 = c64[ti][hi]
                prev = {k: sv[f"{k}_{t}"][hi].cpu().numpy() for k in ("assign", "mu", "sums", "sizes", "subset")}
                a, mo, zo, no, d1, d2 = oracle.subset_update(X1, prev["assign"].astype(np.int64), prev["mu"].astype(np.float64),
                                                             prev["sums"].astype(np.float64), prev["sizes"].astype(np.int64),
                                                             prev["subset"].astype(np.int64), refresh_all=bool(refresh))
                ag = new["assign_" + t][hi].cpu().numpy().astype(np.int64)
                diff = np.nonzero(ag != a)[0]
                pos = {int(tok): k for k, tok in enumerate(prev["subset"])}
                for l in diff:
                    k = pos[int(l)]
                    assert (d2[k] - d1[k]) / max(d1[k], 1e-300) < GAP
                assert np.array_equal(new["subset_" + t][hi].cpu().numpy(), prev["subset"])    # the subset is cached until the next anchor
                if len(diff) == 0:
                    assert np.array_equal(new["sizes_" + t][hi].cpu().numpy(), no)
                    tol = _mu_tol(X1) * 4
                    assert np.abs(new["mu_" + t][hi].cpu().numpy() - mo).max() <= tol + 1e-6 * np.abs(mo).max()
        for hi in range(2):
            check_downstream(wl, fwd, O, hi, [c64[0][hi], c64[1][hi], c64[2][hi]], wl.top_p, wl.merge_rounds, 0.0, 192)
        sv = new
    st = fwd.stats_dicts()
    assert all(s["q_rows_valid"] == wl.n for s in st)


def test_single_candidate_window_with_lowe_ratio():
    """A window of ONE candidate (win = (1,1,1), or a one-cell grid) on the tensor-pipe path with the Lowe ratio requested:
    rho = 0 (R-H1), every token keeps its home cell, sizes sum to n (the second-best score is +inf there, which must not admit
    the pad slots of the 16-wide score tile as contenders)."""
    b = _b()
    for T, H, W, cell, win in ((6, 8, 16, (2, 4, 4), (1, 1, 1)), (3, 5, 8, (3, 5, 8), (3, 3, 3)), (6, 8, 16, (2, 4, 4), (1, 1, 2))):
        wl = dataclasses.replace(inputs.C2, name="nwin1", heads=2, T=T, H=H, W=W, cell=cell, win=win, seed=23)
        (Qd, Kd, _), f64 = _heads(wl, [0, 1])
        shape = b.make_shape(wl, heads=2)
        for iters in (1, 2):
            g = b.hva_cluster(shape, wl.cell, wl.win, iters, Kd, want_lowe=True)
            ref = b.hva_cluster(shape, wl.cell, wl.win, iters, Kd, want_lowe=True, flags=b.HVA_FLAG_CLUSTER_SIMT)
            torch.cuda.synchronize()
            for hi in range(2):
                orc = oracle.local_window_kmeans(f64[1][hi], _lat(wl), wl.cell, wl.win, iters)
                assert np.array_equal(g["assign"][hi].cpu().numpy(), orc["assign"])
                assert np.array_equal(g["sizes"][hi].cpu().numpy(), orc["sizes"]) and int(g["sizes"][hi].sum()) == wl.n
                rho = oracle.lowe_ratio(orc["d1sq"], orc["d2sq"])
                assert np.abs(g["lowe"][hi].cpu().numpy() - rho).max() <= 2e-5
                if math.prod(win) == 1 or cell == (T, H, W):
                    assert float(g["lowe"][hi].abs().max()) == 0.0
            assert torch.equal(g["assign"], ref["assign"])
            if iters == 1:                 # (later passes start from centroids that differ in the last bits between the two kernels)
                assert torch.equal(g["lowe"], ref["lowe"])


def test_cross_check_kernels_agree_with_the_oracle():
    """The CUDA-core cross-check kernels behind HVA_FLAG_* (block-sort mask, bit-loop merge, direct-form subset assignment) against
    the same oracle results as the product kernels: they are independent implementations, not dead code."""
    b = _b()
    wl = inputs.C2
    heads = [2, 6]
    dev, f64 = _heads(wl, heads)
    cl = _oracle_stage_inputs(wl, heads, f64)
    i32 = lambda a: torch.from_numpy(np.ascontiguousarray(a).astype(np.int32)).cuda()
    scale32, p32 = float(np.float32(1.0 / math.sqrt(wl.D))), float(np.float32(0.9))
    mu_q32 = np.stack([c[0]["mu"] for c in cl]).astype(np.float32); mu_k32 = np.stack([c[1]["mu"] for c in cl]).astype(np.float32)
    sizes_q = np.stack([c[0]["sizes"] for c in cl]); sizes_k = np.stack([c[1]["sizes"] for c in cl])
    args = (torch.from_numpy(mu_q32).cuda(), torch.from_numpy(mu_k32).cuda(), i32(sizes_k), scale32, p32)
    M0 = b.hva_build_mask(*args)
    M1 = b.hva_build_mask(*args, flags=b.HVA_FLAG_MASK_BLOCKSORT)
    assert torch.equal(M0, M1)
    for hi in range(2):
        M, margin = oracle.build_mask(mu_q32[hi].astype(np.float64), mu_k32[hi].astype(np.float64), sizes_k[hi], scale32, p32, return_margin=True)
        bad = np.nonzero((M != M1[hi].cpu().numpy()).any(axis=1))[0]
        assert all(margin[r] < 1e-9 for r in bad)
    m0 = b.hva_merge(i32(sizes_q), i32(sizes_k), M0, 128, 128, 3, seed=wl.seed)
    m1 = b.hva_merge(i32(sizes_q), i32(sizes_k), M0, 128, 128, 3, seed=wl.seed, flags=b.HVA_FLAG_MERGE_SIMT)
    for x, y in zip(m0, m1):
        assert torch.equal(x, y)
    for hi in range(2):
        gof, gids, chi = oracle.merge_clusters(sizes_q[hi], sizes_k[hi], M0[hi].cpu().numpy(), 128, 128, 3, seed=wl.seed, bh=hi)
        assert np.array_equal(m1[0][hi].cpu().numpy(), gof) and int(m1[1][hi]) == len(gids)
        assert np.array_equal(m1[2][hi].cpu().numpy()[:len(gids)], chi)


def test_forward_different_q_and_k_grids_wide_windows_min_kc():
    """Paper-setting structure (Table 2, App. A of SURVEY.md): different cell sizes for Q and K (N_q != N_k), (3,8,8)
    windows clipped to the grid (32 and 48 candidates per token: several 32-column TMEM chunks in the assignment kernel),
    min-kc > 0 -- end to end through hva_forward against the oracle's forward pass."""
    b = _b()
    wl = dataclasses.replace(inputs.C2, name="qk-grids", heads=2, T=8, H=16, W=16, seed=31)
    cell_q, cell_k, win = (4, 4, 4), (2, 4, 4), (3, 8, 8)
    Q, K, V = inputs.make_qkv(wl, [0, 1])
    cfg = b.make_config(wl, min_kc=0.15)
    i3 = type(cfg.cell_q)
    cfg.cell_q, cfg.cell_k, cfg.win_q, cfg.win_k = i3(*cell_q), i3(*cell_k), i3(*win), i3(*win)
    fwd = b.Forward(b.make_shape(wl, heads=2), cfg)
    O = fwd(Q.cuda(), K.cuda(), V.cuda())
    torch.cuda.synchronize()
    scale32 = float(np.float32(1.0 / math.sqrt(wl.D)))
    for hi in range(2):
        f = [inputs.to_f64(t[0, hi]) for t in (Q, K, V)]
        r = oracle.forward_head(f[0], f[1], f[2], _lat(wl), cell_q, win, cell_k, win, wl.iters, wl.tile, float(np.float32(wl.top_p)),
                                wl.merge_rounds, seed=wl.seed, bh=hi, min_kc=float(np.float32(0.15)), scale=scale32)
        assert fwd.stats_dicts()[hi]["n_groups"] == len(r["gids"])
        got = O[0, hi].float().cpu().numpy().astype(np.float64)[r["rows"]]
        assert np.abs(got - r["O"]).max() <= 2e-2
        assert np.linalg.norm(got - r["O"]) / np.linalg.norm(r["O"]) <= 1e-2


def test_batch_dimension_is_folded_into_heads():
    """B > 1: every (batch, head) is an independent instance, bh = b * heads + head (also the key of the merge hash):
    the same data viewed as [B=2, heads=2] and as [B=1, heads=4] gives the same bits."""
    b = _b()
    wl = inputs.C2
    Q, K, V = [t.cuda().contiguous() for t in inputs.make_qkv(wl, [0, 1, 2, 3])]
    cfg = b.make_config(wl)
    O4 = b.Forward(b.make_shape(wl, heads=4), cfg)(Q, K, V)
    sh = b.make_shape(wl, heads=2)
    sh.B = 2
    view = lambda t: t.view(2, 2, wl.n, wl.D)
    O22 = b.Forward(sh, cfg)(view(Q), view(K), view(V))
    torch.cuda.synchronize()
    assert torch.equal(O4.view(-1), O22.view(-1))


def test_cluster_qk_two_streams_equals_two_cluster_calls():
    """hva_cluster_qk (Q on the caller's stream, K on the library's side stream, joined by events) == two hva_cluster calls, bit
    for bit, with different Q / K grids; twice in a row with reused buffers; overlapping scratch regions are refused."""
    b = _b()
    wl = inputs.CONFIGS["C2"]
    heads = list(range(8))
    Q, K, _ = inputs.make_qkv(wl, heads=heads)
    Q, K = Q.cuda().contiguous(), K.cuda().contiguous()
    shape = b.make_shape(wl, heads=len(heads))
    cfg = b.make_config(wl)
    cfg.cell_k[0], cfg.cell_k[1], cfg.cell_k[2] = 3, 3, 4
    rq = b.hva_cluster(shape, list(cfg.cell_q), list(cfg.win_q), wl.iters, Q, want_lowe=False)
    rk = b.hva_cluster(shape, list(cfg.cell_k), list(cfg.win_k), wl.iters, K, want_lowe=False)
    bufs = None
    for _ in range(2):
        q, k, bufs = b.hva_cluster_qk(shape, cfg, Q, K, bufs=bufs)
        torch.cuda.synchronize()
        for got, ref in ((q, rq), (k, rk)):
            for key in ("assign", "mu", "sizes", "sums"):
                assert torch.equal(got[key], ref[key]), key
        for d in (q, k):       # the next round must rewrite everything
            d["assign"].fill_(-1); d["mu"].fill_(float("nan"))
    import ctypes as C
    ws = bufs[0]["ws"]
    rc = b.lib().hva_cluster_qk(C.byref(shape), C.byref(cfg), b._p(Q), b._p(K), b._p(q["assign"]), b._p(q["mu"]), b._p(q["sizes"]), b._p(q["sums"]),
                                b._p(k["assign"]), b._p(k["mu"]), b._p(k["sizes"]), b._p(k["sums"]), b._p(ws), C.c_size_t(ws.numel()),
                                b._p(ws), C.c_size_t(ws.numel()), b._stream())
    assert rc == -1


@pytest.mark.parametrize("dtype,D", [("bf16", 64), ("bf16", 128), ("f32", 64), ("f32", 128)])
def test_permute_row_gather_all_row_widths(dtype, D):
    """hva_permute / hva_unpermute against torch indexing for every row width the gather kernel is instantiated for (8, 16 and 32
    16-byte chunks per row), a row count that is not a multiple of the rows one warp moves per iteration, and per-head random
    permutations (bit-exact: byte copies)."""
    b = _b()
    heads, T, H, W = 3, 3, 7, 11                      # n = 231 rows per head
    n = T * H * W
    g = torch.Generator().manual_seed(100 + D + (0 if dtype == "bf16" else 1))
    tdt = torch.bfloat16 if dtype == "bf16" else torch.float32
    X = torch.randn((1, heads, n, D), generator=g, dtype=torch.float32).to(tdt).cuda().contiguous()
    perm = torch.stack([torch.randperm(n, generator=g) for _ in range(heads)]).to(torch.int32).cuda().contiguous()
    shape = b.make_shape((1, heads, T, H, W, D), dtype=dtype)
    Xp = b.hva_permute(shape, X, perm)
    torch.cuda.synchronize()
    ref = torch.stack([X[0, h][perm[h].long()] for h in range(heads)]).unsqueeze(0)
    assert torch.equal(Xp, ref)
    assert torch.equal(b.hva_unpermute(shape, Xp, perm), X)
