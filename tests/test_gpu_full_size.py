"""GPU parity at the sizes the kernels actually run at (BASELINE.json configs[2..4]).

The small-size tests (test_gpu_parity.py) never reach: the persistent multi-tile path of the assignment kernel
(n_items > 4 x 148 CTAs), the <128,32> mask instantiation and the 8-block merge contraction (N_k > 512), the ring
wrap-around / TMEM buffer reuse of the subset kernel (N_c > 256), the 116-pass radix select at n = 118 800, the block-sort mask
kernel with top-p < 1 (N_k > 1024: the paper's K grid).  Here every one of them is compared with the fp64 oracle:
labels under the R-C10 gap rule (each differing token must be a near tie holding the oracle's runner-up), masks / merge
plans / permutations bit for bit, attention on sampled query rows within BASELINE.json's tolerance.

hva_forward is checked as a chain: GPU iteration i (hva_cluster with iters = i, same kernels, same bits as inside
hva_forward) against ONE oracle iteration started from the GPU's own mu^(i-1), so that a legitimate near-tie flip cannot
hide a real error downstream of it; everything after clustering is compared with the oracle re-run from the GPU's own
clustering result (read from the state buffer), the mask / merge / plan arrays being read back from the workspace
(hva_workspace_describe)."""
import dataclasses
import functools
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


def _lat(wl):
    return (wl.T, wl.H, wl.W)


@functools.lru_cache(maxsize=2)
def _device_inputs(name):
    """All heads of a full-size config, resident on the device (the launch configuration bench.py times)."""
    wl = inputs.CONFIGS[name]
    return [t.cuda().contiguous() for t in inputs.make_qkv(wl)]


def _mu_err_units(got, ref, X):
    """max |got - ref| in units of 2^-24 max|x| (printed: the observed accuracy of the fixed-order fp32 sums)."""
    return float(np.abs(got - ref).max() / (2.0 ** -24 * np.abs(X).max()))


def check_labels(lab_gpu, X, orc, mu_used):
    """Bit-exact except near ties: a differing token must have oracle gap < 1e-5 and hold the runner-up (R-C10)."""
    diff = np.nonzero(lab_gpu != orc["assign"])[0]
    for l in diff:
        gap = (orc["d2sq"][l] - orc["d1sq"][l]) / max(orc["d1sq"][l], 1e-300)
        d_g = float(((X[l] - mu_used[lab_gpu[l]]) ** 2).sum())
        assert gap < GAP, f"token {l}: labels differ with gap {gap:.3e}"
        assert abs(d_g - orc["d2sq"][l]) <= 1e-9 * max(1.0, orc["d2sq"][l]), f"token {l}: not the runner-up"
    return diff


def cluster_chain(b, wl, Xd1, X64, cell, win, iters, mu_tol_units=4.0):
    """GPU iterations 1..iters of one (head, tensor), each checked against one oracle iteration from the GPU's own
    previous centroids.  Xd1: [1,1,n,D] device tensor.  Returns the final GPU result and the number of exempt flips."""
    shape1 = b.make_shape(wl, heads=1)
    lat = _lat(wl)
    mu_in = oracle.cluster.init_centroids(X64, lat, cell)
    flips, worst = 0, 0.0
    g = None
    for i in range(1, iters + 1):
        g = b.hva_cluster(shape1, cell, win, i, Xd1, want_lowe=(i == iters))
        torch.cuda.synchronize()
        orc = oracle.local_window_kmeans(X64, lat, cell, win, 1, mu_init=mu_in)
        lab = g["assign"][0].cpu().numpy().astype(np.int64)
        diff = check_labels(lab, X64, orc, mu_in)
        flips += len(diff)
        sz = g["sizes"][0].cpu().numpy()
        assert sz.sum() == wl.n and np.array_equal(sz, np.bincount(lab, minlength=len(sz)))
        touched = set(lab[diff]) | set(orc["assign"][diff])
        keep = np.array([u not in touched for u in range(len(sz))])
        assert np.array_equal(sz[keep], orc["sizes"][keep])
        mg = g["mu"][0].cpu().numpy().astype(np.float64)
        e = _mu_err_units(mg[keep], orc["mu"][keep], X64)
        worst = max(worst, e)
        assert e <= mu_tol_units, f"iteration {i}: centroid error {e:.1f} x 2^-24 max|x|"
        if i == iters:
            rho = oracle.lowe_ratio(orc["d1sq"], orc["d2sq"])
            same = lab == orc["assign"]
            assert np.abs(g["lowe"][0].cpu().numpy()[same] - rho[same]).max() <= 2e-5
        mu_in = mg                                            # the GPU's own fp32 centroids, widened exactly
    print(f"[cluster_chain] {wl.name} cell={tuple(cell)} win={tuple(win)}: exempt flips {flips}, centroid error {worst:.2f} x 2^-24 max|x|")
    return g, flips


def check_attention_rows(wl, Q64, K64, V64, O_head, aq, ak, gof, gids, chi, rows):
    scale32 = float(np.float32(1.0 / math.sqrt(wl.D)))
    ref = oracle.masked_attention_rows(Q64, K64, V64, rows, aq, ak, gof, gids, chi, scale32)
    got = O_head[torch.from_numpy(rows).to(O_head.device)].float().cpu().numpy().astype(np.float64)
    rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    mx = np.abs(got - ref).max()
    assert mx <= 2e-2 and rel <= 1e-2, (mx, rel)             # BASELINE.json north_star, bf16
    return mx, rel


def check_downstream(wl, fwd, O, hi, f64, top_p, rounds, min_kc, rows_per_head):
    """Everything after clustering of head `hi` of the last sparse hva_forward call, against the oracle re-run from the GPU's
    own clustering result (state buffer): mask, merge, plan read back from the workspace bit for bit; attention on sampled rows."""
    sv, wv, st = fwd.state_views(), fwd.ws_views(), fwd.stats_dicts()
    Nq, Nk = sv["sizes_q"].shape[1], sv["sizes_k"].shape[1]
    aq = sv["assign_q"][hi].cpu().numpy().astype(np.int64)
    ak = sv["assign_k"][hi].cpu().numpy().astype(np.int64)
    sq, sk = np.bincount(aq, minlength=Nq), np.bincount(ak, minlength=Nk)
    assert np.array_equal(sq, sv["sizes_q"][hi].cpu().numpy()) and np.array_equal(sk, sv["sizes_k"][hi].cpu().numpy())
    # S5 mask, bit for bit (rows whose cut lies within 1e-9 Z of the threshold are exempt, R-K3)
    scale32, p32 = float(np.float32(1.0 / math.sqrt(wl.D))), float(np.float32(top_p))
    M, margin = oracle.build_mask(sv["mu_q"][hi].cpu().numpy().astype(np.float64), sv["mu_k"][hi].cpu().numpy().astype(np.float64),
                                  sk, scale32, p32, float(np.float32(min_kc)), return_margin=True)
    Mg = wv["mask"][hi].cpu().numpy()
    bad = np.nonzero((M != Mg).any(axis=1))[0]
    assert all(margin[r] < 1e-9 for r in bad), f"mask rows differ away from the threshold: {bad[:5]}"
    # S6 merge, bit for bit (fed the GPU's mask, so that an exempt mask row cannot masquerade as a merge error)
    gof, gids, chi = oracle.merge_clusters(sq, sk, Mg, wl.tile[0], wl.tile[1], rounds, seed=wl.seed, bh=hi)
    ng = len(gids)
    assert int(wv["n_groups"][hi]) == ng == st[hi]["n_groups"]
    assert np.array_equal(wv["group_of"][hi].cpu().numpy(), gof)
    gm = wv["group_mask"][hi].cpu().numpy()
    assert np.array_equal(gm[:ng], chi) and not gm[ng:].any()
    # S7 plan, bit for bit
    po = oracle.build_plan(aq, ak, gof, Nq, Nk)
    pl = wv["plan"]
    for k in ("perm_q", "inv_perm_q", "perm_k", "koff"):
        assert np.array_equal(getattr(pl, k)[hi].cpu().numpy(), po[k]), k
    assert np.array_equal(pl.gid[hi].cpu().numpy()[:ng], po["gids"]) and np.array_equal(pl.goff[hi].cpu().numpy()[:ng + 1], po["goff"])
    kap = (chi.astype(np.int64) * sk[None, :]).sum(1)
    assert np.array_equal(pl.kappa[hi].cpu().numpy()[:ng], kap)
    rows_g = np.diff(po["goff"])
    assert st[hi]["k_cols_valid"] == int(kap.sum()) and st[hi]["pairs_valid"] == int((rows_g * kap).sum())
    assert st[hi]["tiles_executed"] == int((-(-rows_g // wl.tile[0]) * -(-kap // wl.tile[1])).sum())
    # S9 + S10 attention on sampled query rows: rows of merged groups, of multi-tile groups and of ragged tails included
    rng = np.random.default_rng(hi)
    rows = np.sort(rng.choice(wl.n, rows_per_head, replace=False))
    if rounds > 0:
        multi = np.nonzero(rows_g > wl.tile[0])[0]
        if len(multi):
            k = int(multi[0])
            rows = np.unique(np.concatenate([rows, po["perm_q"][[po["goff"][k], po["goff"][k + 1] - 1]]]))
    mx, rel = check_attention_rows(wl, f64[0], f64[1], f64[2], O[0, hi], aq, ak, gof, gids, chi, rows)
    return ng, len(bad), mx, rel, len(rows)


def forward_full_check(wl_name, check_head, rows_per_head, top_p=None, rounds=None, cells=None, min_kc=0.0, chain=True, heads=None):
    """hva_forward on the full call; the checked head against the oracle, stage by stage, bit for bit."""
    b = _b()
    wl = inputs.CONFIGS[wl_name]
    Q, K, V = _device_inputs(wl_name)
    if heads is not None:
        Q, K, V = [t[:, heads].contiguous() for t in (Q, K, V)]
    nh = Q.shape[1]
    top_p = wl.top_p if top_p is None else top_p
    rounds = wl.merge_rounds if rounds is None else rounds
    cfg = b.make_config(wl, top_p=top_p, merge_rounds=rounds, min_kc=min_kc)
    cell_q, cell_k, win_q, win_k = wl.cell, wl.cell, wl.win, wl.win
    if cells is not None:
        cell_q, cell_k, win_q, win_k = cells
        i3 = type(cfg.cell_q)
        cfg.cell_q, cfg.cell_k, cfg.win_q, cfg.win_k = i3(*cell_q), i3(*cell_k), i3(*win_q), i3(*win_k)
    shape = b.make_shape(wl, heads=nh)
    fwd = b.Forward(shape, cfg, with_state=True)
    O = fwd(Q, K, V)
    torch.cuda.synchronize()
    sv, wv, st = fwd.state_views(), fwd.ws_views(), fwd.stats_dicts()
    Nq, Nk = sv["sizes_q"].shape[1], sv["sizes_k"].shape[1]
    for s in st:                                              # properties that hold at any size, every head
        assert s["q_rows_valid"] == wl.n and 0 < s["n_groups"] <= Nq
        assert s["pairs_valid"] <= wl.n * wl.n and s["q_rows_padded"] >= wl.n
    assert torch.isfinite(O.float()).all()
    hi = check_head
    f64 = [inputs.to_f64(t[0, hi]) for t in (Q, K, V)]
    aq = sv["assign_q"][hi].cpu().numpy().astype(np.int64)
    ak = sv["assign_k"][hi].cpu().numpy().astype(np.int64)
    flips = 0
    if chain:                                                 # S0-S2: every GPU iteration is a correct iteration (R-C10)
        for which, cell, win, lab in ((0, cell_q, win_q, aq), (1, cell_k, win_k, ak)):
            Xd1 = (Q, K)[which][:, hi:hi + 1].contiguous()
            g, f = cluster_chain(b, wl, Xd1, f64[which], cell, win, wl.iters)
            flips += f
            t = "qk"[which]
            assert np.array_equal(g["assign"][0].cpu().numpy(), lab)                       # hva_forward ran exactly this
            assert torch.equal(g["mu"][0], sv["mu_" + t][hi]) and torch.equal(g["sizes"][0], sv["sizes_" + t][hi])
    ng, nbad, mx, rel, nrows = check_downstream(wl, fwd, O, hi, f64, top_p, rounds, min_kc, rows_per_head)
    print(f"[forward_full_check] {wl.name} head {hi} p={top_p} R={rounds}: groups {ng}, exempt flips {flips}, mask rows exempt {nbad}, "
          f"attention max-abs {mx:.2e} rel-L2 {rel:.2e} on {nrows} rows")
    return fwd, O, flips


# ----------------------------------------------------------------------------- full-size calls (bench launch configuration)
def test_c4_full_call_every_stage_bit_exact():
    """C4 (HunyuanVideo shape, all 24 heads resident, what bench.py times)."""
    fwd, O, flips = forward_full_check("C4", check_head=5, rows_per_head=48)
    Q, K, V = _device_inputs("C4")
    assert torch.equal(fwd(Q, K, V), O)                       # deterministic at full size


def test_c3_full_call_every_stage_bit_exact():
    """C3 (Wan shape, 40 heads x 75 600 tokens, 630 clusters): second lattice; 1024-wide register sort with 394 pads,
    5-block merge contraction."""
    forward_full_check("C3", check_head=17, rows_per_head=32)


@pytest.mark.parametrize("top_p,rounds", [(0.8, 0), (0.8, 3), (0.95, 0), (0.95, 3)])
def test_c4_sweep_cells(top_p, rounds):
    """BASELINE.json configs[3]: top-p {0.8, 0.95} x merging {off, on} at full size (the 0.9 cells are the tests above / below);
    clustering is the same in every cell and chain-checked once above."""
    forward_full_check("C4", check_head=11, rows_per_head=24, top_p=top_p, rounds=rounds, chain=False)


def test_c4_merge_off():
    forward_full_check("C4", check_head=2, rows_per_head=24, rounds=0, chain=False)


def test_c4_paper_grids_wide_windows_min_kc():
    """The paper's HunyuanVideo hyper-parameters on the C4 lattice (Table 2): Q grid (11,5,5) -> 432 clusters of 275 tokens
    (split over three CTA tiles), K grid (11,3,3) -> 1215 clusters (N_k > 1024: the block-sort mask kernel with top-p < 1),
    (3,8,8) windows = 192 candidates (six 32-column TMEM chunks), min-kc 0.15 -- four heads resident, one checked end to end."""
    cells = ((11, 5, 5), (11, 3, 3), (3, 8, 8), (3, 8, 8))
    forward_full_check("C4", check_head=1, rows_per_head=24, cells=cells, min_kc=0.15, heads=[0, 7, 13, 22])


# ----------------------------------------------------------------------------- persistent multi-tile assignment path
@pytest.mark.parametrize("which", [0, 1])
def test_assign_persistent_path_teacher_forced_c2_8_heads(which):
    """C2 x 8 heads = 1152 tiles > 4 x 148 resident CTAs: CTAs draw further tiles from the device counter and issue the next
    tile's boxes under the epilogue.  Teacher-forced by the ORACLE's centroids, every head checked (R-C10)."""
    from test_gpu_parity import run_cluster_parity
    flips = run_cluster_parity(inputs.C2, list(range(8)), which)
    assert flips <= 8


def test_assign_persistent_path_c4_head_pair():
    """A head pair of C4 (1980 tiles), Q and K: the GPU chain against the oracle, every iteration."""
    b = _b()
    wl = inputs.C4
    Q, K, V = _device_inputs("C4")
    shape2 = b.make_shape(wl, heads=2)
    for which, X in ((0, Q), (1, K)):
        Xd = X[:, [3, 20]].contiguous()
        both = b.hva_cluster(shape2, wl.cell, wl.win, wl.iters, Xd)
        for j in range(2):
            g, _ = cluster_chain(b, wl, Xd[:, j:j + 1].contiguous(), inputs.to_f64(Xd[0, j]), wl.cell, wl.win, wl.iters)
            for k in ("assign", "mu", "sizes", "sums", "lowe"):       # a head's bits do not depend on its neighbours in the launch
                assert torch.equal(g[k][0], both[k][j]), k


# ----------------------------------------------------------------------------- hybrid step at the size it is specified for
@pytest.mark.parametrize("head", [0, 9])
def test_c5_hybrid_step_full_size(head):
    """BASELINE.json configs[4]: n = 118 800, m = 17 820, N_c = 990 -- 8 candidate tiles through the 2-stage
    ring and both TMEM score buffers of hva_subset_assign_tc_kernel, 116 passes of the radix select.  S3 bit-exact on identical
    fp32 rho (with a block of exact ties straddling the threshold), S4 (R-H3 and R-H3') under the gap rule over all N_c."""
    b = _b()
    wl = inputs.C5
    n, lat = wl.n, _lat(wl)
    m = int(math.floor(0.15 * n + 0.5))
    assert m == 17820
    x0 = inputs.make_head(wl, head, 0)
    rms0 = x0.float().pow(2).mean(dim=(1, 2)).sqrt()
    x1 = inputs.hybrid_next(wl, x0, head, 1, rms0)
    shape1 = b.make_shape(wl, heads=1)
    for which in (0, 1):
        X0, X1 = inputs.to_f64(x0[which]), inputs.to_f64(x1[which])
        orc = oracle.local_window_kmeans(X0, lat, wl.cell, wl.win, wl.iters)
        Nc = len(orc["sizes"])
        rho32 = oracle.lowe_ratio(orc["d1sq"], orc["d2sq"]).astype(np.float32)
        # S3, as the oracle produced it and with exact ties around the m-th value
        for ties in (False, True):
            r = rho32.copy()
            if ties:
                thr = np.sort(r)[::-1][m - 1]
                near = np.argsort(np.abs(r - thr))[:2000]
                r[near] = thr
            sub_g = b.hva_select_subset(torch.from_numpy(r[None]).cuda(), m)[0].cpu().numpy()
            sub_o = oracle.select_subset(r.astype(np.float64), 0.15)
            assert np.array_equal(sub_g, sub_o), f"subset differs (ties={ties})"
        sub_o = oracle.select_subset(rho32.astype(np.float64), 0.15)
        # S4 on the next step's features, cached oracle state rounded to fp32
        Xd = x1[which][None, None].cuda().contiguous()
        mu32, z32 = orc["mu"].astype(np.float32), orc["sums"].astype(np.float32)
        for refresh in (0, 1):
            assign = torch.from_numpy(orc["assign"].astype(np.int32))[None].cuda()
            mu, sums = torch.from_numpy(mu32)[None].cuda(), torch.from_numpy(z32)[None].cuda()
            sizes = torch.from_numpy(orc["sizes"].astype(np.int32))[None].cuda()
            b.hva_cluster_update(shape1, Xd, torch.from_numpy(sub_o.astype(np.int32))[None].cuda(), assign, mu, sums, sizes, refresh)
            torch.cuda.synchronize()
            a, mo, zo, no, d1, d2 = oracle.subset_update(X1, orc["assign"], mu32.astype(np.float64), z32.astype(np.float64),
                                                         orc["sizes"], sub_o, refresh_all=bool(refresh))
            ag = assign[0].cpu().numpy().astype(np.int64)
            diff = np.nonzero(ag != a)[0]
            pos = {int(t): k for k, t in enumerate(sub_o)}
            for l in diff:                                            # near-tie rule over all N_c candidates
                k = pos[int(l)]
                assert (d2[k] - d1[k]) / max(d1[k], 1e-300) < GAP, f"token {l}"
                assert abs(float(((X1[l] - mu32[ag[l]].astype(np.float64)) ** 2).sum()) - d2[k]) <= 1e-9 * max(1.0, d2[k])
            rest = np.setdiff1d(np.arange(n), sub_o)
            assert np.array_equal(ag[rest], orc["assign"][rest])      # non-subset labels untouched
            moved = int((a[sub_o] != orc["assign"][sub_o]).sum())
            assert moved > 100                                        # the step does something at this size
            touched = set(ag[diff]) | set(a[diff]) | set(orc["assign"][diff])
            keep = np.array([u not in touched for u in range(Nc)])
            sg = sizes[0].cpu().numpy()
            assert sg.sum() == n and np.array_equal(sg[keep], no[keep])
            e_mu = _mu_err_units(mu[0].cpu().numpy()[keep], mo[keep], X1)
            e_z = _mu_err_units(sums[0].cpu().numpy()[keep], zo[keep], X1) / max(1, int(no.max()))
            print(f"[c5 hybrid] head {head} tensor {'QK'[which]} refresh {refresh}: moved {moved}, exempt {len(diff)}, "
                  f"mu err {e_mu:.2f}, sums err/size {e_z:.2f} (x 2^-24 max|x|)")
            assert e_mu <= 4.0 and e_z <= 4.0


# ----------------------------------------------------------------------------- N_k > 1024 through the stage entry points
def test_mask_merge_plan_paper_cluster_counts():
    """N_q = 432, N_k = 1215 (the paper's HunyuanVideo counts) with seeded centroids and sizes through hva_build_mask (block-sort
    kernel, top-p < 1, with and without min-kc) -> hva_merge -> hva_build_plan, bit for bit against the oracle."""
    b = _b()
    rng = np.random.default_rng(41)
    BH, Nq, Nk, D, n = 2, 432, 1215, 128, 118800
    base = rng.standard_normal((BH, 16, D))
    mu_q = (base[:, rng.integers(0, 16, Nq)] + 0.6 * rng.standard_normal((BH, Nq, D))).astype(np.float32)
    mu_k = (base[:, rng.integers(0, 16, Nk)] + 0.6 * rng.standard_normal((BH, Nk, D))).astype(np.float32)
    aq = rng.integers(0, Nq, size=(BH, n)); ak = rng.integers(0, Nk, size=(BH, n))
    ak[:, : n // 3] = ak[:, : n // 3] % 200                    # uneven key clusters, a few empty ones
    ak[ak == 77] = 78
    sizes_q = np.stack([np.bincount(a, minlength=Nq) for a in aq]); sizes_k = np.stack([np.bincount(a, minlength=Nk) for a in ak])
    assert (sizes_k == 0).any()
    i32 = lambda a: torch.from_numpy(np.ascontiguousarray(a).astype(np.int32)).cuda()
    scale32 = float(np.float32(1.0 / math.sqrt(D)))
    for top_p, min_kc in ((0.9, 0.0), (0.9, 0.15), (0.5, 0.0)):
        p32, kc32 = float(np.float32(top_p)), float(np.float32(min_kc))
        Mg = b.hva_build_mask(torch.from_numpy(mu_q).cuda(), torch.from_numpy(mu_k).cuda(), i32(sizes_k), scale32, p32, kc32).cpu().numpy()
        for hi in range(BH):
            M, margin = oracle.build_mask(mu_q[hi].astype(np.float64), mu_k[hi].astype(np.float64), sizes_k[hi], scale32, p32, kc32,
                                          return_margin=True)
            bad = np.nonzero((M != Mg[hi]).any(axis=1))[0]
            assert all(margin[r] < 1e-9 for r in bad), (top_p, min_kc, bad[:5])
            assert 0 < M.sum() < M.size
        gof_g, ng_g, gm_g = b.hva_merge(i32(sizes_q), i32(sizes_k), torch.from_numpy(Mg).cuda(), 128, 128, 3, seed=7)
        plan = b.hva_build_plan(n, i32(aq), i32(ak), i32(sizes_q), i32(sizes_k), gof_g, ng_g, gm_g, 128, 128)
        torch.cuda.synchronize()
        for hi in range(BH):
            gof, gids, chi = oracle.merge_clusters(sizes_q[hi], sizes_k[hi], Mg[hi], 128, 128, 3, seed=7, bh=hi)
            assert np.array_equal(gof_g[hi].cpu().numpy(), gof) and int(ng_g[hi]) == len(gids)
            gm = gm_g[hi].cpu().numpy()
            assert np.array_equal(gm[:len(gids)], chi) and not gm[len(gids):].any()
            po = oracle.build_plan(aq[hi], ak[hi], gof, Nq, Nk)
            for k in ("perm_q", "inv_perm_q", "perm_k", "koff"):
                assert np.array_equal(getattr(plan, k)[hi].cpu().numpy(), po[k]), k
            assert np.array_equal(plan.goff[hi].cpu().numpy()[:len(gids) + 1], po["goff"])


def test_c4_forward_is_deterministic_and_ignores_stale_workspace():
    """The whole C4 call three times on the same inputs, the workspace filled with random bytes in between: the output, the mask, the
    merge result and every meaningful array of the plan are the same bits each time (no floating-point atomics, no dependence on
    what a previous call -- or anybody else -- left in the workspace, no race between the two streams the call runs on)."""
    b = _b()
    wl = inputs.CONFIGS["C4"]
    Q, K, V = _device_inputs("C4")
    shape, cfg = b.make_shape(wl), b.make_config(wl)
    fwd = b.Forward(shape, cfg)
    ref = None
    for it in range(3):
        O = torch.empty_like(Q)
        fwd(Q, K, V, O)
        torch.cuda.synchronize()
        views = fwd.ws_views()
        pl, ng = views["plan"], views["n_groups"]
        snap = [O.clone()] + [v.clone() for v in views.values() if torch.is_tensor(v)]
        snap += [getattr(pl, k).clone() for k in ("perm_q", "inv_perm_q", "perm_k", "koff", "stats")]
        for h in range(0, pl.BH, 5):
            g, wc = int(ng[h]), int(pl.work_cnt[h])
            snap += [pl.gid[h, :g].clone(), pl.goff[h, :g + 1].clone(), pl.kappa[h, :g].clone(), pl.run_cnt[h, :g].clone(),
                     pl.work[h, :wc].clone()]
        if ref is None:
            ref = snap
        else:
            for i, (x, y) in enumerate(zip(ref, snap)):
                assert torch.equal(x, y), (it, i)
        fwd.ws.random_(0, 255)
