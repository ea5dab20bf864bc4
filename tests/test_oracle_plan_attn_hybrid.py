"""Pins for oracle O8 (plan), O9 (attention), O4-O5 (hybrid).  CPU only."""
import math

import numpy as np
import torch

import oracle
from paper_2607_03012_b200 import inputs


def _c1_head(head=0):
    wl = inputs.C1
    Q, K, V = [inputs.to_f64(t) for t in inputs.make_head(wl, head)]
    return wl, Q, K, V


def _fwd(wl, Q, K, V, top_p=None, rounds=None, rows=None):
    return oracle.forward_head(Q, K, V, (wl.T, wl.H, wl.W), wl.cell, wl.win, wl.cell, wl.win, wl.iters, wl.tile,
                               wl.top_p if top_p is None else top_p,
                               wl.merge_rounds if rounds is None else rounds, seed=wl.seed, rows=rows)


def test_plan_bijection_and_segments():
    wl, Q, K, V = _c1_head()
    r = _fwd(wl, Q, K, V)
    p, n = r["plan"], wl.n
    for perm in (p["perm_q"], p["perm_k"]):
        assert sorted(perm.tolist()) == list(range(n))
    assert np.array_equal(p["inv_perm_q"][p["perm_q"]], np.arange(n))
    ak, aq, gof = r["ck"]["assign"], r["cq"]["assign"], r["group_of"]
    assert np.array_equal(np.diff(p["koff"]), r["ck"]["sizes"])
    for j in range(len(r["ck"]["sizes"])):                   # key clusters contiguous, ascending tokens
        seg = p["perm_k"][p["koff"][j]:p["koff"][j + 1]]
        assert (ak[seg] == j).all() and (np.diff(seg) > 0).all()
    for k, g in enumerate(p["gids"]):                        # groups contiguous; clusters inside too
        seg = p["perm_q"][p["goff"][k]:p["goff"][k + 1]]
        assert (gof[aq[seg]] == g).all()
        assert (np.diff(aq[seg]) >= 0).all()
    assert p["goff"][-1] == n and list(p["gids"]) == r["gids"]


def test_attention_vs_dense_masked_softmax_loops():
    wl, Q, K, V = _c1_head(1)
    rows = np.array([0, 17, 100, 255])
    r = _fwd(wl, Q, K, V, rows=rows)
    aq, ak, gof = r["cq"]["assign"], r["ck"]["assign"], r["group_of"]
    chi = {g: r["chi"][k] for k, g in enumerate(r["gids"])}
    scale = 1 / math.sqrt(wl.D)
    for o, l in zip(r["O"], rows):                           # explicit per-element mask as -inf
        s = np.array([float(Q[l] @ K[m]) * scale if chi[gof[aq[l]]][ak[m]] else -np.inf for m in range(wl.n)])
        w = np.exp(s - s.max())
        w /= w.sum()
        assert abs(w.sum() - 1) < 1e-12
        assert np.allclose(o, w @ V, rtol=1e-12, atol=1e-12)
    # union semantics: every query of a merged group sees the OR of its members' rows (Eq. 8)
    for k, g in enumerate(r["gids"]):
        mem = np.where(gof == g)[0]
        assert np.array_equal(r["chi"][k], r["M"][mem].max(0))


def test_top_p_one_is_full_attention():
    wl, Q, K, V = _c1_head()
    r = _fwd(wl, Q, K, V, top_p=1.0)
    ref = torch.nn.functional.scaled_dot_product_attention(
        torch.from_numpy(Q)[None], torch.from_numpy(K)[None], torch.from_numpy(V)[None])[0].numpy()
    assert (r["M"] == 1).all()
    assert np.allclose(r["O"], ref, rtol=1e-11, atol=1e-12)


def test_merge_changes_output_only_through_union_masks():
    wl, Q, K, V = _c1_head()
    a = _fwd(wl, Q, K, V, rounds=0)
    b = _fwd(wl, Q, K, V, rounds=3)
    assert np.array_equal(a["M"], b["M"]) and len(b["gids"]) < len(a["gids"])
    same = [l for l in range(wl.n)
            if np.array_equal(b["chi"][b["gids"].index(b["group_of"][b["cq"]["assign"][l]])],
                              a["M"][a["cq"]["assign"][l]])]
    assert same and np.allclose(a["O"][same], b["O"][same], rtol=1e-12, atol=1e-13)


# ----------------------------------------------------------------------------- hybrid
def test_select_subset_size_order_ties():
    rho = np.array([0.5, 0.9, 0.9, 0.1, 0.9, 0.3, 0.7])
    assert oracle.select_subset(rho, 3 / 7).tolist() == [1, 2, 4]
    assert oracle.select_subset(rho, 2 / 7).tolist() == [1, 2]          # tie -> lower index
    assert oracle.select_subset(rho, 0.5).tolist() == [1, 2, 4, 6]      # floor(3.5 + .5) = 4
    rng = np.random.default_rng(0)
    rho = rng.random(1000)
    sub = oracle.select_subset(rho, 0.15)
    assert len(sub) == 150 and (np.diff(sub) > 0).all()
    rest = np.setdiff1d(np.arange(1000), sub)
    assert rho[rest].max() <= rho[sub].min()


def test_subset_update_f1_refresh_is_global_kmeans_step():
    wl, Q, K, V = _c1_head()
    lat = (wl.T, wl.H, wl.W)
    c = oracle.local_window_kmeans(K, lat, wl.cell, wl.win, 2)
    rng = np.random.default_rng(1)
    X2 = K + 0.3 * rng.standard_normal(K.shape)
    a, mu, z, n, d1, d2 = oracle.subset_update(X2, c["assign"], c["mu"], c["sums"], c["sizes"],
                                               np.arange(wl.n), refresh_all=True)
    d = ((X2[:, None, :] - c["mu"][None]) ** 2).sum(-1)     # textbook global assignment step
    assert np.array_equal(a, d.argmin(1))
    for u in range(8):
        if (a == u).any():
            assert np.allclose(mu[u], X2[a == u].mean(0), rtol=1e-13)
    assert np.array_equal(n, np.bincount(a, minlength=8))
    ds = np.sort(d, axis=1)
    assert np.allclose(d1, ds[:, 0]) and np.allclose(d2, ds[:, 1])


def test_subset_update_noop_and_consistency():
    wl, Q, K, V = _c1_head()
    lat = (wl.T, wl.H, wl.W)
    c = oracle.local_window_kmeans(Q, lat, wl.cell, wl.win, 3)
    # make labels optimal w.r.t. the cached mu (window covers all at C1), then update -> no-op
    a0 = ((Q[:, None, :] - c["mu"][None]) ** 2).sum(-1).argmin(1)
    z0 = np.zeros_like(c["sums"]); np.add.at(z0, a0, Q)
    n0 = np.bincount(a0, minlength=8)
    sub = oracle.select_subset(oracle.lowe_ratio(c["d1sq"], c["d2sq"]), 0.15)
    a, mu, z, n, _, _ = oracle.subset_update(Q, a0, c["mu"], z0, n0, sub)
    assert np.array_equal(a, a0) and np.array_equal(mu, c["mu"]) and np.array_equal(n, n0)
    # perturbed X: non-subset labels untouched, counts consistent, sums adjusted by current x
    rng = np.random.default_rng(3)
    X2 = Q + 0.5 * rng.standard_normal(Q.shape)
    a, mu, z, n, _, _ = oracle.subset_update(X2, c["assign"], c["mu"], c["sums"], c["sizes"], sub)
    rest = np.setdiff1d(np.arange(wl.n), sub)
    assert np.array_equal(a[rest], c["assign"][rest])
    assert np.array_equal(n, np.bincount(a, minlength=8)) and n.sum() == wl.n
    moved = sub[a[sub] != c["assign"][sub]]
    assert len(moved) > 0
    zz = c["sums"].copy()
    for l in moved:
        zz[c["assign"][l]] -= X2[l]; zz[a[l]] += X2[l]
    assert np.allclose(z, zz, rtol=1e-12, atol=1e-12)
    touched = np.unique(np.concatenate([a[moved], c["assign"][moved]]))
    for u in range(8):
        if u in touched and n[u] > 0:
            assert np.allclose(mu[u], z[u] / n[u])
        else:
            assert np.array_equal(mu[u], c["mu"][u])


def test_subset_update_incremental_equals_recomputation_when_x_is_unchanged():
    """Pin of the R-H3 branch (refresh_all=False; P:101 'updating the corresponding centroids'): with UNCHANGED features the
    cached sums are exactly the member sums of the cached labels, so after the subset has been re-assigned against the
    full centroid set the incrementally adjusted sums / sizes / mu of every touched centroid must equal a from-scratch
    recomputation over the NEW labels (and every untouched centroid keeps its members, hence its mean).  The lattice is
    chosen so that the (2,3,3) window does not cover the (2,4,8) grid: local-window labels are not globally optimal and
    subset tokens do move.  A forgotten subtraction, a wrong sign, the wrong feature row or a wrong 'moved' test fails it."""
    import dataclasses
    wl = dataclasses.replace(inputs.C1, name="pin-h3", heads=1, D=64, T=4, H=8, W=16, cell=(2, 2, 2), win=(3, 3, 3), seed=17,
                             noise=0.8)
    X = inputs.to_f64(inputs.make_head(wl, 0)[1])
    lat = (wl.T, wl.H, wl.W)
    c = oracle.local_window_kmeans(X, lat, wl.cell, wl.win, 2)
    Nc = len(c["sizes"])
    assert Nc == 64
    # the cached state is self-consistent: sums = member sums, mu = member means (Alg. 2 l.21-23)
    z0 = np.zeros_like(c["sums"]); np.add.at(z0, c["assign"], X)
    assert np.allclose(z0, c["sums"], rtol=1e-13, atol=1e-13)
    for frac in (0.15, 0.5, 1.0):
        sub = oracle.select_subset(oracle.lowe_ratio(c["d1sq"], c["d2sq"]), frac)
        a, mu, z, n, d1, d2 = oracle.subset_update(X, c["assign"], c["mu"], c["sums"], c["sizes"], sub, refresh_all=False)
        moved = sub[a[sub] != c["assign"][sub]]
        assert len(moved) > 0, "the pin needs tokens that move (window must not cover the grid)"
        # the re-assignment itself: global first minimum for subset tokens, everything else untouched
        dall = ((X[sub][:, None, :] - c["mu"][None]) ** 2).sum(-1)
        assert np.array_equal(a[sub], dall.argmin(1))
        rest = np.setdiff1d(np.arange(wl.n), sub)
        assert np.array_equal(a[rest], c["assign"][rest])
        # from-scratch recomputation over the new labels
        n_ref = np.bincount(a, minlength=Nc)
        z_ref = np.zeros((Nc, wl.D)); np.add.at(z_ref, a, X)
        assert np.array_equal(n, n_ref)
        assert np.allclose(z, z_ref, rtol=1e-12, atol=1e-11)
        touched = np.unique(np.concatenate([a[moved], c["assign"][moved]]))
        for u in range(Nc):
            if n_ref[u] > 0:
                assert np.allclose(mu[u], X[a == u].mean(0), rtol=1e-11, atol=1e-12), u
            if u not in touched:
                assert np.array_equal(mu[u], c["mu"][u])           # untouched centroids are not rewritten
            elif n_ref[u] == 0:
                assert np.array_equal(mu[u], c["mu"][u])           # emptied cluster keeps mu (Alg. 2 l.23)
        # and it agrees with the R-H3' branch on unchanged X (both are then exact member statistics)
        a2, mu2, z2, n2, _, _ = oracle.subset_update(X, c["assign"], c["mu"], c["sums"], c["sizes"], sub, refresh_all=True)
        assert np.array_equal(a2, a) and np.array_equal(n2, n)
        nz = n > 0
        assert np.allclose(mu2[nz], mu[nz], rtol=1e-11, atol=1e-12)
