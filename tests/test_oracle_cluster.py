"""Pins for oracle O1-O4 (grid, local-window k-means, Lowe ratio).  CPU only."""
import itertools

import numpy as np
import pytest

import oracle
from oracle.cluster import init_centroids
from paper_2607_03012_b200 import inputs
from conftest import read_golden


def test_grid_counts_paper():
    g = read_golden("grid_counts.txt")
    for key in ("hunyuan_q", "hunyuan_k", "wan_q", "wan_k"):
        T, H, W, kt, kh, kw, N = [int(v) for v in g[key]]
        K = oracle.grid_dims((T, H, W), (kt, kh, kw))
        assert K[0] * K[1] * K[2] == N
    Nc, wt, wh, ww, red = g["reduction"]
    assert round(Nc / (wt * wh * ww), 1) == red
    assert [21 * 45 * 80, 33 * 45 * 80] == [int(v) for v in g["tokens"]]


@pytest.mark.parametrize("K,w", [(4, 3), (10, 3), (9, 8), (2, 3), (1, 3), (5, 5)])
def test_window_brute_force(K, w):
    """Window = the w consecutive cells containing u that are closest to centred, i.e. start
    u - floor(w/2) shifted into [0, K-w] (Alg. 2 l.369-373): always full size and contains u."""
    wc = min(w, K)
    for u in range(K):
        st = oracle.window_start(u, wc, K)
        cells = list(range(st, st + wc))
        assert len(cells) == wc and 0 <= cells[0] and cells[-1] <= K - 1 and u in cells
        ideal = u - wc // 2
        # brute force: among all valid starts, the one nearest to the ideal start
        best = min(range(0, K - wc + 1), key=lambda s: (abs(s - ideal), s))
        assert st == best


def test_window_ids_order_and_c1_covers_all():
    wl = inputs.C1
    K = oracle.grid_dims((wl.T, wl.H, wl.W), wl.cell)
    win = oracle.clip_window(wl.win, K)
    assert K == (2, 2, 2) and win == (2, 2, 2)
    for u3 in itertools.product(range(2), repeat=3):
        assert oracle.window_ids(u3, win, K) == list(range(8))     # ascending ids, all 8
    ids = oracle.window_ids((5, 4, 3), (3, 3, 3), (11, 9, 10))
    assert ids == sorted(ids) and len(set(ids)) == 27


def test_f1_hand_fixture():
    g = read_golden("f1_cluster.txt")
    X = np.array(g["x"])[:, None]
    lat, cell, win = (1, 1, 8), (1, 1, 2), (1, 1, 3)
    assert np.array_equal(init_centroids(X, lat, cell)[:, 0], g["mu0"])
    r1 = oracle.local_window_kmeans(X, lat, cell, win, 1)
    assert r1["assign"].tolist() == g["assign1"]
    assert r1["sizes"].tolist() == g["sizes1"]
    assert r1["J"] == g["J1"]
    assert np.allclose(r1["mu"][:, 0], g["mu1"], rtol=0, atol=1e-15)
    assert np.allclose(oracle.lowe_ratio(r1["d1sq"], r1["d2sq"]), g["rho1"], rtol=1e-15)
    r2 = oracle.local_window_kmeans(X, lat, cell, win, 2)
    assert r2["assign"].tolist() == g["assign2"]
    assert r2["J"] == g["J1"] + g["J2"]
    assert np.allclose(r2["mu"][:, 0], g["mu2"])


def _brute_assign(X, mu, lattice, cell, win):
    """Exhaustive argmin over ALL centroids with the non-window ones masked to +inf."""
    T, H, W = lattice
    K = oracle.grid_dims(lattice, cell)
    win = oracle.clip_window(win, K)
    out = np.empty(len(X), dtype=np.int64)
    for t in range(T):
        for h in range(H):
            for w in range(W):
                l = (t * H + h) * W + w
                g = (t // cell[0], h // cell[1], w // cell[2])
                best, arg = np.inf, -1
                for u in range(mu.shape[0]):
                    u3 = (u // (K[1] * K[2]), (u // K[2]) % K[1], u % K[2])
                    ok = all(abs(0) == 0 and oracle.window_start(g[a], win[a], K[a]) <= u3[a]
                             < oracle.window_start(g[a], win[a], K[a]) + win[a] for a in range(3))
                    d = float(((X[l] - mu[u]) ** 2).sum()) if ok else np.inf
                    if d < best:
                        best, arg = d, u
                out[l] = arg
    return out


@pytest.mark.parametrize("lat,cell,win", [((4, 6, 7), (2, 2, 3), (3, 3, 3)), ((3, 5, 9), (1, 2, 2), (3, 2, 4))])
def test_assignment_vs_brute_force_and_invariants(lat, cell, win):
    rng = np.random.default_rng(5)
    n = lat[0] * lat[1] * lat[2]
    X = rng.standard_normal((n, 6))
    prev = None
    for it in (1, 2, 3):
        r = oracle.local_window_kmeans(X, lat, cell, win, it)
        mu_before = init_centroids(X, lat, cell) if prev is None else prev["mu"]
        assert np.array_equal(r["assign"], _brute_assign(X, mu_before, lat, cell, win))
        assert r["sizes"].sum() == n and np.array_equal(r["sizes"], np.bincount(r["assign"], minlength=len(r["sizes"])))
        for u in range(len(r["sizes"])):                       # mu = mean of members, empty keeps
            if r["sizes"][u]:
                assert np.allclose(r["mu"][u], X[r["assign"] == u].mean(0), rtol=1e-13, atol=1e-13)
            else:
                assert np.array_equal(r["mu"][u], mu_before[u])
        prev = r
    assert all(a >= b - 1e-9 for a, b in zip(r["J"], r["J"][1:]))    # objective non-increasing
    rho = oracle.lowe_ratio(r["d1sq"], r["d2sq"])
    assert (rho >= 0).all() and (rho <= 1).all()


def test_c1_is_textbook_lloyd_step():
    """At C1 the clipped window covers the whole grid: one iteration == a textbook global
    Lloyd step (argmin over all centroids, then means)."""
    wl = inputs.C1
    X = inputs.to_f64(inputs.make_head(wl, 1)[0])
    lat = (wl.T, wl.H, wl.W)
    mu = init_centroids(X, lat, wl.cell)
    for it in range(1, 4):
        r = oracle.local_window_kmeans(X, lat, wl.cell, wl.win, it)
        d = ((X[:, None, :] - mu[None]) ** 2).sum(-1)
        lab = d.argmin(1)
        assert np.array_equal(r["assign"], lab)
        mu = np.stack([X[lab == u].mean(0) if (lab == u).any() else mu[u] for u in range(8)])
        assert np.allclose(r["mu"], mu, rtol=1e-13, atol=1e-13)
    assert r["J"][0] >= r["J"][1] >= r["J"][2]


def test_empty_cluster_keeps_mu():
    # 1-D lattice W=4, cell 1 -> 4 centroids = the tokens themselves; token 1 sits exactly on
    # token 0's value so centroid 1 ties with centroid 0 and loses (first minimum) -> empty.
    X = np.array([[0.0], [0.0], [5.0], [9.0]])
    r = oracle.local_window_kmeans(X, (1, 1, 4), (1, 1, 1), (1, 1, 3), 1)
    assert r["assign"].tolist() == [0, 0, 2, 3]
    assert r["sizes"].tolist() == [2, 0, 1, 1]
    assert r["mu"][1, 0] == 0.0                                  # kept (Alg. 2 line 23)


def test_lowe_independent_top2():
    wl = inputs.C1
    X = inputs.to_f64(inputs.make_head(wl, 0)[1])
    lat = (wl.T, wl.H, wl.W)
    r = oracle.local_window_kmeans(X, lat, wl.cell, wl.win, 1)
    mu0 = init_centroids(X, lat, wl.cell)
    d = np.sqrt(((X[:, None, :] - mu0[None]) ** 2).sum(-1))
    d.sort(axis=1)
    assert np.allclose(oracle.lowe_ratio(r["d1sq"], r["d2sq"]), d[:, 0] / d[:, 1], rtol=1e-12)
    assert oracle.lowe_ratio([1.0], [np.inf])[0] == 0.0 and oracle.lowe_ratio([0.0], [0.0])[0] == 1.0
