"""Oracle O2-O4: 3D local-window k-means and Lowe's ratio (test infrastructure, fp64).

Follows PAPER.md Alg. 2 (l.346-388) step by step: centre-token init (lines 7-11), then
N_iter Jacobi passes of {reset z,n; per home cell: local argmin, accumulate; update mu}
(lines 12-23); Eq. 5 (l.81) for the assignment, Eq. 6 (l.97) for Lowe's ratio.

Readings: R-C1 first minimum in ascending centroid id; R-C2 shifted full-size
window; R-C5 centroids never rounded; R-C7 empty cluster keeps mu; R-H1 rho from the
window-restricted distances of the LAST pass, unsquared ratio.

Pinned by (tests/test_oracle_cluster.py): the hand fixture F1 (tests/golden/f1_cluster.txt),
exhaustive all-centroid argmin with non-window centroids masked, a textbook Lloyd step
when the window covers the grid, mu == independently recomputed member means, an
empty-cluster construction, J non-increasing, sum of sizes == n.
"""
from __future__ import annotations

import numpy as np

from .grid import grid_dims, clip_window, centre_token, window_ids


def _cell_tokens(u3, cell, lattice):
    T, H, W = lattice
    ts = range(u3[0] * cell[0], min((u3[0] + 1) * cell[0], T))
    hs = range(u3[1] * cell[1], min((u3[1] + 1) * cell[1], H))
    ws = range(u3[2] * cell[2], min((u3[2] + 1) * cell[2], W))
    return np.array([(t * H + h) * W + w for t in ts for h in hs for w in ws], dtype=np.int64)


def init_centroids(X, lattice, cell):
    """mu_u <- X[c_t, c_h, c_w, :]   (Alg. 2 lines 7-11, l.357-363)."""
    T, H, W = lattice
    K = grid_dims(lattice, cell)
    mu = np.empty((K[0] * K[1] * K[2], X.shape[1]), dtype=np.float64)
    for ut in range(K[0]):
        for uh in range(K[1]):
            for uw in range(K[2]):
                ct = centre_token(ut, cell[0], T)
                ch = centre_token(uh, cell[1], H)
                cw = centre_token(uw, cell[2], W)
                mu[(ut * K[1] + uh) * K[2] + uw] = X[(ct * H + ch) * W + cw]
    return mu


def local_window_kmeans(X, lattice, cell, win, iters, mu_init=None):
    """X: [n, D] float64 tokens of one (batch, head) in (t,h,w) row-major order.

    Returns dict: assign [n] int64 (last pass), mu [Nc, D] (AFTER the last update, Alg. 2
    line 24), sizes [Nc] int64, sums [Nc, D] (z of the last pass), d1sq / d2sq [n] (nearest / second-nearest squared distance of
    the last pass, within the window), J (list of per-iteration objectives sum d1sq).
    """
    X = np.asarray(X, dtype=np.float64)
    n, D = X.shape
    K = grid_dims(lattice, cell)
    win = clip_window(win, K)
    Nc = K[0] * K[1] * K[2]
    mu = init_centroids(X, lattice, cell) if mu_init is None else np.array(mu_init, dtype=np.float64)
    assert mu.shape == (Nc, D)
    cells = [(ut, uh, uw) for ut in range(K[0]) for uh in range(K[1]) for uw in range(K[2])]
    toks = [_cell_tokens(u3, cell, lattice) for u3 in cells]
    cands = [np.array(window_ids(u3, win, K), dtype=np.int64) for u3 in cells]
    assign = np.zeros(n, dtype=np.int64)
    d1sq = np.zeros(n)
    d2sq = np.zeros(n)
    J = []
    for _ in range(iters):
        z = np.zeros((Nc, D))
        cnt = np.zeros(Nc, dtype=np.int64)
        for tk, cd in zip(toks, cands):                       # Alg. 2 line 14 "for each grid u"
            diff = X[tk][:, None, :] - mu[cd][None, :, :]     # [tokens, candidates, D]
            d2 = np.einsum("tcd,tcd->tc", diff, diff)         # ||x - mu_v||^2
            j = np.argmin(d2, axis=1)                         # first minimum (R-C1)
            rows = np.arange(len(tk))
            best = d2[rows, j]
            d2[rows, j] = np.inf
            second = d2.min(axis=1) if d2.shape[1] > 1 else np.full(len(tk), np.inf)
            a = cd[j]
            assign[tk] = a
            d1sq[tk] = best
            d2sq[tk] = second
            np.add.at(z, a, X[tk])                            # z_a += x   (line 21)
            np.add.at(cnt, a, 1)                              # n_a += 1
        J.append(float(d1sq.sum()))
        nz = cnt > 0
        mu = mu.copy()
        mu[nz] = z[nz] / cnt[nz][:, None]                     # line 23; empty keeps mu
    return dict(assign=assign, mu=mu, sizes=cnt, sums=z, d1sq=d1sq, d2sq=d2sq, J=J)


def lowe_ratio(d1sq, d2sq):
    """rho = d_1 / d_2 with unsquared distances (Eq. 6, l.97).  Single-candidate window
    (d2 = inf) -> 0; d2 = 0 (then d1 = 0) -> 1 (R-H1)."""
    d1sq = np.asarray(d1sq, dtype=np.float64)
    d2sq = np.asarray(d2sq, dtype=np.float64)
    rho = np.ones_like(d1sq)
    pos = d2sq > 0
    rho[pos] = np.sqrt(d1sq[pos] / d2sq[pos])
    rho[np.isinf(d2sq)] = 0.0
    return rho
