"""Oracle O4-O5: hybrid clustering across denoising steps (test infrastructure, fp64).

Follows PAPER.md section 4.2 (l.93-103) and A.1 (l.322): at anchor steps cache the indices
of the tokens with the largest Lowe ratio rho (top 15 %); at intermediate steps "update only
this subset by performing a standard k-means reassignment against the current centroid set
and then updating the corresponding centroids" (l.101), "reassigned using the full centroid
set" (l.103).

Readings: R-H2 m = floor(f n + 1/2), ties -> lower token index, subset stored
ascending by index; R-H3 all reassignments see the same cached mu (Jacobi), first minimum
over ALL N_c centroids; sums/counts are adjusted incrementally for MOVED tokens using their
CURRENT features; mu_u <- z_u / n_u for touched u with n_u > 0; no non-subset token is read.
R-H3' (`refresh_all`): after the reassignment every centroid is recomputed as the mean of the
CURRENT features of its members.

Pins (tests/test_oracle_plan_attn_hybrid.py): `select_subset` -- hand ties, order statistics.
`subset_update(refresh_all=True)` -- f = 1 is one textbook global k-means step (brute force).
`subset_update(refresh_all=False)` -- with UNCHANGED X (cached sums are then exact member sums) the
incrementally adjusted sums / sizes / mu of every touched centroid equal a from-scratch
recomputation over the new labels, on a lattice whose window does not cover the grid so that
subset tokens do move; unchanged X + already optimal labels -> no-op; counts stay consistent;
non-subset labels untouched.  What the paper does NOT pin is the READING itself (R-H3: which
centroids "the corresponding centroids" are and with which features they are adjusted); the
arithmetic of the reading is pinned by the identities above.
"""
from __future__ import annotations

import math

import numpy as np


def select_subset(rho, frac):
    """Indices (ascending) of the m = floor(f n + 1/2) tokens with the largest rho;
    ties -> lower token index (l.101; l.322; R-H2)."""
    rho = np.asarray(rho, dtype=np.float64)
    n = rho.shape[0]
    m = int(math.floor(frac * n + 0.5))
    order = np.lexsort((np.arange(n), -rho))
    return np.sort(order[:m]).astype(np.int64)


def subset_update(X, assign, mu, sums, sizes, subset, refresh_all=False):
    """One intermediate step on one (batch, head, tensor).

    X [n, D] current features; assign [n]; mu [Nc, D]; sums [Nc, D] cached z; sizes [Nc]
    cached n; subset: token ids.  Returns new (assign, mu, sums, sizes, d1sq, d2sq) where
    d1sq / d2sq are the best / second-best squared distances of the subset tokens (for the
    near-tie exemption of the parity test).
    """
    X = np.asarray(X, np.float64)
    assign = np.array(assign, dtype=np.int64)
    mu = np.array(mu, dtype=np.float64)
    sums = np.array(sums, dtype=np.float64)
    sizes = np.array(sizes, dtype=np.int64)
    subset = np.asarray(subset, dtype=np.int64)
    xs = X[subset]
    # ||x - mu_u||^2 for every centroid u, written out term by term (no expansion)
    d2 = np.empty((len(subset), mu.shape[0]))
    for u in range(mu.shape[0]):
        diff = xs - mu[u][None, :]
        d2[:, u] = np.einsum("td,td->t", diff, diff)
    new = np.argmin(d2, axis=1)                               # first minimum
    r = np.arange(len(subset))
    d1sq = d2[r, new].copy()
    d2[r, new] = np.inf
    d2sq = d2.min(axis=1) if mu.shape[0] > 1 else np.full(len(subset), np.inf)
    old = assign[subset]
    moved = new != old
    touched = np.zeros(mu.shape[0], dtype=bool)
    for l, o, a in zip(subset[moved], old[moved], new[moved]):
        sums[o] -= X[l]
        sizes[o] -= 1
        sums[a] += X[l]
        sizes[a] += 1
        touched[o] = touched[a] = True
    assign[subset] = new
    if refresh_all:
        sums = np.zeros_like(sums)
        np.add.at(sums, assign, X)
        sizes = np.bincount(assign, minlength=mu.shape[0]).astype(np.int64)
        touched[:] = True
    upd = touched & (sizes > 0)
    mu[upd] = sums[upd] / sizes[upd][:, None]
    return assign, mu, sums, sizes, d1sq, d2sq
