"""Oracle O6: centroid scores, size-weighted softmax, row-wise top-p (test infrastructure).

Follows PAPER.md Eq. 2 (l.47), Eq. 3 (l.50-54) and A.1 "Top-p" / "Min-kc" (l.332-334):
  S_ij = <mu^q_i, mu^k_j> * scale,   P'_ij = s^k_j exp(S_ij) / sum_o s^k_o exp(S_io),
  A_i = smallest prefix, in descending order of P'_i:, with cumulative probability >= p,
  at least ceil(min_kc * N_k) clusters kept.

Readings: R-K1 `>= p*Z` on the unnormalised weights w_ij = s^k_j exp(S_ij -
max_j S_ij); ties in w -> lower j first; p >= 1 selects every cluster; R-K2 ceil for min-kc.

Pinned by (tests/test_oracle_mask.py): closed forms (equal scores + equal sizes ->
ceil(p N_k) clusters; sizes 3:1 with equal scores -> P' = (0.75, 0.25)), p = 1 -> all ones,
minimality of the selected set, rows of P' sum to 1, independent brute force.
"""
from __future__ import annotations

import math

import numpy as np


def cluster_probs(mu_q, mu_k, sizes_k, scale):
    """P' of Eq. 2 (returned for the pins; build_mask works on unnormalised w)."""
    S = (np.asarray(mu_q, np.float64) @ np.asarray(mu_k, np.float64).T) * scale
    w = np.asarray(sizes_k, np.float64)[None, :] * np.exp(S - S.max(axis=1, keepdims=True))
    return w / w.sum(axis=1, keepdims=True)


def build_mask(mu_q, mu_k, sizes_k, scale, top_p, min_kc=0.0, return_margin=False):
    """M [N_q, N_k] uint8.  With return_margin: also per-row |cum_k - p Z| / Z distance of
    the cut from the threshold (rows within 1e-9 are exempt from bit parity, R-K3)."""
    mu_q = np.asarray(mu_q, np.float64)
    mu_k = np.asarray(mu_k, np.float64)
    s_k = np.asarray(sizes_k, np.float64)
    Nq, Nk = mu_q.shape[0], mu_k.shape[0]
    M = np.zeros((Nq, Nk), dtype=np.uint8)
    margin = np.full(Nq, np.inf)
    kmin = int(math.ceil(min_kc * Nk))
    for i in range(Nq):
        S = (mu_k @ mu_q[i]) * scale                          # S_ij, j = 0..Nk-1
        w = s_k * np.exp(S - S.max())
        order = np.lexsort((np.arange(Nk), -w))               # w descending, ties -> lower j
        c = np.cumsum(w[order])                               # sequential cumulative sum
        Z = c[-1]
        if top_p >= 1.0:
            k = Nk
        else:
            k = int(np.argmax(c >= top_p * Z)) + 1            # smallest k with cum >= p Z
            near = [abs(c[k - 1] - top_p * Z)]
            if k >= 2:
                near.append(abs(c[k - 2] - top_p * Z))
            margin[i] = min(near) / Z
        k = max(k, kmin)
        M[i, order[:k]] = 1
    return (M, margin) if return_margin else M
