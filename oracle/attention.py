"""Oracle O9: block-sparse attention in original token order (test infrastructure, fp64).

Follows PAPER.md Eq. 4 (l.56): O'_i = Attn(Q'_i, {K'_j, V'_j}_{j in A_i}), O = Pi^{q-1} O',
"standard scaled dot-product attention restricted to the selected key/value clusters"
(l.59), with the merged-group union chi_j(S) = max_{i in S} m_ij (Eq. 8, l.115) as the
key set of every query of the group (DESIGN.md R-A1, R-A2).  Because the result does not
depend on the permutation, the oracle works in original token order: query l attends to
the keys m whose key cluster is selected for the group of l's query cluster.

Pinned by (tests/test_oracle_attention.py): dense softmax over all n keys with the
token-level mask applied elementwise as -inf, top_p = 1 == full attention
(torch.nn.functional.scaled_dot_product_attention in fp64), softmax weights sum to 1.
"""
from __future__ import annotations

import numpy as np


def token_key_mask(rows, assign_q, assign_k, group_of_cluster, gids, chi):
    """[len(rows), n] bool: key m allowed for query l  <=>  chi[group(a^q_l)][a^k_m] = 1."""
    gids = np.asarray(gids, dtype=np.int64)
    g = np.asarray(group_of_cluster, np.int64)[np.asarray(assign_q, np.int64)[rows]]
    gi = np.searchsorted(gids, g)
    return np.asarray(chi, bool)[gi][:, np.asarray(assign_k, np.int64)]


def masked_attention_rows(Q, K, V, rows, assign_q, assign_k, group_of_cluster, gids, chi, scale):
    """O[rows] in fp64.  Q, K, V: [n, D] float64 (one batch-head); rows: query token ids."""
    rows = np.asarray(rows, dtype=np.int64)
    allow = token_key_mask(rows, assign_q, assign_k, group_of_cluster, gids, chi)
    S = (Q[rows] @ K.T) * scale                               # [r, n]
    S = np.where(allow, S, -np.inf)
    S = S - S.max(axis=1, keepdims=True)                      # max-subtraction
    P = np.exp(S)
    P /= P.sum(axis=1, keepdims=True)
    return P @ V
