"""Oracle O8: canonical permutations Pi^q, Pi^k (test infrastructure).

PAPER.md Eq. 1 (l.37) only requires that the tokens of a cluster be contiguous; the
canonical order (DESIGN.md R-P1) makes the permutations comparable bit for bit:
  perm_k : tokens sorted by (a^k_l, l)
  perm_q : tokens sorted by (gid(a^q_l), a^q_l, l)      gid = merged group id (Alg. 1)
perm[i] = original token index placed at permuted row i;  inv_perm_q[perm_q[i]] = i.

Pinned by (tests/test_oracle_plan.py): bijection, inv o perm = id, segments contiguous
with lengths equal to the cluster / group sizes.
"""
from __future__ import annotations

import numpy as np


def build_plan(assign_q, assign_k, group_of_cluster, n_q_clusters, n_k_clusters):
    aq = np.asarray(assign_q, dtype=np.int64)
    ak = np.asarray(assign_k, dtype=np.int64)
    gof = np.asarray(group_of_cluster, dtype=np.int64)
    n = aq.shape[0]
    tok = np.arange(n, dtype=np.int64)
    perm_k = np.lexsort((tok, ak))
    perm_q = np.lexsort((tok, aq, gof[aq]))
    inv_perm_q = np.empty(n, dtype=np.int64)
    inv_perm_q[perm_q] = tok
    sizes_k = np.bincount(ak, minlength=n_k_clusters)
    koff = np.concatenate([[0], np.cumsum(sizes_k)])           # K' row offset of key cluster j
    sizes_q = np.bincount(aq, minlength=n_q_clusters)
    gids = np.unique(gof[sizes_q > 0]) if n else np.zeros(0, np.int64)
    gsize = np.array([sizes_q[gof == g].sum() for g in gids], dtype=np.int64)
    goff = np.concatenate([[0], np.cumsum(gsize)])             # Q' row offset of group (gid order)
    return dict(perm_q=perm_q, inv_perm_q=inv_perm_q, perm_k=perm_k, koff=koff, goff=goff, gids=gids)
