"""Oracle pipeline for one (batch, head): cluster -> mask -> merge -> plan -> attention
(test infrastructure, fp64).

Stage order follows the data flow the paper implies: Alg. 2 for Q and
K separately (R-C8), Eq. 2-3 for the mask from the final centroids and sizes (R-C6), Alg. 1
with that mask as its input (l.134), Eq. 1 permutations, Eq. 4 attention.
"""
from __future__ import annotations

import math

import numpy as np

from .cluster import local_window_kmeans
from .mask import build_mask
from .merge import merge_clusters
from .plan import build_plan
from .attention import masked_attention_rows


def forward_head(Q, K, V, lattice, cell_q, win_q, cell_k, win_k, iters, tile, top_p, merge_rounds,
                 seed=0, bh=0, min_kc=0.0, scale=None, rows=None, max_q_tiles=0):
    """Q, K, V: [n, D] float64.  rows: query token ids to evaluate (None = all).
    Returns dict with every intermediate (cq, ck: clustering dicts; M; group_of; gids; chi;
    plan; rows; O[rows])."""
    Q = np.asarray(Q, np.float64)
    K = np.asarray(K, np.float64)
    V = np.asarray(V, np.float64)
    n, D = Q.shape
    scale = 1.0 / math.sqrt(D) if scale is None else scale
    cq = local_window_kmeans(Q, lattice, cell_q, win_q, iters)
    ck = local_window_kmeans(K, lattice, cell_k, win_k, iters)
    M = build_mask(cq["mu"], ck["mu"], ck["sizes"], scale, top_p, min_kc)
    group_of, gids, chi = merge_clusters(cq["sizes"], ck["sizes"], M, tile[0], tile[1], merge_rounds,
                                         seed=seed, bh=bh, max_q_tiles=max_q_tiles)
    plan = build_plan(cq["assign"], ck["assign"], group_of, len(cq["sizes"]), len(ck["sizes"]))
    rows = np.arange(n) if rows is None else np.asarray(rows, np.int64)
    O = masked_attention_rows(Q, K, V, rows, cq["assign"], ck["assign"], group_of, gids, chi, scale)
    return dict(cq=cq, ck=ck, M=M, group_of=group_of, gids=gids, chi=chi, plan=plan, rows=rows, O=O)
