"""Oracle O7: hardware cost model and parallel agglomerative merging (test infrastructure).

Follows PAPER.md Eq. 7-8 (l.111-117), Eq. 9-10 (l.121-125), the selection rule of l.127
and Alg. 1 (l.131-168) line by line.  Costs are kept in TILE units
c(S) = ceil(s^q(S)/tau_q) * ceil(kappa(S)/tau_k), kappa(S) = sum_j chi_j(S) s^k_j, i.e.
Eq. 8 divided by the constant tau_q*tau_k (DESIGN.md R-M7), in Python integers.

Readings: R-M1 the "random bipartition" (Alg. 1 line 6) is an independent fair
coin per group from the counter-based hash `side_hash` whose constants are also printed in
include/hva.h (each side implements it separately); R-M2 active groups = groups with
s^q > 0; R-M3 ties -> lower group id, both in pi(A) and in the per-B conflict resolution;
gid(S) = smallest member; optional literal one-tile cap `max_q_tiles`.

Pinned by (tests/test_oracle_merge.py): hand fixture F2 (tests/golden/f2_merge.txt), hand
cases (60,60)/(120,120)/(130,100), invariants (partition, chi = OR of members, sum of
costs strictly decreasing per accepted merge, <= 1 merge per group per round, row-tile
saving R-M6), exhaustive optimal partition for N_q <= 7 as a lower bound, hash vectors.
The exact partition for a given seed is pinned only by our own hash spec (paper's RNG unknown).
"""
from __future__ import annotations

import numpy as np

_M32 = 0xFFFFFFFF


def side_hash(seed, bh, rnd, gid):
    """1 -> side A, 0 -> side B.  32-bit counter-based hash of (seed, b*heads+head, round
    (1-based), gid); constants as printed in include/hva.h (R-M1)."""
    h = ((seed * 0x9E3779B1) ^ (bh * 0x85EBCA77) ^ (rnd * 0xC2B2AE3D) ^ (gid * 0x27D4EB2F)) & _M32
    h ^= h >> 16
    h = (h * 0x7FEB352D) & _M32
    h ^= h >> 15
    h = (h * 0x846CA68B) & _M32
    h ^= h >> 16
    return h >> 31


def _cdiv(a, b):
    return -(-int(a) // int(b))


def tile_cost(sq, kappa, tau_q, tau_k):
    """c(S) in tile units (Eq. 8 / (tau_q tau_k))."""
    return _cdiv(sq, tau_q) * _cdiv(kappa, tau_k)


def merge_clusters(sizes_q, sizes_k, M, tau_q, tau_k, rounds, seed=0, bh=0, max_q_tiles=0,
                   sides=None, trace=None):
    """Alg. 1.  sizes_q [N_q], sizes_k [N_k], M [N_q, N_k] {0,1}.

    Returns (group_of_cluster [N_q] int64 (= gid of the cluster's group; clusters with
    s^q = 0 keep their own id and take no part), gids (ascending list of active group ids),
    chi [len(gids), N_k] uint8 union masks in gid order).
    `sides`: optional callable (round, gid) -> 0/1 overriding the hash (for hand fixtures).
    `trace`: optional list receiving (round, A, B, delta_c) per accepted merge.
    """
    sq0 = [int(v) for v in sizes_q]
    sk = np.asarray(sizes_k, dtype=np.int64)
    Nq = len(sq0)
    chi = {i: np.asarray(M[i], dtype=bool).copy() for i in range(Nq) if sq0[i] > 0}   # line 4
    sq = {i: sq0[i] for i in chi}                                                        # line 3
    members = {i: [i] for i in chi}
    kap = {i: int(sk[chi[i]].sum()) for i in chi}
    for r in range(1, rounds + 1):                                                       # line 5
        side = (lambda g: sides(r, g)) if sides is not None else (lambda g: side_hash(seed, bh, r, g))
        gl = sorted(chi)
        A_set = [g for g in gl if side(g) == 1]                                          # line 6
        B_set = [g for g in gl if side(g) == 0]
        best_for_B = {}
        for A in A_set:                                                                  # line 7
            best = None
            for B in B_set:                                                              # line 8
                s_u = sq[A] + sq[B]                                                      # line 9
                chi_u = chi[A] | chi[B]                                                  # line 10
                c_u = tile_cost(s_u, int(sk[chi_u].sum()), tau_q, tau_k)                 # line 11
                dc = c_u - tile_cost(sq[A], kap[A], tau_q, tau_k) - tile_cost(sq[B], kap[B], tau_q, tau_k)  # 12
                if max_q_tiles > 0 and _cdiv(s_u, tau_q) > max_q_tiles:
                    continue
                if best is None or dc < best[0]:                                         # line 13, ties -> lower B
                    best = (dc, B)
            if best is None:
                continue
            dc, B = best
            if dc < 0:                                                                   # line 14
                cur = best_for_B.get(B)
                if cur is None or (dc, A) < cur:                                         # argmin_A', ties -> lower A
                    best_for_B[B] = (dc, A)
        for B, (dc, A) in sorted(best_for_B.items()):                                    # lines 15-16
            g, o = min(A, B), max(A, B)
            chi[g] = chi[A] | chi[B]
            sq[g] = sq[A] + sq[B]
            members[g] = sorted(members[A] + members[B])
            kap[g] = int(sk[chi[g]].sum())
            del chi[o], sq[o], members[o], kap[o]
            if trace is not None:
                trace.append((r, A, B, dc))
    group_of = np.arange(Nq, dtype=np.int64)
    for g, ms in members.items():
        group_of[ms] = g
    gids = sorted(chi)
    chi_out = np.stack([chi[g] for g in gids]).astype(np.uint8) if gids else np.zeros((0, len(sk)), np.uint8)
    return group_of, gids, chi_out
