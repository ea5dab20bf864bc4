"""Pins for oracle O6 (mask) and O7 (cost model + merging).  CPU only."""
import itertools
import math

import numpy as np
import pytest

import oracle
from oracle.mask import cluster_probs
from conftest import read_golden


# ----------------------------------------------------------------------------- mask (Eq. 2-3)
def test_mask_equal_scores_equal_sizes_closed_form():
    Nk, D = 10, 4
    mu_q = np.zeros((3, D))
    mu_k = np.ones((Nk, D))
    for p in (0.05, 0.33, 0.57, 0.91):                      # off the lattice k/Nk
        M = oracle.build_mask(mu_q, mu_k, np.full(Nk, 7), 0.5, p)
        assert (M.sum(1) == math.ceil(p * Nk)).all()
        assert (M[:, : math.ceil(p * Nk)] == 1).all()       # ties -> lower j first


def test_mask_size_weighting_3_to_1():
    mu_q = np.array([[1.0, 0.0]])
    mu_k = np.array([[0.3, 0.2], [0.3, -0.9]])              # equal scores <mu_q, mu_k> = 0.3
    P = cluster_probs(mu_q, mu_k, [3, 1], 1.0)
    assert np.allclose(P, [[0.75, 0.25]])
    assert oracle.build_mask(mu_q, mu_k, [3, 1], 1.0, 0.7).tolist() == [[1, 0]]
    assert oracle.build_mask(mu_q, mu_k, [3, 1], 1.0, 0.8).tolist() == [[1, 1]]
    assert oracle.build_mask(mu_q, mu_k, [1, 3], 1.0, 0.7).tolist() == [[0, 1]]


def test_mask_minimality_p1_minkc_and_brute_force():
    rng = np.random.default_rng(2)
    mu_q, mu_k = rng.standard_normal((9, 16)), rng.standard_normal((13, 16))
    s_k = rng.integers(0, 40, 13)
    s_k[4] = 0                                              # empty key cluster: P' = 0 (R-C7)
    scale = 0.25
    P = cluster_probs(mu_q, mu_k, s_k, scale)
    assert np.allclose(P.sum(1), 1.0)
    # independent brute force of Eq. 2 with explicit loops
    for i, j in itertools.product(range(9), range(13)):
        num = s_k[j] * math.exp(float(mu_q[i] @ mu_k[j]) * scale)
        den = sum(s_k[o] * math.exp(float(mu_q[i] @ mu_k[o]) * scale) for o in range(13))
        assert abs(P[i, j] - num / den) < 1e-12
    for p in (0.5, 0.9):
        M = oracle.build_mask(mu_q, mu_k, s_k, scale, p)
        for i in range(9):
            sel = M[i].astype(bool)
            assert P[i, sel].sum() >= p - 1e-12
            assert P[i, sel].sum() - P[i, sel].min() < p + 1e-12      # dropping the last -> < p
            assert P[i, sel].min() >= P[i, ~sel].max() - 1e-15          # descending-order prefix
    assert (oracle.build_mask(mu_q, mu_k, s_k, scale, 1.0) == 1).all()  # p = 1 -> all ones
    M = oracle.build_mask(mu_q, mu_k, s_k, scale, 0.01, min_kc=0.5)
    assert (M.sum(1) == math.ceil(0.5 * 13)).all()


# ----------------------------------------------------------------------------- merge (Eq. 7-10, Alg. 1)
def test_side_hash_vectors():
    # literal re-evaluation of the spec printed in include/hva.h with Python big ints
    def ref(seed, bh, r, g):
        h = (seed * 0x9E3779B1 ^ bh * 0x85EBCA77 ^ r * 0xC2B2AE3D ^ g * 0x27D4EB2F) % 2 ** 32
        h ^= h >> 16; h = h * 0x7FEB352D % 2 ** 32; h ^= h >> 15; h = h * 0x846CA68B % 2 ** 32; h ^= h >> 16
        return h >> 31
    bits = [oracle.side_hash(3, 5, r, g) for r in (1, 2, 3) for g in range(200)]
    assert bits == [ref(3, 5, r, g) for r in (1, 2, 3) for g in range(200)]
    assert 0.35 < np.mean(bits) < 0.65                      # a fair-ish coin
    assert [oracle.side_hash(0, 0, 1, g) for g in range(8)] != [oracle.side_hash(0, 0, 2, g) for g in range(8)]


def test_f2_hand_fixture():
    g = read_golden("f2_merge.txt")
    tq, tk = [int(v) for v in g["tau"]]
    sq, sk = [int(v) for v in g["sq"]], [int(v) for v in g["sk"]]
    M = np.array([g["m0"], g["m1"], g["m2"], g["m3"]], dtype=np.uint8)
    kap = M.astype(int) @ np.array(sk)
    assert [oracle.tile_cost(sq[i], kap[i], tq, tk) for i in range(4)] == g["cost"]
    gains = []
    for a, b in itertools.combinations(range(4), 2):
        ku = int(((M[a] | M[b]).astype(int) * sk).sum())
        gains.append(oracle.tile_cost(sq[a] + sq[b], ku, tq, tk) - g["cost"][a] - g["cost"][b])
    assert gains == g["gain"]
    tr = []
    gof, gids, chi = oracle.merge_clusters(sq, sk, M, tq, tk, 1, sides=lambda r, x: int(x in (0, 2)), trace=tr)
    assert gof.tolist() == g["groupsA02"] and gids == [0, 2, 3] and tr == [(1, 0, 1, -2)]
    assert chi.tolist() == [[1, 1, 0], [0, 1, 1], [1, 0, 1]]
    gof, _, _ = oracle.merge_clusters(sq, sk, M, tq, tk, 1, sides=lambda r, x: int(x in (0, 1)))
    assert gof.tolist() == g["groupsA01"]


@pytest.mark.parametrize("sizes,merges", [((60, 60), True), ((120, 120), False)])
def test_hand_cases_tau128(sizes, merges):
    sk = [128, 128, 128]
    M = np.array([[1, 1, 0], [1, 1, 0]], dtype=np.uint8)    # identical key sets, k = 2 tiles
    tr = []
    gof, _, _ = oracle.merge_clusters(sizes, sk, M, 128, 128, 1, sides=lambda r, g: int(g == 0), trace=tr)
    assert (gof.tolist() == [0, 0]) == merges
    if merges:
        assert tr[0][3] == -2                               # gain = -k tiles


def test_hand_case_130_100():
    # rows 130 + 100 -> 2 tiles instead of 2 + 1; merges iff 2 k_U < 2 k_A + k_B
    sk = [128] * 6
    A = [1, 1, 1, 0, 0, 0]
    for B, expect in (([1, 1, 0, 0, 0, 0], True),           # kU=3,kA=3,kB=2: 6 < 8
                      ([0, 0, 0, 1, 1, 1], False)):         # kU=6,kA=3,kB=3: 12 < 9 false
        gof, _, _ = oracle.merge_clusters([130, 100], sk, np.array([A, B], np.uint8), 128, 128, 1,
                                          sides=lambda r, g: int(g == 0))
        assert (gof.tolist() == [0, 0]) == expect


def _total_cost(gof, sq, sk, M, tq, tk):
    tot = 0
    for g in np.unique(gof):
        mem = np.where(gof == g)[0]
        s = int(np.asarray(sq)[mem].sum())
        if s == 0:
            continue
        chi = M[mem].max(0).astype(bool)
        tot += oracle.tile_cost(s, int(np.asarray(sk)[chi].sum()), tq, tk)
    return tot


def _optimal_partition_cost(sq, sk, M, tq, tk):
    n = len(sq)
    best = [None]

    def rec(i, blocks):
        if i == n:
            gof = np.empty(n, dtype=np.int64)
            for b in blocks:
                gof[b] = b[0]
            c = _total_cost(gof, sq, sk, M, tq, tk)
            best[0] = c if best[0] is None else min(best[0], c)
            return
        for b in blocks:
            b.append(i); rec(i + 1, blocks); b.pop()
        blocks.append([i]); rec(i + 1, blocks); blocks.pop()
    rec(0, [])
    return best[0]


@pytest.mark.parametrize("seed", range(6))
def test_merge_invariants_and_optimal_lower_bound(seed):
    rng = np.random.default_rng(seed)
    Nq, Nk, tq, tk = 7, 9, 16, 16
    sq = rng.integers(0, 30, Nq); sq[rng.integers(Nq)] = 0     # one empty query cluster
    sk = rng.integers(1, 30, Nk)
    M = (rng.random((Nq, Nk)) < 0.45).astype(np.uint8); M[:, 0] = 1
    prev_cost = _total_cost(np.arange(Nq), sq, sk, M, tq, tk)
    prev_gof = np.arange(Nq)
    for R in (1, 2, 3):
        tr = []
        gof, gids, chi = oracle.merge_clusters(sq, sk, M, tq, tk, R, seed=seed, bh=1, trace=tr)
        # partition of non-empty clusters, gid = smallest member, chi = OR of members
        assert sorted(set(gof[sq > 0])) == gids
        for k, g in enumerate(gids):
            mem = np.where(gof == g)[0]
            assert mem.min() == g and np.array_equal(chi[k], M[mem].max(0))
        assert all(gof[i] == i for i in range(Nq) if sq[i] == 0)
        cost = _total_cost(gof, sq, sk, M, tq, tk)
        this_round = [t for t in tr if t[0] == R]
        assert cost == prev_cost + sum(t[3] for t in this_round)      # sum of costs drops by the gains
        assert all(t[3] < 0 for t in tr)                               # strictly decreasing per merge
        used = [x for t in this_round for x in t[1:3]]
        assert len(used) == len(set(used))                             # <= 1 merge per group per round
        for (_, A, B, _) in this_round:                                # R-M6: a row tile is saved
            sA = sq[prev_gof == A].sum(); sB = sq[prev_gof == B].sum()
            assert -(-(sA + sB) // tq) == -(-sA // tq) + -(-sB // tq) - 1
        prev_cost, prev_gof = cost, gof
    assert _optimal_partition_cost(sq, sk, M, tq, tk) <= prev_cost


def test_max_q_tiles_cap():
    sk = [128, 128]
    M = np.ones((2, 2), np.uint8)
    # 130 + 100 rows: 3 row tiles -> 2, so the merge is accepted uncapped but spans 2 tiles
    kw = dict(sides=lambda r, g: int(g == 0))
    assert oracle.merge_clusters([130, 100], sk, M, 128, 128, 1, **kw)[0].tolist() == [0, 0]
    assert oracle.merge_clusters([130, 100], sk, M, 128, 128, 1, max_q_tiles=1, **kw)[0].tolist() == [0, 1]
