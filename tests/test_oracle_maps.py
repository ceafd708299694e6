"""Pins for the oracle's jump maps (CPU only)."""
import math
import os

import numpy as np
import pytest

import oracle
from oracle import brute


def _pairs(M):
    return [(k, s) for k in range(M) for s in range(k, M)]


@pytest.mark.parametrize("N,M", [(3, 3), (4, 5), (6, 4), (2, 6), (1, 4), (5, 1)])
def test_map1_against_brute_force(N, M):
    confs = brute.enumerate_configs(N, M)
    pos = {c: i for i, c in enumerate(confs)}
    nc = len(confs)
    m1 = oracle.map1(N, M, 0, nc)
    for b, n in enumerate(confs):
        for k in range(M):
            for l in range(M):
                if n[k] == 0:
                    assert m1[b, k, l] == -1                   # reading A12
                else:
                    t = list(n); t[k] -= 1; t[l] += 1
                    assert m1[b, k, l] == pos[tuple(t)]        # incl. diagonal == b (A13)


@pytest.mark.parametrize("N,M", [(10, 5), (7, 6), (30, 3)])
def test_map1_involution_count_and_range(N, M):
    nc = math.comb(N + M - 1, M - 1)
    nc1 = math.comb(N + M - 2, M - 1)
    m1 = oracle.map1(N, M, 0, nc)
    assert ((m1 == -1) | ((m1 >= 0) & (m1 < nc))).all()          # particle number conserved
    assert int((m1 >= 0).sum()) == M * M * nc1                   # #{(b,k): n_k>=1} = M nc1, times M targets
    b, k, l = np.nonzero(m1 >= 0)
    assert (m1[m1[b, k, l], l, k] == b).all()                    # jump back


def test_map1_window_matches_full():
    N, M = 10, 5
    full = oracle.map1(N, M, 0, 1001)
    assert (oracle.map1(N, M, 300, 77) == full[300:377]).all()


def test_fig3_count(golden_dir):
    # 4 possible removals x 5^2 = 100 instead of 5^4 = 625
    with open(os.path.join(golden_dir, "paper_fig3_double_jump.txt")) as f:
        line = [ln for ln in f if ln.strip() and not ln.startswith("#")][0]
    N, M, allowed, stored, naive = (int(x) for x in line.split())
    b = int(oracle.rank(N, M, np.array([[2, 1, 1, 0, 0]]))[0])
    m2 = oracle.map2(N, M, b, 1)[0]                               # [P, P]
    rows_allowed = (m2 >= 0).all(axis=1)
    assert ((m2 >= 0).any(axis=1) == rows_allowed).all()          # a removal pair is allowed or not as a whole
    assert int(rows_allowed.sum()) == allowed
    assert allowed * M * M == stored and M ** 4 == naive
    pairs = _pairs(M)
    assert [pairs[i] for i in np.nonzero(rows_allowed)[0]] == [(0, 0), (0, 1), (0, 2), (1, 2)]
    # 30 of the 70 configurations have exactly 4 allowed removal pairs (re-derived here)
    allm2 = oracle.map2(N, M, 0, math.comb(N + M - 1, M - 1))
    counts = (allm2 >= 0).all(axis=2).sum(axis=1)
    assert int((counts == 4).sum()) == 30


@pytest.mark.parametrize("N,M", [(4, 5), (3, 3), (6, 4), (2, 5), (1, 3)])
def test_map2_against_brute_force(N, M):
    confs = brute.enumerate_configs(N, M)
    pos = {c: i for i, c in enumerate(confs)}
    nc = len(confs)
    P = M * (M + 1) // 2
    pairs = _pairs(M)
    m2 = oracle.map2(N, M, 0, nc)
    total_allowed = 0
    for b, n in enumerate(confs):
        for a, (k, s) in enumerate(pairs):
            t = list(n); t[k] -= 1; t[s] -= 1
            if min(t) < 0:
                assert (m2[b, a] == -1).all()
                continue
            total_allowed += 1
            for c, (q, l) in enumerate(pairs):
                u = list(t); u[q] += 1; u[l] += 1
                assert m2[b, a, c] == pos[tuple(u)]
    nc2 = math.comb(N - 2 + M - 1, M - 1) if N >= 2 else 0
    assert total_allowed == P * nc2                              # each (N-2)-config m and pair (k<=s) once


def test_compact_double_jump_table_fig3_and_counts(golden_dir):
    """oracle.map2_compact (the paper's variable-length table) against what the paper fixes: the Fig. 3
    configuration has 4 strides, and "the transitions that come from removing the last two particles" are 3 strides in
    (PAPER.md:222); in the paper's M^2-stride count that is 4 x 5^2 = 100 stored targets against 5^4 = 625 (golden file).
    Against the mathematics: sum over lines of the strides = P nc2; every stride equals the allowed row of the dense table
    (itself pinned by brute-force particle moves above)."""
    line = [l for l in open(os.path.join(golden_dir, "paper_fig3_double_jump.txt")) if not l.startswith("#")][0].split()
    N, M, allowed, stored, naive = map(int, line)
    occ = np.array([[2, 1, 1, 0, 0]])
    b = int(oracle.rank(N, M, occ)[0])
    off, strides, pairs = oracle.map2_compact(N, M, b, 1)
    assert off.tolist() == [0, allowed] and allowed * M * M == stored and M ** 4 == naive
    assert pairs.tolist() == [[0, 0], [0, 1], [0, 2], [1, 2]]            # k = 0..M-1, s = k..M-1, allowed ones only
    assert pairs.tolist().index([1, 2]) == 3                              # "we need to skip 3 strides"
    for N, M in [(4, 5), (3, 3), (6, 4), (2, 6), (5, 2), (2, 2), (7, 3)]:
        nc, nc2, P = math.comb(N + M - 1, M - 1), math.comb(N + M - 3, M - 1), M * (M + 1) // 2
        off, strides, pairs = oracle.map2_compact(N, M, 0, nc)
        assert off[-1] == P * nc2 == strides.shape[0]
        dense = oracle.map2(N, M, 0, nc)
        ok = dense[:, :, 0] >= 0
        assert (np.diff(off) == ok.sum(axis=1)).all()
        assert (strides == dense[ok]).all()
        # a window of the table is the same lines
        o2, s2, _ = oracle.map2_compact(N, M, nc // 3, nc - nc // 3)
        assert (o2 + off[nc // 3] == off[nc // 3:]).all() and (s2 == strides[off[nc // 3]:]).all()
