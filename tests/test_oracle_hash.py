"""Pins for the oracle's combinatorics and hashing (CPU only).

Each test pins oracle/mcb_oracle.c to something that is not itself: a value the paper prints, a closed
form, an independent brute-force enumeration (oracle/brute.py shares no code with the C file).
"""
import itertools
import math
import os

import numpy as np
import pytest

import oracle
from oracle import brute

TINY = [(1, 1), (1, 4), (4, 1), (2, 2), (3, 3), (4, 3), (2, 4), (5, 2), (3, 4), (3, 5), (4, 5), (6, 4), (10, 5), (5, 7)]


def _read_golden(golden_dir, name):
    rows = []
    with open(os.path.join(golden_dir, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            rows.append(line)
    return rows


def test_table_matches_binomial_definition():
    # Eq. (7): N_c(n,m) = binom(n+m-1, m-1); Eq. (14): N_c(n,0) = 0
    N, M = 40, 9
    tab = oracle.binom_table(N, M)
    for n in range(N + 1):
        assert tab[n, 0] == 0
        for m in range(1, M + 1):
            assert tab[n, m] == math.comb(n + m - 1, m - 1)
    assert (tab[:, 1] == 1).all()
    assert (tab[:, 2] == np.arange(N + 1) + 1).all()
    # Pascal identity N_c(n,m) = N_c(n-1,m) + N_c(n,m-1) for m >= 2
    assert (tab[1:, 2:] == tab[:-1, 2:] + tab[1:, 1:-1]).all()


def test_nc_of_the_five_configs(golden_dir):
    for line in _read_golden(golden_dir, "baseline_nc.txt"):
        cfg, N, M, nc = (int(x) for x in line.split())
        assert oracle.nc(N, M) == nc == math.comb(N + M - 1, M - 1)


def test_fig1_worked_example(golden_dir):
    # |0,1,0,2,0>, N=3, M=5 -> N_c(3,3) + N_c(2,3) + N_c(1,1) = 17
    (line,) = _read_golden(golden_dir, "paper_fig1_hash.txt")
    left, right = line.split("|")
    vals = [int(x) for x in left.split()]
    N, M, occ, index = vals[0], vals[1], vals[2:7], vals[7]
    costs = [int(x) for x in right.split()]
    tab = oracle.binom_table(N, M)
    assert [tab[3, 3], tab[2, 3], tab[1, 1]] == costs
    assert sum(costs) == index
    assert oracle.rank(N, M, np.array([occ]))[0] == index
    assert oracle.unrank(N, M, np.array([index]))[0].tolist() == occ


@pytest.mark.parametrize("N,M", TINY)
def test_bijection_and_enumeration_order(N, M):
    # "maps uniquely integers to configurations without any left number";
    # order = n_{M-1} most significant ... n_1 least, n_0 remainder (independent nested loops).
    confs = brute.enumerate_configs(N, M)
    nc = math.comb(N + M - 1, M - 1)
    assert len(confs) == nc == len(set(confs))
    occ = np.array(confs, dtype=np.int32)
    assert (occ.sum(axis=1) == N).all()
    idx = oracle.rank(N, M, occ)
    assert idx.tolist() == list(range(nc))                      # Alg. 1 == position in brute list
    back = oracle.unrank(N, M, np.arange(nc))
    assert (back == occ).all()                                  # Alg. 2 == brute list entry


@pytest.mark.parametrize("N,M", [(3, 5), (10, 5), (7, 6), (25, 4)])
def test_first_and_last_configuration(N, M):
    nc = math.comb(N + M - 1, M - 1)
    first = [N] + [0] * (M - 1)
    last = [0] * (M - 1) + [N]
    assert oracle.rank(N, M, np.array([first, last])).tolist() == [0, nc - 1]
    assert oracle.unrank(N, M, np.array([0, nc - 1])).tolist() == [first, last]


@pytest.mark.parametrize("N,M", [(6, 4), (10, 5), (4, 7), (30, 3)])
def test_rank_closed_forms(N, M):
    # hockey-stick collapse of Alg. 1 and the combinatorial-number-system form (derived; SURVEY 8(c) pins)
    confs = brute.enumerate_configs(N, M)
    occ = np.array(confs, dtype=np.int32)
    idx = oracle.rank(N, M, occ)
    nc = math.comb(N + M - 1, M - 1)
    for n, want in zip(confs, idx.tolist()):
        S = list(itertools.accumulate(n))
        hockey = sum(math.comb(S[m] + m, m) - math.comb(S[m] - n[m] + m, m) for m in range(1, M))
        cns = nc - 1 - sum(math.comb(S[j] + j, j + 1) for j in range(M - 1))
        assert hockey == want == cns


@pytest.mark.parametrize("N,M", [(100, 5), (400, 4), (20, 10), (15, 12)])
def test_roundtrip_on_big_spaces(N, M):
    nc = math.comb(N + M - 1, M - 1)
    rng = np.random.default_rng(1234 + N + M)
    idx = np.unique(np.concatenate([rng.integers(0, nc, 5000), [0, 1, nc - 2, nc - 1]]))
    occ = oracle.unrank(N, M, idx)
    assert (occ >= 0).all() and (occ.sum(axis=1) == N).all()
    assert (oracle.rank(N, M, occ) == idx).all()
    # strictly increasing index <=> lexicographic order with n_{M-1} most significant
    keys = [tuple(int(x) for x in row[:0:-1]) for row in occ]
    assert keys == sorted(keys)
    # closed form at full size
    S = np.cumsum(occ.astype(object), axis=1)
    for row, b in list(zip(S, idx))[:200]:
        assert nc - 1 - sum(math.comb(int(row[j]) + j, j + 1) for j in range(M - 1)) == b
