"""Pins of the density-matrix oracle (oracle.rho; Eq. 10-11, App. B).

None of these re-types the oracle's formula: they are the brute-force ladder-operator matrices of oracle/brute.py,
trace / partial-trace identities of the number operator, Hermiticity, closed forms for one occupied configuration
and a coherent two-configuration state (App. B rules), and the energy identity that ties rho to the H.C oracle.
"""
import math

import numpy as np
import pytest

import oracle
import workloads
from oracle import brute


def _state(nc, seed):
    return workloads.random_normalised_C(nc, np.random.default_rng(seed))


@pytest.mark.parametrize("N,M", [(1, 3), (2, 2), (3, 3), (2, 4), (4, 3), (5, 2)])
def test_rho_matches_brute_force_operators(N, M):
    nc = math.comb(N + M - 1, M - 1)
    C = _state(nc, 700 + 10 * N + M)
    r1, r2 = oracle.rho(N, M, C)
    # rho1_kl = <C| a+_k a_l |C>: dense operator of the unit matrix E_kl through brute.dense_H (no hash, no tables)
    for k in range(M):
        for l in range(M):
            E = np.zeros((M, M), dtype=np.complex128)
            E[k, l] = 1.0
            A, _ = brute.dense_H(N, M, E, None)
            assert abs(np.vdot(C, A @ C) - r1[k, l]) < 1e-12
    # rho2_ksql = <C| a+_k a+_s a_q a_l |C>: H with T = 0 and V = 2 * unit tensor (H carries 1/2 V)
    Z = np.zeros((M, M), dtype=np.complex128)
    for idx in np.ndindex(M, M, M, M):
        V = np.zeros((M, M, M, M), dtype=np.complex128)
        V[idx] = 2.0
        A, _ = brute.dense_H(N, M, Z, V)
        assert abs(np.vdot(C, A @ C) - r2[idx]) < 1e-12, idx


@pytest.mark.parametrize("N,M", [(1, 4), (3, 3), (6, 4), (10, 5), (4, 7)])
def test_rho_traces_hermiticity_partial_trace(N, M):
    nc = math.comb(N + M - 1, M - 1)
    C = _state(nc, 800 + 10 * N + M)
    r1, r2 = oracle.rho(N, M, C)
    assert abs(np.trace(r1) - N) < 1e-12                                     # sum_k <n_k> = N
    assert abs(np.einsum("ksks->", r2) - N * (N - 1)) < 1e-10                # sum_ks <a+_k a+_s a_k a_s> = N(N-1)
    assert np.abs(r1 - r1.conj().T).max() < 1e-13                            # rho1 Hermitian
    assert np.abs(r2 - r2.conj().transpose(3, 2, 1, 0)).max() < 1e-12        # <a+k a+s aq al>* = <a+l a+q as ak>
    assert np.abs(r2 - r2.transpose(1, 0, 2, 3)).max() < 1e-12               # bosons: symmetric under k<->s
    assert np.abs(r2 - r2.transpose(0, 1, 3, 2)).max() < 1e-12               # ... and q<->l
    # sum_s a+_k a+_s a_s a_l = a+_k (N^ ) a_l acting on N-1 particles
    assert np.abs(np.einsum("kssl->kl", r2) - (N - 1) * r1).max() < 1e-11


def test_rho_closed_forms_app_b():
    # one occupied configuration |n>: rho_kk = n_k, rho_ksks = n_k n_s (k != s), rho_kkkk = n_k (n_k - 1)   (App. B)
    N, M = 7, 4
    occ = np.array([[3, 0, 2, 2]], dtype=np.int32)
    nc = math.comb(N + M - 1, M - 1)
    C = np.zeros(nc, dtype=np.complex128)
    C[oracle.rank(N, M, occ)[0]] = np.exp(0.3j)
    r1, r2 = oracle.rho(N, M, C)
    n = occ[0]
    assert np.allclose(r1, np.diag(n), atol=1e-14)
    for k in range(M):
        assert abs(r2[k, k, k, k] - n[k] * (n[k] - 1)) < 1e-13
        for s in range(M):
            if s != k:
                assert abs(r2[k, s, k, s] - n[k] * n[s]) < 1e-13 and abs(r2[k, s, s, k] - n[k] * n[s]) < 1e-13
    # two configurations connected by one jump k -> l: rho_kl = conj(c_bra) c_ket sqrt((n_l+1) n_k), n of the bra
    bra = np.array([[3, 0, 2, 2]], dtype=np.int32)
    ket = np.array([[2, 1, 2, 2]], dtype=np.int32)         # bra with one particle moved 0 -> 1
    a, b = 0.6, 0.8j
    C[:] = 0
    C[oracle.rank(N, M, bra)[0]] = a
    C[oracle.rank(N, M, ket)[0]] = b
    r1, r2 = oracle.rho(N, M, C)
    assert abs(r1[0, 1] - np.conj(a) * b * math.sqrt((0 + 1) * 3)) < 1e-14       # App. B rho_kl
    assert abs(r1[1, 0] - np.conj(b) * a * math.sqrt((0 + 1) * 3)) < 1e-14
    # App. B rho_kssl = sum C*_b C_{b_k^l} n_s sqrt(n_k (n_l + 1)), s = 2 (n_s = 2)
    assert abs(r2[0, 2, 2, 1] - np.conj(a) * b * 2 * math.sqrt(3 * 1)) < 1e-14
    # App. B "rho_kskl" = rho_kkkl = (n_k - 1) sqrt(n_k (n_l + 1))
    assert abs(r2[0, 0, 0, 1] - np.conj(a) * b * (3 - 1) * math.sqrt(3 * 1)) < 1e-14


@pytest.mark.parametrize("cfg_like", [(6, 4, "dense"), (8, 5, "ll"), (12, 3, "dense")])
def test_energy_identity_ties_rho_to_hc_apply(cfg_like):
    # <C|H|C> = sum T_kl rho1_kl + 1/2 sum V_ksql rho2_ksql, with H.C from the (independently pinned) apply oracle
    N, M, kind = cfg_like
    nc = math.comb(N + M - 1, M - 1)
    T, V, C = workloads.make_small_inputs(N, M, nc, seed=900 + N + M, kind=kind, general_V=(kind == "dense"))
    HC, _ = oracle.hc_apply(N, M, T, V, C)
    r1, r2 = oracle.rho(N, M, C)
    e_rho = np.einsum("kl,kl->", T, r1) + 0.5 * np.einsum("ksql,ksql->", V, r2)
    assert abs(np.vdot(C, HC) - e_rho) < 1e-10 * max(1.0, abs(e_rho))
