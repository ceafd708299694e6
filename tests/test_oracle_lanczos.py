"""Pins of the Lanczos oracle (oracle/lanczos.py): complete Krylov space = spectrum of the brute-force
dense H, orthonormal basis, Lieb-Liniger ground state vs exact diagonalisation and the Bethe-ansatz bound."""
import math

import numpy as np
import pytest

import workloads
from oracle import brute
from oracle import lanczos as olz
from test_oracle_apply import bethe_E0


@pytest.mark.parametrize("N,M", [(3, 3), (2, 4), (4, 3)])
def test_complete_krylov_space_reproduces_dense_spectrum(N, M):
    nc = math.comb(N + M - 1, M - 1)
    T, V, C = workloads.make_small_inputs(N, M, nc, seed=77 + N + M)
    H, _ = brute.dense_H(N, M, T, V)
    assert np.abs(H - H.conj().T).max() < 1e-12
    alpha, beta, basis = olz.lanczos(N, M, T, V, C, nc)
    assert len(alpha) == nc                                   # a random start vector has components along every eigenvector
    G = basis.conj() @ basis.T
    assert np.abs(G - np.eye(len(basis))).max() < 1e-10       # orthonormal
    assert np.abs(olz.ritz_values(alpha, beta) - np.linalg.eigvalsh(H)).max() < 1e-9 * max(1.0, np.abs(H).max())


def test_invariant_subspace_stops_early():
    # start from an eigenvector of a diagonal H (V = 0, T diagonal): one step, beta_0 = 0
    N, M = 3, 3
    nc = math.comb(N + M - 1, M - 1)
    T = np.diag([0.3, 1.1, 2.5]).astype(np.complex128)
    V = np.zeros((M,) * 4, dtype=np.complex128)
    v0 = np.zeros(nc, dtype=np.complex128); v0[4] = 1.0
    alpha, beta, _ = olz.lanczos(N, M, T, V, v0, 5)
    assert len(alpha) == 1 and beta[0] < 1e-12


@pytest.mark.parametrize("N,M", [(2, 5), (5, 5), (4, 7)])
def test_lieb_liniger_ground_state(N, M):
    nc = math.comb(N + M - 1, M - 1)
    T, V, _ = workloads.lieb_liniger_TV(M)
    H, _ = brute.dense_H(N, M, T, V)
    e_ed = np.linalg.eigvalsh(H)[0]
    rng = np.random.default_rng(5 + N + M)
    alpha, beta, _ = olz.lanczos(N, M, T, V, workloads.random_normalised_C(nc, rng), min(nc, 60))
    e_lz = olz.ritz_values(alpha, beta)[0]
    assert abs(e_lz - e_ed) < 1e-8 * max(1.0, abs(e_ed))
    assert e_lz >= bethe_E0(N, 10.0) - 1e-9                   # truncated plane-wave basis lies above the exact value
