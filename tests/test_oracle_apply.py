"""Pins for the oracle's H.C (CPU only): brute-force dense H from one-at-a-time ladder operators,
App. B rules, invariants, closed forms, Lieb-Liniger energies.  SURVEY.md 8(c) "What pins each part".
"""
import itertools
import math

import numpy as np
import pytest

import oracle
import workloads
from oracle import brute


def _nc(N, M):
    return math.comb(N + M - 1, M - 1)


def oracle_dense(N, M, T, V):
    """Dense H through the oracle: column b = hc_apply(e_b)."""
    nc = _nc(N, M)
    H = np.zeros((nc, nc), dtype=np.complex128)
    for b in range(nc):
        e = np.zeros(nc, dtype=np.complex128)
        e[b] = 1.0
        H[:, b], _ = oracle.hc_apply(N, M, T, V, e)
    return H


@pytest.mark.parametrize("N,M", [(3, 3), (4, 3), (2, 4), (5, 2), (3, 4), (1, 3), (4, 1), (2, 2)])
@pytest.mark.parametrize("general_V", [False, True])
def test_dense_H_element_by_element(N, M, general_V):
    # O5 vs O6: ladder operators one at a time + dictionary lookup vs gather form + Alg. 1
    nc = _nc(N, M)
    T, V, _ = workloads.make_small_inputs(N, M, nc, seed=77 + 10 * N + M, general_V=general_V)
    if general_V:
        T = T + 0.3j * np.triu(np.ones((M, M)), 1)      # non-Hermitian T as well
    Hb, _ = brute.dense_H(N, M, T, V)
    Ho = oracle_dense(N, M, T, V)
    scale = max(np.abs(T).max(), np.abs(V).max())
    assert np.abs(Hb - Ho).max() <= 1e-13 * scale * N * N


def test_sampled_columns_N10_M5():
    # config 0 size: a few columns of the brute-force matrix (full dense_H in Python is too slow)
    N, M = 10, 5
    nc = _nc(N, M)
    T, V, C = workloads.make_small_inputs(N, M, nc, seed=5)
    confs = brute.enumerate_configs(N, M)
    pos = {c: i for i, c in enumerate(confs)}
    for b in (0, 17, 500, 1000):
        col = np.zeros(nc, dtype=np.complex128)
        ket = confs[b]
        for k, l in itertools.product(range(M), repeat=2):
            r = brute.annihilate(ket, l)
            if r is None:
                continue
            a2, st = brute.create(r[1], k)
            col[pos[st]] += T[k, l] * r[0] * a2
        for k, s, q, l in itertools.product(range(M), repeat=4):
            r1 = brute.annihilate(ket, l)
            if r1 is None:
                continue
            r2 = brute.annihilate(r1[1], q)
            if r2 is None:
                continue
            a3, st = brute.create(r2[1], s)
            a4, st = brute.create(st, k)
            col[pos[st]] += 0.5 * V[k, s, q, l] * r1[0] * r2[0] * a3 * a4
        e = np.zeros(nc, dtype=np.complex128)
        e[b] = 1.0
        got, _ = oracle.hc_apply(N, M, T, V, e)
        assert np.abs(got - col).max() <= 1e-12 * np.abs(V).max()


def test_appendix_B_rules():
    # PAPER.md:377 (garbled): <n| a+_k a+_s a_q a_l |n - e_k - e_s + e_q + e_l>, n = bra occupations
    N, M = 6, 4
    nc = _nc(N, M)
    confs = brute.enumerate_configs(N, M)
    pos = {c: i for i, c in enumerate(confs)}
    Z = np.zeros((M, M), dtype=np.complex128)
    rules = {
        # (k, s, q, l): amplitude(n)
        (0, 1, 2, 3): lambda n: math.sqrt(n[0] * n[1] * (n[2] + 1) * (n[3] + 1)),     # rho_ksql
        (0, 0, 2, 3): lambda n: math.sqrt((n[0] - 1) * n[0] * (n[2] + 1) * (n[3] + 1)),  # rho_kkql
        (0, 1, 2, 2): lambda n: math.sqrt(n[0] * n[1] * (n[2] + 1) * (n[2] + 2)),     # rho_ksqq
        (0, 0, 2, 2): lambda n: math.sqrt((n[0] - 1) * n[0] * (n[2] + 1) * (n[2] + 2)),  # rho_kkqq (by analogy)
        (0, 0, 0, 3): lambda n: (n[0] - 1) * math.sqrt(n[0] * (n[3] + 1)),            # rho_kkkl
        (0, 1, 1, 3): lambda n: n[1] * math.sqrt(n[0] * (n[3] + 1)),                  # rho_kssl
        (0, 1, 0, 1): lambda n: n[0] * n[1],                                          # rho_ksks
        (2, 2, 2, 2): lambda n: n[2] * (n[2] - 1),                                    # rho_kkkk
    }
    for (k, s, q, l), amp in rules.items():
        V = np.zeros((M, M, M, M), dtype=np.complex128)
        V[k, s, q, l] = 2.0                      # cancels the 1/2 of H
        H = oracle_dense(N, M, Z, V)
        want = np.zeros_like(H)
        for g, n in enumerate(confs):
            t = list(n)
            t[k] -= 1; t[s] -= 1
            if min(t) < 0:
                continue
            t[q] += 1; t[l] += 1
            want[g, pos[tuple(t)]] += amp(n)
        assert np.abs(H - want).max() < 1e-12, (k, s, q, l)
    # one-body rules: rho_kl = sqrt((n_l+1) n_k), rho_kk = n_k
    for (k, l) in [(1, 3), (2, 2)]:
        T = Z.copy(); T[k, l] = 1.0
        H = oracle_dense(N, M, T, np.zeros((M,) * 4, dtype=np.complex128))
        want = np.zeros_like(H)
        for g, n in enumerate(confs):
            if n[k] == 0:
                continue
            t = list(n); t[k] -= 1; t[l] += 1
            want[g, pos[tuple(t)]] += n[k] if k == l else math.sqrt((n[l] + 1) * n[k])
        assert np.abs(H - want).max() < 1e-12


@pytest.mark.parametrize("N,M", [(10, 5), (6, 6), (40, 3)])
def test_hermiticity_and_linearity(N, M):
    nc = _nc(N, M)
    T, V, u = workloads.make_small_inputs(N, M, nc, seed=11)
    _, _, v = workloads.make_small_inputs(N, M, nc, seed=12)
    Hu, _ = oracle.hc_apply(N, M, T, V, u)
    Hv, _ = oracle.hc_apply(N, M, T, V, v)
    assert abs(np.vdot(u, Hv) - np.vdot(Hu, v)) < 1e-10 * N * N
    a, b = 0.7 - 0.2j, -1.3 + 0.5j
    Hw, _ = oracle.hc_apply(N, M, T, V, a * u + b * v)
    assert np.abs(Hw - (a * Hu + b * Hv)).max() < 1e-11 * N * N


def test_only_bosonic_symmetric_part_of_V_contributes():
    # V and its (k<->s), (q<->l) symmetrisation give the same H
    N, M = 5, 4
    nc = _nc(N, M)
    T, V, C = workloads.make_small_inputs(N, M, nc, seed=3, general_V=True)
    Vs = (V + V.transpose(1, 0, 2, 3) + V.transpose(0, 1, 3, 2) + V.transpose(1, 0, 3, 2)) / 4
    a, _ = oracle.hc_apply(N, M, T, V, C)
    b, _ = oracle.hc_apply(N, M, T, Vs, C)
    assert np.abs(a - b).max() < 1e-12 * N * N


def test_single_particle_is_a_matvec():
    # N = 1: configurations are |e_j>, index j (n_j = 1 costs N_c(1,j) = j); HC = T @ C, two-body part vanishes
    M = 7
    T, V, C = workloads.make_small_inputs(1, M, M, seed=21, general_V=True)
    got, _ = oracle.hc_apply(1, M, T, V, C)
    assert np.abs(got - T @ C).max() < 1e-13


def test_single_orbital():
    # M = 1: one configuration |N>; H = T_00 N + V_0000 N (N-1) / 2
    N = 9
    T = np.array([[0.3 - 0.1j]]); V = np.array([1.7 + 0.4j]).reshape(1, 1, 1, 1)
    C = np.array([0.6 + 0.8j])
    got, _ = oracle.hc_apply(N, 1, T, V, C)
    assert abs(got[0] - (T[0, 0] * N + V[0, 0, 0, 0] * N * (N - 1) / 2) * C[0]) < 1e-12


@pytest.mark.parametrize("N,M", [(4, 3), (3, 4), (6, 2)])
def test_noninteracting_spectrum(N, M):
    # V = 0: eigenvalues of H are sums of N eigenvalues of T with repetition
    nc = _nc(N, M)
    T, _, _ = workloads.make_small_inputs(N, M, nc, seed=31)
    H = oracle_dense(N, M, T, np.zeros((M,) * 4, dtype=np.complex128))
    assert np.abs(H - H.conj().T).max() < 1e-12
    eps = np.linalg.eigvalsh(T)
    want = sorted(sum(eps[list(c)]) for c in itertools.combinations_with_replacement(range(M), N))
    got = np.linalg.eigvalsh(H)
    assert np.abs(got - np.array(want)).max() < 1e-10


@pytest.mark.parametrize("N,M", [(10, 5), (50, 3)])
def test_constant_interaction(N, M):
    # V_ksql = U d_kq d_sl  =>  1/2 sum a+_k a+_s a_k a_s = U N (N-1) / 2
    nc = _nc(N, M)
    _, _, C = workloads.make_small_inputs(N, M, nc, seed=41)
    U = 0.37 - 0.11j
    d = np.eye(M)
    V = U * np.einsum("kq,sl->ksql", d, d)
    got, _ = oracle.hc_apply(N, M, np.zeros((M, M), dtype=np.complex128), V, C)
    assert np.abs(got - U * N * (N - 1) / 2 * C).max() < 1e-12 * N * N


@pytest.mark.parametrize("N,M", [(10, 5), (7, 6)])
def test_product_interaction(N, M):
    # V_ksql = A_kq A_sl  =>  two-body part = 1/2 [ A^(A^ C) - (A.A)^ C ], A^ = sum A_kl a+_k a_l
    nc = _nc(N, M)
    A, _, C = workloads.make_small_inputs(N, M, nc, seed=51)
    A = A + 0.5j * np.triu(np.ones((M, M)), 1)
    V = np.einsum("kq,sl->ksql", A, A)
    Z4 = np.zeros((M,) * 4, dtype=np.complex128)
    two, _ = oracle.hc_apply(N, M, np.zeros((M, M), dtype=np.complex128), V, C)
    AC, _ = oracle.hc_apply(N, M, A, Z4, C)
    AAC, _ = oracle.hc_apply(N, M, A, Z4, AC)
    A2C, _ = oracle.hc_apply(N, M, A @ A, Z4, C)
    assert np.abs(two - 0.5 * (AAC - A2C)).max() < 1e-11 * N * N


def test_row_subset_matches_full():
    N, M = 10, 5
    nc = _nc(N, M)
    T, V, C = workloads.make_small_inputs(N, M, nc, seed=61)
    full, _ = oracle.hc_apply(N, M, T, V, C)
    rows = workloads.sample_rows(nc, 5, 40, seed=1)
    sub, _ = oracle.hc_apply(N, M, T, V, C, rows=rows)
    assert (sub == full[rows]).all()
    one, used = oracle.hc_apply(N, M, T, V, C, nthreads=1)
    assert used == 1 and (one == full).all()


# ---- Lieb-Liniger ---------------------------------------------------------------------

def bethe_E0(N, g, L=1.0):
    """Eq. (17)-(18) PAPER.md:310-316, hbar = m = 1 (c = g), I_j = j - (N+1)/2.  Damped Newton on
    F_j(k) = k_j - 2 pi I_j / L + (2/L) sum_i arctan((k_j - k_i)/g) (gradient of the convex Yang-Yang action)."""
    I = np.arange(1, N + 1) - (N + 1) / 2
    k = 2 * math.pi * I / L * min(1.0, math.sqrt(g))
    for _ in range(500):
        d = k[:, None] - k[None, :]
        F = k - 2 * math.pi * I / L + (2 / L) * np.arctan(d / g).sum(axis=1)
        K = (2 / L) * (1 / g) / (1 + (d / g) ** 2)
        J = np.eye(N) + np.diag(K.sum(axis=1)) - K
        step = np.linalg.solve(J, F)
        t = 1.0
        while t > 1e-6:
            kn = k - t * step
            dn = kn[:, None] - kn[None, :]
            Fn = kn - 2 * math.pi * I / L + (2 / L) * np.arctan(dn / g).sum(axis=1)
            if np.linalg.norm(Fn) < np.linalg.norm(F):
                break
            t /= 2
        k = kn
        if np.abs(Fn).max() < 1e-13:
            break
    assert np.abs(Fn).max() < 1e-10
    return 0.5 * float((k ** 2).sum())


def test_bethe_solver_limits():
    # g -> 0: first-order perturbation theory E = g N (N-1) / (2L); g -> inf (Tonks-Girardeau): free fermions
    N = 5
    assert abs(bethe_E0(N, 1e-3) / (1e-3 * N * (N - 1) / 2) - 1) < 1e-3
    I = np.arange(1, N + 1) - (N + 1) / 2
    assert abs(bethe_E0(N, 1e7) / (0.5 * ((2 * math.pi * I) ** 2).sum()) - 1) < 1e-5
    # N = 2 reduces to one transcendental equation: k = (pi - 2 arctan(2k/g)) / L, E = k^2
    g = 10.0
    k = 1.0
    for _ in range(200):
        k = math.pi - 2 * math.atan(2 * k / g)
    assert abs(bethe_E0(2, g) - k * k) < 1e-10


def lanczos_E0(N, M, T, V, iters, seed=0):
    """Lanczos with full re-orthogonalisation through the oracle's hc_apply."""
    nc = _nc(N, M)
    rng = np.random.default_rng(seed)
    q = workloads.random_normalised_C(nc, rng)
    Q = [q]
    alpha, beta = [], []
    for j in range(iters):
        w, _ = oracle.hc_apply(N, M, T, V, Q[-1])
        a = np.vdot(Q[-1], w).real
        alpha.append(a)
        for qi in Q:                                    # full re-orthogonalisation
            w = w - np.vdot(qi, w) * qi
        b = np.linalg.norm(w)
        if b < 1e-12 or j == iters - 1:
            break
        beta.append(b)
        Q.append(w / b)
    Tm = np.diag(alpha) + np.diag(beta[:len(alpha) - 1], 1) + np.diag(beta[:len(alpha) - 1], -1)
    return float(np.linalg.eigvalsh(Tm)[0])


@pytest.mark.parametrize("N,M", [(2, 5), (5, 5), (3, 7)])
def test_LL_ground_state_vs_exact_diagonalisation(N, M):
    T, V, p = workloads.lieb_liniger_TV(M, g=10.0, L=1.0)
    Hb, confs = brute.dense_H(N, M, T, V)
    assert np.abs(Hb - Hb.conj().T).max() < 1e-12
    E_ed = float(np.linalg.eigvalsh(Hb)[0])
    nc = len(confs)
    E_lz = lanczos_E0(N, M, T, V, iters=min(nc, 60))
    assert abs(E_lz - E_ed) < 1e-8 * max(1.0, abs(E_ed))
    assert E_ed > bethe_E0(N, 10.0)                       # truncated basis: variational upper bound
    # H commutes with total momentum: block structure
    P = np.array([sum(n[j] * p[j] for j in range(M)) for n in confs])
    assert np.abs(Hb[P[:, None] != P[None, :]]).max() == 0.0


def test_LL_energy_decreases_with_M_towards_bethe():
    # "the approximation is better as larger is the multiconfigurational space"
    N, g = 3, 10.0
    E = []
    for M in (3, 5, 7, 9):
        T, V, _ = workloads.lieb_liniger_TV(M, g=g)
        E.append(lanczos_E0(N, M, T, V, iters=50))
    Eb = bethe_E0(N, g)
    assert E[0] > E[1] > E[2] > E[3] > Eb
    assert E[3] - Eb < 0.25 * (E[0] - Eb)


def test_LL_momentum_sector_is_invariant():
    # a C supported on one total-momentum sector stays there under H (full oracle path, N=12)
    N, M = 12, 5
    nc = _nc(N, M)
    T, V, p = workloads.lieb_liniger_TV(M)
    occ = oracle.unrank(N, M, np.arange(nc))
    Ptot = occ @ p
    _, _, C = workloads.make_small_inputs(N, M, nc, seed=71)
    C = np.where(Ptot == 1, C, 0)
    HC, _ = oracle.hc_apply(N, M, T, V, C)
    assert np.abs(HC[Ptot != 1]).max() == 0.0 and np.abs(HC[Ptot == 1]).max() > 0


def test_extended_precision_reference_two_orbitals():
    """oracle.extended (M = 2, numpy longdouble) against the fp64 oracle: the same operator, and the size of the fp64
    oracle's OWN rounding.  For M = 2 the order of Eq. (14) gives |n_0, n_1> the index n_1 (checked against Algorithm 1).
    At N = 2000 (beyond the paper's range) the oracle's fp64 error is as large as the north-star tolerance
    1e-12 * ||T,V||max * ||C||_1 itself: that bound does not grow with the amplitudes (~N^2) and cannot be promised by ANY
    fp64 evaluation there -- which is why the one GPU test at N = 2000 uses the arithmetic bound."""
    from oracle import extended
    assert np.finfo(np.longdouble).nmant >= 63, "needs the x87 extended format"
    for N in (1, 2, 3, 7, 40, 300):
        assert (oracle.rank(N, 2, np.stack([N - np.arange(N + 1), np.arange(N + 1)], 1)) == np.arange(N + 1)).all()
        T, V, C = workloads.make_small_inputs(N, 2, N + 1, seed=4242 + 31 * N + 2, general_V=(N + 2) % 2 == 1)
        ref, _ = oracle.hc_apply(N, 2, T, V, C)
        ld = extended.hc_apply_m2_longdouble(N, T, V, C)
        assert float(np.abs(ref - ld).max()) <= 8 * 2.0 ** -53 * max(1.0, float(np.abs(ref).max())), N
        assert float(np.abs(ref - ld).max()) <= 0.25 * 1e-12 * max(np.abs(T).max(), np.abs(V).max()) * np.abs(C).sum(), N
    N = 2000
    T, V, C = workloads.make_small_inputs(N, 2, N + 1, seed=4242 + 31 * N + 2, general_V=(N + 2) % 2 == 1)
    ref, _ = oracle.hc_apply(N, 2, T, V, C)
    ld = extended.hc_apply_m2_longdouble(N, T, V, C)
    own = float(np.abs(ref - ld).max())
    t = 1e-12 * max(np.abs(T).max(), np.abs(V).max()) * np.abs(C).sum()
    assert own > 0.5 * t                                              # the fp64 oracle itself sits at the north-star bound here
    assert own <= 8 * 2.0 ** -53 * float(np.abs(ref).max())             # ... while being accurate to a few ulp of max|HC|
