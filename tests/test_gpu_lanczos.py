"""GPU parity of mcb_lanczos + mcb_tridiag_eigvals against the numpy Lanczos oracle, exact
diagonalisation and the Bethe-ansatz value (Eq. 17-18).  The Ritz values under test come from the PRODUCT's own host
eigen-solver (mcb.tridiag_eigvals); the oracle's (numpy eigvalsh of the dense tridiagonal matrix) is what they are compared with."""
import math

import numpy as np
import pytest

import oracle
import workloads
from oracle import brute
from oracle import lanczos as olz
from test_oracle_apply import bethe_E0

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def mcb():
    import paper_2005_13679_b200 as m
    from paper_2005_13679_b200 import build
    build.build()    # no-op when libmcb.so is current; the library normally travels with the snapshot
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    m.lib()
    return m


@pytest.mark.parametrize("N,M,kind", [(3, 3, "dense"), (5, 5, "ll"), (6, 4, "dense"), (8, 7, "ll"), (4, 9, "dense"), (1, 4, "dense")])
def test_lanczos_matches_oracle(mcb, N, M, kind):
    sp = mcb.Space(N, M)
    nc = sp.nc
    T, V, C = workloads.make_small_inputs(N, M, nc, seed=300 + N + M, kind=kind)
    sp.build_structure(mcb.FOCK_TABLE)
    k = min(nc, 30)
    a_ref, b_ref, _ = olz.lanczos(N, M, T, V, C, k)
    a, b = sp.lanczos(T, V, torch.from_numpy(C).cuda(), k)
    assert len(a) == len(a_ref)
    scale = max(1.0, np.abs(a_ref).max())
    # the recurrence amplifies rounding differences as Ritz values converge: compare the first steps tightly, the
    # extremal Ritz value (what the method is for) over the whole run
    e = min(8, len(a))
    assert np.abs(a[:e] - a_ref[:e]).max() < 1e-9 * scale and np.abs(b[:e] - b_ref[:e]).max() < 1e-9 * scale
    ritz = mcb.tridiag_eigvals(a, b[:-1])                      # the product's own host solve
    assert np.abs(ritz - olz.ritz_values(a, b)).max() < 1e-12 * scale         # ... against numpy on the same tridiagonal matrix
    assert abs(ritz[0] - olz.ritz_values(a_ref, b_ref)[0]) < 1e-9 * scale
    if k == nc:                                               # complete Krylov space: the whole spectrum of the dense H
        H, _ = brute.dense_H(N, M, T, V)
        assert np.abs(ritz - np.linalg.eigvalsh(H)).max() < 1e-8 * scale
    sp.close()


@pytest.mark.parametrize("mode", ["GEMM", "RUNS", "REHASH", "SPARSE", "MAPS"])
def test_lanczos_every_mode_stages_coefficients_once(mcb, mode):
    """mcb_lanczos packs and uploads T, V in its first H.C only (every mode keeps what it staged for the rest of the run): the
    coefficients of ALL steps must still be the oracle's, and the hold must be gone afterwards -- an apply with other matrix
    elements right after the run uses its own."""
    N, M = 6, 5                                                   # (the Lieb-Liniger list wants an odd M)
    sp = mcb.Space(N, M)
    nc = sp.nc
    T, V, C = workloads.make_small_inputs(N, M, nc, seed=911, kind="ll" if mode == "SPARSE" else "dense")
    sp.build_structure(mcb.FOCK_TABLE)
    if mode == "MAPS":
        sp.build_structure(mcb.MAP2C)
    k = 20
    a_ref, b_ref, _ = olz.lanczos(N, M, T, V, C, k)
    a, b = sp.lanczos(T, V, torch.from_numpy(C).cuda(), k, mode=getattr(mcb, mode))
    assert not sp.lanczos_truncated and len(a) == len(a_ref)
    scale = max(1.0, np.abs(a_ref).max())
    assert np.abs(a[:8] - a_ref[:8]).max() < 1e-9 * scale and np.abs(b[:8] - b_ref[:8]).max() < 1e-9 * scale
    assert abs(mcb.tridiag_eigvals(a, b[:-1])[0] - olz.ritz_values(a_ref, b_ref)[0]) < 1e-9 * scale
    T2, V2, C2 = workloads.make_small_inputs(N, M, nc, seed=912, kind="dense")
    ref, _ = oracle.hc_apply(N, M, T2, V2, C2)
    got = sp.hc_apply(T2, V2, torch.from_numpy(C2).cuda(), mode=getattr(mcb, mode) if mode != "SPARSE" else mcb.AUTO).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-12 * max(np.abs(T2).max(), np.abs(V2).max()) * np.abs(C2).sum()
    sp.close()


def test_lanczos_lieb_liniger_ground_state_vs_ed(mcb):
    # the paper's end-to-end use, shrunk: N = 5 bosons, M = 5 plane waves, g = 10
    N, M = 5, 5
    sp = mcb.Space(N, M)
    T, V, _ = workloads.lieb_liniger_TV(M)
    H, _ = brute.dense_H(N, M, T, V)
    e_ed = np.linalg.eigvalsh(H)[0]
    sp.build_structure(mcb.FOCK_TABLE)
    v0 = workloads.random_normalised_C(sp.nc, np.random.default_rng(11))
    a, b = sp.lanczos(T, V, torch.from_numpy(v0).cuda(), 60)
    assert abs(mcb.tridiag_eigvals(a, b[:-1])[0] - e_ed) < 1e-9 * abs(e_ed)
    sp.close()


def test_lanczos_paper_run_N5_M11_vs_bethe(mcb):
    # the paper's own ground-state run: N = 5, M = 11 plane waves, nc / 8 Lanczos iterations, E0 from the
    # tridiagonal solve -- everything from the product; the truncated basis gives an upper bound of the Bethe value (Eq. 17-18)
    # that improves on the M = 5 one
    N, g = 5, 10.0
    e_bethe = bethe_E0(N, g)
    e0 = {}
    for M in (5, 11):
        sp = mcb.Space(N, M)
        T, V, _ = workloads.lieb_liniger_TV(M, g=g)
        sp.build_structure(mcb.FOCK_TABLE)
        v0 = workloads.random_normalised_C(sp.nc, np.random.default_rng(5 + M))
        steps = sp.lanczos_steps(0)
        assert steps == max(1, min(1024, sp.nc // 8))                 # the paper's cap
        a, b = sp.lanczos(T, V, torch.from_numpy(v0).cuda(), 0)
        assert len(a) <= steps
        e0[M] = mcb.tridiag_eigvals(a, b[:-1])[0]
        sp.close()
    assert e0[5] > e0[11] > e_bethe
    # M = 11 against the dense spectrum of the oracle's operator restricted to the same Krylov question: the numpy oracle run
    T, V, _ = workloads.lieb_liniger_TV(11, g=g)
    v0 = workloads.random_normalised_C(math.comb(N + 10, 10), np.random.default_rng(16))
    a_ref, b_ref, _ = olz.lanczos(N, 11, T, V, v0, 120)
    assert abs(e0[11] - olz.ritz_values(a_ref, b_ref)[0]) < 1e-6 * abs(e0[11])


def test_lanczos_full_size_lieb_liniger_runs_and_converges(mcb):
    # configs[1] (N = 100, M = 5, nc = 4.6e6): 24 steps; the lowest Ritz value can only go down as the space grows
    c, T, V, (C,) = workloads.make_inputs(1)
    sp = mcb.Space(c.N, c.M)
    sp.build_structure(mcb.FOCK_TABLE)
    a, b = sp.lanczos(T, V, torch.from_numpy(C).cuda(), 24)
    assert len(a) == 24 and np.isfinite(a).all() and (b > 0).all()
    lows = [mcb.tridiag_eigvals(a[:k], b[:max(k - 1, 0)])[0] for k in range(1, 25)]
    assert all(lows[i + 1] <= lows[i] + 1e-9 * abs(lows[0]) for i in range(23))
    # alpha_0 is the Rayleigh quotient <C|H|C> of the start vector
    HC = sp.hc_apply(T, V, torch.from_numpy(C).cuda())
    assert abs(a[0] - torch.vdot(torch.from_numpy(C).cuda(), HC).real.item()) < 1e-9 * abs(a[0])
    sp.close()
