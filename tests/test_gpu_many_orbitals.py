"""GPU parity for MANY orbitals (12 < M <= 32): the paper's second sweep, N = 5 with M up to 25, and its ground-state runs
N = 5, M = 11 and 21.  hc_apply, rho and lanczos through the generic path
(csrc/mcb_apply_big.cu) against the CPU oracle; tolerance of the north star, 1e-12 * ||T,V||max * ||C||_1."""
import math

import numpy as np
import pytest

import oracle
import workloads
from test_oracle_apply import bethe_E0

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def mcb():
    import paper_2005_13679_b200 as m
    from paper_2005_13679_b200 import build
    build.build()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    m.lib()
    return m


def tol(T, V, C):
    return 1e-12 * max(np.abs(T).max(), np.abs(V).max()) * np.abs(C).sum()


@pytest.mark.parametrize("N,M,nrows", [(5, 13, 0), (2, 14, 0), (1, 20, 0), (4, 16, 0), (5, 21, 6000), (5, 25, 4000), (3, 32, 0), (6, 14, 3000),
                                          (8, 14, 2000)])            # nc2 = 27,132: 424 column tiles with a ragged tail, 2 row tiles
def test_hc_apply_many_orbitals(mcb, N, M, nrows):
    sp = mcb.Space(N, M)
    nc = sp.nc
    assert nc == math.comb(N + M - 1, M - 1)
    T, V, C = workloads.make_small_inputs(N, M, nc, seed=9000 + 37 * N + M, general_V=(N + M) % 2 == 0)
    rows = None if nrows == 0 else workloads.sample_rows(nc, 8, nrows, 3)       # the ordered M^4 oracle is slow here
    ref, _ = oracle.hc_apply(N, M, T, V, C, rows=rows)
    sp.build_structure(mcb.FOCK_TABLE)
    dC = torch.from_numpy(C).cuda()
    got = sp.hc_apply(T, V, dC).cpu().numpy()
    if rows is not None:
        got = got[rows]
    err = np.abs(got - ref).max()
    assert err <= tol(T, V, C), (err, tol(T, V, C))
    assert sp.resolve_mode(T, V) == mcb.GEMM and sp.last_apply_launches() == (2 if N >= 2 else 1)
    # host path and a second call through the same workspace
    again = sp.hc_apply_host(T, V, C).numpy()
    assert np.array_equal(again if rows is None else again[rows], got)
    sp.close()


@pytest.mark.parametrize("N,M", [(3, 13), (5, 14), (1, 15), (2, 20)])
def test_rho_many_orbitals(mcb, N, M):
    sp = mcb.Space(N, M)
    T, V, C = workloads.make_small_inputs(N, M, sp.nc, seed=9100 + N + M)
    if N >= 2:
        sp.build_structure(mcb.FOCK_TABLE)
    r1, r2 = sp.rho(torch.from_numpy(C).cuda())
    r1_ref, r2_ref = oracle.rho(N, M, C)
    scale = max(1.0, N * (N - 1))
    assert np.abs(r1.cpu().numpy() - r1_ref).max() <= 1e-12 * scale
    assert np.abs(r2.cpu().numpy() - r2_ref).max() <= 1e-12 * scale
    sp.close()


def test_lanczos_paper_run_N5_M21_vs_bethe(mcb):
    # N = 5, M = 11 and 21 plane waves, nc / 8 Lanczos iterations (capped at 1024 here), E0 from the host
    # tridiagonal solve; the energy lies above the Bethe value of Eq. 17-18 and comes closer as M grows
    N, g = 5, 10.0
    e_bethe = bethe_E0(N, g)
    e0 = {}
    for M in (11, 21):
        sp = mcb.Space(N, M)
        T, V, _ = workloads.lieb_liniger_TV(M, g=g)
        sp.build_structure(mcb.FOCK_TABLE)
        v0 = workloads.random_normalised_C(sp.nc, np.random.default_rng(40 + M))
        a, b = sp.lanczos(T, V, torch.from_numpy(v0).cuda(), 0 if M == 11 else 200)
        assert not sp.lanczos_truncated                           # nc / 8 = 375 at M = 11; an explicit kmax is never "truncated"
        e0[M] = mcb.tridiag_eigvals(a, b[:-1])[0]
        sp.close()
    assert e0[11] > e0[21] > e_bethe
    assert (e0[21] - e_bethe) < 0.6 * (e0[11] - e_bethe)         # the truncation error shrinks markedly from M = 11 to 21


def test_lanczos_reports_when_the_paper_cap_is_cut(mcb):
    # N = 5, M = 21 runs nc / 8 = 6,641 iterations in the paper; the library stops at 1,024 and must say so
    N, M, g = 5, 21, 10.0
    sp = mcb.Space(N, M)
    assert sp.nc // 8 == 6641 and sp.lanczos_steps(0) == 1024
    T, V, _ = workloads.lieb_liniger_TV(M, g=g)
    sp.build_structure(mcb.FOCK_TABLE)
    v0 = torch.from_numpy(workloads.random_normalised_C(sp.nc, np.random.default_rng(61))).cuda()
    a200, b200 = sp.lanczos(T, V, v0, 200)
    assert not sp.lanczos_truncated
    a, b = sp.lanczos(T, V, v0, 0)
    assert sp.lanczos_truncated and len(a) == 1024                # MCB_TRUNCATED: a completed, shortened run
    assert np.abs(a[:200] - a200).max() <= 1e-9 * np.abs(a200).max()          # same run, continued
    e200, e1024 = mcb.tridiag_eigvals(a200, b200[:-1])[0], mcb.tridiag_eigvals(a, b[:-1])[0]
    assert bethe_E0(N, g) < e1024 <= e200 + 1e-9 * abs(e200)
    sp.close()
