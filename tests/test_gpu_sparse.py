"""GPU parity of MCB_SPARSE (structured matrix elements) against the CPU oracle."""
import math

import numpy as np
import pytest

import oracle
import workloads

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


def tol(T, V, C):
    return 1e-12 * max(np.abs(T).max(), np.abs(V).max()) * np.abs(C).sum()


CASES = [(1, 4, "bh"), (2, 2, "bh"), (5, 5, "ll"), (8, 7, "ll"), (6, 6, "bh"), (4, 12, "bh"), (12, 3, "ll"), (40, 3, "bh"),
         (3, 3, "dense"), (6, 4, "dense"), (4, 7, "dense"), (30, 5, "ll"),
         # more than 12 orbitals (run-time-M kernel): a 16-site and a 20-site Bose-Hubbard ring, plane waves with 13 momenta,
         # a 32-site ring with two particles, and one particle on 14 sites
         (4, 16, "bh"), (3, 20, "bh"), (4, 13, "ll"), (2, 32, "bh"), (1, 14, "bh")]


@pytest.mark.parametrize("N,M,kind", CASES)
def test_sparse_matches_oracle(mcb, N, M, kind):
    sp = mcb.Space(N, M)
    T, V, C = workloads.make_small_inputs(N, M, sp.nc, seed=600 + 7 * N + M, kind=kind, general_V=(kind == "dense"))
    ref, _ = oracle.hc_apply(N, M, T, V, C)
    sp.build_structure(mcb.FOCK_TABLE)
    dC = torch.from_numpy(C).cuda()
    got = sp.hc_apply(T, V, dC, mode=mcb.SPARSE).cpu().numpy()
    assert np.abs(got - ref).max() <= tol(T, V, C)
    assert sp.last_apply_launches() == 1
    # MCB_AUTO takes the sparse path for the structured workloads and the dense one otherwise; same answer either way
    resolved = sp.resolve_mode(T, V)
    if kind in ("ll", "bh") and not (M > 12 and N < 2):          # (one particle on many orbitals: MCB_AUTO keeps the M x M mat-vec)
        assert resolved == mcb.SPARSE
    else:
        assert resolved != mcb.SPARSE
    auto = sp.hc_apply(T, V, dC).cpu().numpy()
    assert np.abs(auto - ref).max() <= tol(T, V, C)
    sp.close()


def test_sparse_refuses_long_lists(mcb):
    N, M = 3, 8                                  # dense V: P (P - 1) = 1260 off-diagonal entries > 1024
    sp = mcb.Space(N, M)
    T, V, C = workloads.make_small_inputs(N, M, sp.nc, seed=5)
    sp.build_structure(mcb.FOCK_TABLE)
    with pytest.raises(mcb.McbError) as e:
        sp.hc_apply(T, V, torch.from_numpy(C).cuda(), mode=mcb.SPARSE)
    assert e.value.status == mcb.EUNSUPPORTED
    sp.close()


def test_sparse_full_size_lieb_liniger_sampled_rows(mcb):
    c, T, V, (C,) = workloads.make_inputs(1)     # configs[1]: N = 100, M = 5, 29 of 225 packed elements non-zero
    sp = mcb.Space(c.N, c.M)
    sp.build_structure(mcb.FOCK_TABLE)
    rows = workloads.sample_rows(c.nc, 48, 1500, workloads.seed_for(1, 9))
    ref, _ = oracle.hc_apply(c.N, c.M, T, V, C, rows=rows)
    dC = torch.from_numpy(C).cuda()
    assert sp.resolve_mode(T, V) == mcb.SPARSE
    got = sp.hc_apply(T, V, dC)[torch.from_numpy(rows).cuda()].cpu().numpy()
    assert np.abs(got - ref).max() <= tol(T, V, C)
    runs = sp.hc_apply(T, V, dC, mode=mcb.RUNS)[torch.from_numpy(rows).cuda()].cpu().numpy()
    assert np.abs(runs - ref).max() <= tol(T, V, C)
    sp.close()


def test_bose_hubbard_mid_size(mcb):
    N, M = 12, 10                                # nc = 293,930
    sp = mcb.Space(N, M)
    T, V = workloads.bose_hubbard_TV(M)
    C = workloads.random_normalised_C(sp.nc, np.random.default_rng(3))
    sp.build_structure(mcb.FOCK_TABLE)
    rows = workloads.sample_rows(sp.nc, 32, 800, 17)
    ref, _ = oracle.hc_apply(N, M, T, V, C, rows=rows)
    dC = torch.from_numpy(C).cuda()
    got = sp.hc_apply(T, V, dC)[torch.from_numpy(rows).cuda()].cpu().numpy()
    assert sp.resolve_mode(T, V) == mcb.SPARSE
    assert np.abs(got - ref).max() <= tol(T, V, C)
    gemm = sp.hc_apply(T, V, dC, mode=mcb.GEMM)[torch.from_numpy(rows).cuda()].cpu().numpy()
    assert np.abs(gemm - ref).max() <= tol(T, V, C)
    sp.close()
