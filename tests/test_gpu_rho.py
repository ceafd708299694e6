"""GPU parity of mcb_rho (Eq. 10-11) against the CPU oracle, through the C ABI binding.

rho2 is a sum of nc2 * P^2-term products of magnitude <= N^2 |C|^2; for a normalised C its entries are bounded by
N (N - 1), and any fp64 summation order agrees to a few ulp of that: tolerance 1e-12 * N * max(N - 1, 1).
"""
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


def rtol(N):
    return 1e-12 * N * max(N - 1, 1)


SPACES = [(1, 1), (1, 4), (4, 1), (2, 2), (2, 5), (3, 3), (10, 5), (6, 4), (5, 7), (40, 3), (4, 12), (300, 2), (5, 10), (6, 8), (60, 4)]


@pytest.mark.parametrize("N,M", SPACES)
def test_rho_matches_oracle(mcb, N, M):
    sp = mcb.Space(N, M)
    nc = sp.nc
    C = workloads.random_normalised_C(nc, np.random.default_rng(5000 + 13 * N + M))
    r1_ref, r2_ref = oracle.rho(N, M, C)
    if N >= 2:
        sp.build_structure(mcb.FOCK_TABLE)
    r1, r2 = sp.rho(torch.from_numpy(C).cuda())
    r1, r2 = r1.cpu().numpy(), r2.cpu().numpy()
    assert np.abs(r1 - r1_ref).max() <= rtol(N), np.abs(r1 - r1_ref).max()
    assert np.abs(r2 - r2_ref).max() <= rtol(N), np.abs(r2 - r2_ref).max()
    # deterministic: a second call gives the same bits
    r1b, r2b = sp.rho(torch.from_numpy(C).cuda())
    assert (r1b.cpu().numpy() == r1).all() and (r2b.cpu().numpy() == r2).all()
    sp.close()


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_rho_full_size_invariants_and_energy(mcb, cfg):
    # full-size configs: the oracle's O(nc M^4 N) double sum is out of reach, so check what holds at any size --
    # traces of the number operator, Hermiticity, and <C|H|C> from hc_apply against sum T.rho1 + 1/2 sum V.rho2
    c, T, V, (C,) = workloads.make_inputs(cfg)
    sp = mcb.Space(c.N, c.M)
    sp.build_structure(mcb.FOCK_TABLE)
    dC = torch.from_numpy(C).cuda()
    r1, r2 = sp.rho(dC)
    r1, r2 = r1.cpu().numpy(), r2.cpu().numpy()
    N = c.N
    assert abs(np.trace(r1) - N) <= rtol(N)
    assert abs(np.einsum("ksks->", r2) - N * (N - 1)) <= 10 * rtol(N)
    assert np.abs(r1 - r1.conj().T).max() <= rtol(N)
    assert np.abs(r2 - r2.conj().transpose(3, 2, 1, 0)).max() <= rtol(N)
    HC = sp.hc_apply(T, V, dC)
    e_apply = torch.vdot(dC, HC).item()
    e_rho = np.einsum("kl,kl->", T, r1) + 0.5 * np.einsum("ksql,ksql->", V, r2)
    scale = max(np.abs(T).max(), np.abs(V).max()) * N * N
    assert abs(e_apply - e_rho) <= 1e-11 * scale * c.M ** 2, (e_apply, e_rho)
    sp.close()
