"""mcb_rho_static -- the allocation-free entry point of libmcb -- against mcb_rho, the existing path with a caller workspace.

Why the entry point exists: some users of the library cannot allocate device memory at the moment they need the density
matrices (Eq. 10-11).  A plug-in is handed C and the result buffers by its host program and owns no
allocator; a job's memory pool took the whole GPU at start-up, so one more cudaMalloc fails; a time-propagation loop must not
call cudaMalloc / cudaFree because they synchronise the device and stall every other stream.  mcb_rho asks such a caller for
mcb_rho_workspace_bytes() of scratch it cannot produce; mcb_rho_static keeps that scratch in a fixed 8 MiB array inside
libmcb.so instead (M <= 12), shared by every call on the device.

What is checked, always on TWO CALLS IN A ROW per space (the array keeps what the previous call wrote, so the second call
is the one that would see stale partial sums if a call ever read a word it had not written itself):
  * both calls agree with mcb_rho on the same input within the tolerance of tests/test_gpu_rho.py, 1e-12 N max(N-1, 1)
    (the static variant may run a smaller grid, i.e. another summation order, so equality of bits is not demanded);
  * the calls use different states and, between repeats, a space of another shape dirties the array;
  * repeating a call reproduces its own bits (no dependence on the array's previous contents);
  * M beyond the limit is refused with MCB_ESCRATCH and leaves the outputs alone.
The file sorts last on purpose (pytest -x stops at the first failure: a failure here hides no other test) and builds what
it needs itself, so it passes alone in a fresh process as well as after the rest of the suite.
"""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def mcb():
    import paper_2005_13679_b200 as m
    from paper_2005_13679_b200 import build
    build.build()    # no-op when libmcb.so is current
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    m.lib()
    return m


def rtol(N):
    return 1e-12 * N * max(N - 1, 1)


def _state(nc, seed):
    return torch.from_numpy(workloads.random_normalised_C(nc, np.random.default_rng(seed))).cuda()


def _close(a, b, N):
    return (a - b).abs().max().item() <= rtol(N)


# (N, M): N = 1 (no Gram kernel), one orbital, full-grid shapes (M = 2, 6, 7) and shapes whose grid the 8 MiB array cuts
# (M = 3..5, M >= 8), several tiles with a ragged tail
SPACES = [(1, 4), (4, 1), (300, 2), (40, 3), (60, 4), (10, 5), (7, 6), (5, 7), (6, 8), (5, 10), (4, 12)]


@pytest.mark.parametrize("N,M", SPACES)
def test_rho_static_matches_rho_on_two_calls_in_a_row(mcb, N, M):
    sp = mcb.Space(N, M)
    if N >= 2:
        sp.build_structure(mcb.FOCK_TABLE)
    Ca, Cb = _state(sp.nc, 9100 + 17 * N + M), _state(sp.nc, 9200 + 17 * N + M)
    ref_a, ref_b = sp.rho(Ca), sp.rho(Cb)                                # existing path, caller workspace
    # the caller's own output buffers, filled with a value no density matrix of a normalised state can hold
    r1 = torch.full((M, M), 7e77, dtype=torch.complex128, device="cuda")
    r2 = torch.full((M,) * 4, 7e77, dtype=torch.complex128, device="cuda")
    got = sp.rho_static(Ca, r1, r2)                                      # call 1
    assert got[0] is r1 and got[1] is r2
    a1, a2 = r1.clone(), r2.clone()
    sp.rho_static(Cb, r1, r2)                                            # call 2, straight after, other state
    b1, b2 = r1.clone(), r2.clone()
    assert _close(a1, ref_a[0], N) and _close(a2, ref_a[1], N)
    assert _close(b1, ref_b[0], N) and _close(b2, ref_b[1], N)
    # dirty the shared array through a space of another shape, then repeat call 1: same bits as before
    other = mcb.Space(9, 5)
    other.build_structure(mcb.FOCK_TABLE)
    other.rho_static(_state(other.nc, 77))
    c1, c2 = sp.rho_static(Ca)
    assert torch.equal(c1, a1) and torch.equal(c2, a2)
    other.close()
    sp.close()


def test_rho_static_full_size_config(mcb):
    # BASELINE.json configs[2] (N = 400, M = 4): 1.07e7 intermediates over a grid the array cuts from 592 blocks to 227
    c, _, _, (C,) = workloads.make_inputs(2)
    sp = mcb.Space(c.N, c.M)
    sp.build_structure(mcb.FOCK_TABLE)
    dC = torch.from_numpy(C).cuda()
    ref1, ref2 = sp.rho(dC)
    for _ in range(2):
        r1, r2 = sp.rho_static(dC)
        assert _close(r1, ref1, c.N) and _close(r2, ref2, c.N)
        assert abs(torch.trace(r1).item() - c.N) <= rtol(c.N)
    sp.close()


def test_rho_static_refuses_sizes_beyond_its_array(mcb):
    sp = mcb.Space(3, mcb.RHO_STATIC_MAX_M + 1)
    sp.build_structure(mcb.FOCK_TABLE)
    C = _state(sp.nc, 5)
    r1 = torch.full((sp.M, sp.M), 3.0, dtype=torch.complex128, device="cuda")
    r2 = torch.full((sp.M,) * 4, 3.0, dtype=torch.complex128, device="cuda")
    with pytest.raises(mcb.McbError) as e:
        sp.rho_static(C, r1, r2)
    assert e.value.status == mcb.ESCRATCH and "scratch" in str(e.value)
    torch.cuda.synchronize()
    assert (r1 == 3.0).all() and (r2 == 3.0).all()                       # nothing was launched
    sp.rho(C)                                                            # the path with a workspace serves this size
    sp.close()
