"""mcb_hc_apply_host in the GEMM and SPARSE modes: C streams to the device in pieces, the kernels run slab by slab (slabs cut by
the occupation of the last orbital) behind the arrival of the prefix of C each slab gathers from, and finished slabs of HC go
back while the next one computes.  A slab that started before its data was there, or read beyond its prefix, would pick up the
NaN the scratch vectors are poisoned with."""
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
    build.build()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    m.lib()
    return m


@pytest.mark.parametrize("N,M,kind,mode", [(20, 8, "dense", "GEMM"), (10, 12, "dense", "GEMM"), (60, 5, "ll", "SPARSE"), (1000, 3, "dense", "GEMM"),
                                           (24, 7, "bh", "AUTO")])
def test_host_apply_slab_pipeline(mcb, N, M, kind, mode):
    sp = mcb.Space(N, M)
    assert sp.nc >= 1 << 18                                         # large enough for the pipelined path
    T, V, C = workloads.make_small_inputs(N, M, sp.nc, seed=808 + N + M, kind=kind)
    rows = workloads.sample_rows(sp.nc, 1024, 4000, 5 + N)
    ref, _ = oracle.hc_apply(N, M, T, V, C, rows=rows)
    t = 1e-12 * max(np.abs(T).max(), np.abs(V).max()) * np.abs(C).sum()
    sp.build_structure(mcb.FOCK_TABLE)
    m = getattr(mcb, mode)
    resolved = sp.resolve_mode(T, V, m)
    assert resolved in (mcb.GEMM, mcb.SPARSE)
    dev = sp.hc_apply(T, V, torch.from_numpy(C).cuda(), mode=m).cpu().numpy()
    assert float(np.abs(dev[rows] - ref).max()) <= t
    hC = torch.from_numpy(C).pin_memory()
    out = torch.empty_like(hC).pin_memory()
    for it in range(3):
        for name in ("dC", "dHC"):
            if name in sp._workspace:
                sp._workspace[name].fill_(float("nan"))
        out.fill_(float("nan"))
        got = sp.hc_apply_host(T, V, hC, out_host=out, mode=m).numpy()
        assert np.isfinite(got.view(np.float64)).all(), it
        assert (got == dev).all(), it                                # same kernels, same order of summation: same bits
    # pageable vectors take the plain copy - apply - copy path
    plain = sp.hc_apply_host(T, V, C.copy(), mode=m).numpy()
    assert (plain == dev).all()
    sp.close()
