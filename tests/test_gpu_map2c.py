"""GPU parity of the compact double-jump map (MCB_MAP2C) and of MCB_MAPS streaming it.

The table is integer work: offsets and every stride must equal oracle.map2_compact bit for bit.  hc_apply through it must
agree with the oracle within the north-star tolerance 1e-12 * ||T,V||max * ||C||_1."""
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
    build.build()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    m.lib()
    return m


def tol(T, V, C):
    return 1e-12 * max(np.abs(T).max(), np.abs(V).max()) * np.abs(C).sum()


SPACES = [(2, 2), (2, 5), (3, 3), (4, 5), (10, 5), (6, 4), (5, 7), (7, 6), (40, 3), (3, 9), (4, 12), (2, 12), (300, 2), (5, 10), (6, 8)]


@pytest.mark.parametrize("N,M", SPACES)
def test_map2c_bit_exact_and_maps_mode(mcb, N, M):
    sp = mcb.Space(N, M)
    nc, P = sp.nc, sp.P
    sp.build_structure(mcb.FOCK_TABLE)
    sp.build_structure(mcb.MAP2C)
    assert sp.structure_bytes(mcb.MAP2C) >= 4 * P * P * sp.nc2 + 8 * (nc + 1)
    off, ent = sp.map2c_export(0, nc)
    o_ref, s_ref, _ = oracle.map2_compact(N, M, 0, nc)
    assert off[0] == 0 and (off == o_ref).all()
    assert off[-1] == P * sp.nc2                                # forbidden removals take no memory
    assert ent.shape == s_ref.shape and (ent == s_ref).all()
    # a window
    if nc > 10:
        o2, e2 = sp.map2c_export(nc // 3, nc // 2)
        assert (o2 == o_ref[nc // 3: nc // 3 + nc // 2 + 1]).all() and (e2 == s_ref[o_ref[nc // 3]: o_ref[nc // 3 + nc // 2]]).all()
    # H.C through the compact map alone (T rides inside V): no single-jump map is built here
    T, V, C = workloads.make_small_inputs(N, M, nc, seed=5000 + 13 * N + M, general_V=(N + M) % 2 == 0)
    ref, _ = oracle.hc_apply(N, M, T, V, C)
    got = sp.hc_apply(T, V, torch.from_numpy(C).cuda(), mode=mcb.MAPS).cpu().numpy()
    assert np.abs(got - ref).max() <= tol(T, V, C)
    assert sp.last_apply_launches() == 1
    sp.close()


def test_map2c_needs_table_and_two_particles(mcb):
    sp = mcb.Space(5, 4)
    with pytest.raises(mcb.McbError) as e:
        sp.build_structure(mcb.MAP2C)                           # the allowed-removal counts come from the hashing table
    assert e.value.status == mcb.ENOTREADY
    one = mcb.Space(1, 4)
    with pytest.raises(mcb.McbError) as e:
        one.structure_bytes(mcb.MAP2C)                          # no two-particle removals with one particle
    assert e.value.status == mcb.EUNSUPPORTED
    sp.close(); one.close()


@pytest.mark.parametrize("cfg", [1, 2])
def test_map2c_full_size_windows_and_sampled_rows(mcb, cfg):
    c, T, V, (C,) = workloads.make_inputs(cfg)
    sp = mcb.Space(c.N, c.M)
    sp.build_structure(mcb.FOCK_TABLE)
    sp.build_structure(mcb.MAP2C)
    P = sp.P
    off_all, _ = sp.map2c_export(0, 0)
    tot, _ = sp.map2c_export(c.nc - 1, 1)
    assert tot[-1] == P * sp.nc2
    for b0 in (0, c.nc // 2 - 17, c.nc - 300):
        off, ent = sp.map2c_export(b0, 300)
        o_ref, s_ref, _ = oracle.map2_compact(c.N, c.M, b0, 300)
        assert (off - off[0] == o_ref).all() and (ent == s_ref).all()
    rows = workloads.sample_rows(c.nc, 48, 1500, workloads.seed_for(cfg, 31))
    ref, _ = oracle.hc_apply(c.N, c.M, T, V, C, rows=rows)
    dC = torch.from_numpy(C).cuda()
    out = sp.hc_apply(T, V, dC, mode=mcb.MAPS)
    assert np.abs(out[torch.from_numpy(rows).cuda()].cpu().numpy() - ref).max() <= tol(T, V, C)
    base = sp.hc_apply(T, V, dC, mode=mcb.GEMM)
    assert float((out - base).abs().max()) <= tol(T, V, C)      # everywhere, not only on the sample
    sp.close()
