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


SPACES = [(2, 1), (5, 1), (2, 2), (2, 5), (3, 3), (4, 5), (10, 5), (6, 4), (5, 7), (7, 6), (40, 3), (3, 9), (4, 12), (2, 12), (300, 2), (5, 10), (6, 8)]


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


@pytest.mark.parametrize("N,M", [(3, 13), (2, 16), (4, 14)])
def test_map2c_many_orbitals_bit_exact(mcb, N, M):
    """More than 12 orbitals: the run-time-M fill kernel builds the table (no MCB_MAPS kernel reads it there)."""
    sp = mcb.Space(N, M)
    sp.build_structure(mcb.FOCK_TABLE)
    sp.build_structure(mcb.MAP2C)
    off, ent = sp.map2c_export(0, sp.nc)
    o_ref, s_ref, _ = oracle.map2_compact(N, M, 0, sp.nc)
    assert (off == o_ref).all() and off[-1] == sp.P * sp.nc2
    assert ent.shape == s_ref.shape and (ent == s_ref).all()
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


def _stratified_rows(c, n_random, seed):
    """Indices (oracle Algorithm 1) of configurations covering every top occupation 0..N and every number of occupied
    orbitals 1..min(N, M), plus head, tail and n_random random rows (the recipe of tests/test_gpu_fullvector.py)."""
    rng = np.random.default_rng(seed)
    N, M = c.N, c.M
    occs = []

    def composition(total, parts, positive):
        if parts == 1:
            return [total]
        if positive:
            cuts = np.sort(rng.choice(np.arange(1, total), size=parts - 1, replace=False))
        else:
            cuts = np.sort(rng.integers(0, total + 1, size=parts - 1))
        return np.diff(np.concatenate([[0], cuts, [total]])).tolist()

    for j in range(N + 1):
        for _ in range(6):
            occs.append(composition(N - j, M - 1, False) + [j])
    for k in range(1, min(N, M) + 1):
        for _ in range(24):
            where = np.sort(rng.choice(M, size=k, replace=False))
            v = np.zeros(M, dtype=np.int64)
            v[where] = composition(N, k, True)
            occs.append(v.tolist())
    occ = np.asarray(occs, dtype=np.int32)
    strat = oracle.rank(N, M, occ).astype(np.int64)
    return np.unique(np.concatenate([strat, workloads.sample_rows(c.nc, 64, n_random, seed + 1)]))


@pytest.mark.parametrize("cfg", [3, 4])
def test_map2c_and_maps_beyond_2_31_entries(mcb, cfg):
    """configs[3] / [4]: the compact table has 1.42e10 / 1.52e10 int32 entries (57 / 61 GB), the only sizes at which its 64-bit
    offset arithmetic (stride offset x P, line offset x P) leaves the int32 range.  Lines are compared with
    oracle.map2_compact in windows at the head, at the first line whose entry offset exceeds 2^31, in the middle and over the
    last 300 lines; MCB_MAPS over the table with the oracle on >= 1e4 stratified rows and with MCB_GEMM on every output.
    configs[3] then repeats the apply over the dense planes (Map1 4 GB + Map2 121 GB: plane offsets a * P * ld beyond 2^31
    elements); at configs[4] the dense Map2 needs 188 GB and does not exist on a 180 GB device."""
    c, T, V, (C,) = workloads.make_inputs(cfg)
    sp = mcb.Space(c.N, c.M)
    P, nc = sp.P, c.nc
    sp.build_structure(mcb.FOCK_TABLE)
    assert sp.structure_bytes(mcb.MAP2C) > 4 * 2 ** 31          # more than 2^31 entries
    sp.build_structure(mcb.MAP2C)
    off_all, _ = sp.map2c_export(0, 0)
    tot, _ = sp.map2c_export(nc - 1, 1)
    assert off_all[0] == 0 and tot[-1] == P * sp.nc2 and tot[-1] * P > 2 ** 33
    # first line whose entries start beyond 2^31 int32 elements: bisection on the exported offsets
    lo, hi = 0, nc - 1
    while lo < hi:
        mid = (lo + hi) // 2
        o, _ = sp.map2c_export(mid, 0)
        if o[0] * P > 2 ** 31:
            hi = mid
        else:
            lo = mid + 1
    assert 0 < lo < nc - 400
    for b0, cnt in ((0, 200), (lo - 100, 200), (nc // 2 - 17, 200), (nc - 300, 300)):
        off, ent = sp.map2c_export(b0, cnt)
        o_ref, s_ref, _ = oracle.map2_compact(c.N, c.M, b0, cnt)
        assert (off - off[0] == o_ref).all() and ent.shape == s_ref.shape and (ent == s_ref).all(), b0
    o_last, _ = sp.map2c_export(nc - 300, 0)
    assert o_last[0] * P > 2 ** 33                              # the last window sits far beyond the int32 range
    rows = _stratified_rows(c, 10_000, workloads.seed_for(cfg, 33))
    assert rows.size >= 10_000
    ref, _ = oracle.hc_apply(c.N, c.M, T, V, C, rows=rows)
    dC = torch.from_numpy(C).cuda()
    drows, dref = torch.from_numpy(rows).cuda(), torch.from_numpy(ref).cuda()
    t = tol(T, V, C)
    base = sp.hc_apply(T, V, dC, mode=mcb.GEMM)
    out = sp.hc_apply(T, V, dC, mode=mcb.MAPS)                  # FOCK_TABLE + MAP2C attached: streams the compact table
    assert sp.last_apply_launches() == 1
    err = float((out[drows] - dref).abs().max())
    print(f"cfg {cfg} MAPS/compact: max err over {rows.size} stratified rows {err:.3e}, vs GEMM everywhere "
          f"{float((out - base).abs().max()):.3e} (tol {t:.3e})")
    assert err <= t
    assert float((out - base).abs().max()) <= t
    sp.drop_structure(mcb.MAP2C)
    del out
    torch.cuda.empty_cache()
    dense = sp.structure_bytes(mcb.MAP1) + sp.structure_bytes(mcb.MAP2)
    free, _ = torch.cuda.mem_get_info()
    if cfg == 4:
        assert dense > 180e9                                    # 7.7e6 x 78^2 x 4 bytes: no dense planes at configs[4]
    elif dense + (2 << 30) > free:
        pytest.skip(f"dense Map1 + Map2 need {dense / 1e9:.0f} GB, {free / 1e9:.0f} GB free on this device")
    else:
        sp.build_structure(mcb.MAP1)
        sp.build_structure(mcb.MAP2)
        # one window of the dense map whose plane offsets are beyond 2^31: the last configurations, all P x P planes
        m2 = sp.map2_export(nc - 64, 64)
        assert (m2 == oracle.map2(c.N, c.M, nc - 64, 64)).all()
        out = sp.hc_apply(T, V, dC, mode=mcb.MAPS)              # dense planes attached: one thread per configuration
        err = float((out[drows] - dref).abs().max())
        print(f"cfg {cfg} MAPS/dense: max err over {rows.size} stratified rows {err:.3e}, vs GEMM everywhere "
              f"{float((out - base).abs().max()):.3e}")
        assert err <= t
        assert float((out - base).abs().max()) <= t
        sp.drop_structure(mcb.MAP2)
        sp.drop_structure(mcb.MAP1)
    sp.close()
    torch.cuda.empty_cache()
