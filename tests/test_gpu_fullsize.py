"""GPU parity at BASELINE.json's full sizes (configs 1-4), in the launch configuration bench.py times.

The oracle cannot produce the whole vector in seconds at these sizes, so (task statement, parity rules):
  * sampled outputs: a seeded row subset (head, tail, random rows; rows of H.C are independent) is computed by
    the oracle one by one and compared with the same rows of the GPU result, for every hc_apply mode that fits;
  * properties that hold at any size, evaluated on the full GPU vectors: Hermiticity <u|Hv> = <Hu|v>, the constant-
    interaction closed form V_ksql = U d_kq d_sl -> H2 = U N(N-1)/2 (every element), modes agree with each other;
  * integer structures: windows of the hashing table and Map1/Map2 against the oracle, bit-exact, and the GPU's own
    rank(unrank(b) - e_k + e_l) against its stored Map1 (cross-checks two independent kernels).
Tolerance (north_star): max_i |HC_gpu - HC_ref|_i <= 1e-12 * max(|T|_max, |V|_max) * ||C||_1.
"""
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


def _maps_fit(sp, mcb):
    need = sp.structure_bytes(mcb.MAP1) + sp.structure_bytes(mcb.MAP2)
    free, _ = torch.cuda.mem_get_info()
    return need < 0.5 * free and need < 16e9        # keep the test quick: configs 1 and 2 only


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_hc_apply_sampled_rows_all_modes(mcb, cfg):
    c, T, V, (C,) = workloads.make_inputs(cfg)
    sp = mcb.Space(c.N, c.M)
    assert sp.nc == c.nc
    sp.build_structure(mcb.FOCK_TABLE)
    rows = workloads.sample_rows(c.nc, 48, 1500, workloads.seed_for(cfg, 3))
    ref, _ = oracle.hc_apply(c.N, c.M, T, V, C, rows=rows)
    dC = torch.from_numpy(C).cuda()
    modes = [("GEMM", mcb.GEMM), ("REHASH", mcb.REHASH)]
    if 2 <= c.M <= 5:
        modes.append(("RUNS", mcb.RUNS))
    if _maps_fit(sp, mcb):
        sp.build_structure(mcb.MAP1)
        sp.build_structure(mcb.MAP2)
        modes.append(("MAPS", mcb.MAPS))
    t = tol(T, V, C)
    drows = torch.from_numpy(rows).cuda()
    results = {}
    for name, mode in modes:
        out = sp.hc_apply(T, V, dC, mode=mode)
        got = out[drows].cpu().numpy()
        err = np.abs(got - ref).max()
        assert err <= t, (name, err, t)
        results[name] = out
    # the modes are different algorithms over the same data: they must agree everywhere, not only on the sample
    base = results["GEMM"]
    for name, out in results.items():
        assert float((out - base).abs().max()) <= t, name
    sp.close()


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_hermiticity_and_constant_interaction_full_size(mcb, cfg):
    c, T, V, (u, v) = workloads.make_inputs(cfg, n_vectors=2)
    sp = mcb.Space(c.N, c.M)
    sp.build_structure(mcb.FOCK_TABLE)
    du, dv = torch.from_numpy(u).cuda(), torch.from_numpy(v).cuda()
    Hu = sp.hc_apply(T, V, du)
    Hv = sp.hc_apply(T, V, dv)
    lhs = torch.vdot(du, Hv).item()          # <u|Hv>
    rhs = torch.vdot(Hu, dv).item()          # <Hu|v>
    scale = max(np.abs(T).max(), np.abs(V).max()) * c.N * c.N
    assert abs(lhs - rhs) <= 1e-11 * scale, (lhs, rhs)
    # V_ksql = U delta_kq delta_sl, T = 0:  H = U/2 sum_ks a+_k a+_s a_k a_s = U N(N-1)/2  (closed form, all elements)
    M = c.M
    U = 0.37 - 0.11j
    Vc = np.zeros((M,) * 4, dtype=np.complex128)
    for k in range(M):
        for s in range(M):
            Vc[k, s, k, s] = U
    T0 = np.zeros((M, M), dtype=np.complex128)
    expect = U * c.N * (c.N - 1) / 2
    for mode in (mcb.GEMM, mcb.REHASH) + ((mcb.RUNS,) if 2 <= M <= 5 else ()):
        out = sp.hc_apply(T0, Vc, du, mode=mode)
        err = float((out - expect * du).abs().max())
        assert err <= 1e-12 * abs(U) * c.N * c.N * np.abs(u).max() * 4, (mode, err)
    # T = diag(eps), V = 0: every configuration is an eigenvector with eigenvalue sum_k n_k eps_k; check through
    # the GPU's own hashing table on a window
    eps = np.linspace(-1.0, 2.0, M)
    out = sp.hc_apply(np.diag(eps).astype(np.complex128), np.zeros((M,) * 4, dtype=np.complex128), du, mode=mcb.REHASH)
    b0 = c.nc // 3
    occ = oracle.unrank(c.N, c.M, np.arange(b0, b0 + 4096))
    lam = occ @ eps
    got = out[b0:b0 + 4096].cpu().numpy()
    assert np.abs(got - lam * u[b0:b0 + 4096]).max() <= 1e-12 * np.abs(lam).max() * np.abs(u).max() * 4
    sp.close()


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_structures_windows_full_size(mcb, cfg):
    c = workloads.CONFIGS[cfg]
    sp = mcb.Space(c.N, c.M)
    sp.build_structure(mcb.FOCK_TABLE)
    nc, nc2 = sp.nc, sp.nc2
    W = 512
    for b0 in (0, nc // 2 - 77, nc - W):
        assert (sp.fock_export(b0, W) == oracle.unrank(c.N, c.M, np.arange(b0, b0 + W))).all()
    for b0 in (0, nc2 // 3, nc2 - W):
        assert (sp.fock_export(b0, W, removed=2) == oracle.unrank(c.N - 2, c.M, np.arange(b0, b0 + W))).all()
    sp.build_structure(mcb.MAP1)
    for b0 in (0, nc // 2 - 77, nc - W):
        got = sp.map1_export(b0, W)
        assert (got == oracle.map1(c.N, c.M, b0, W)).all()
        # GPU-internal cross-check: rank(unrank(b) - e_k + e_l) from the hashing kernels == stored map entry
        occ = sp.unrank(torch.arange(b0, b0 + W, dtype=torch.int32, device="cuda"))
        for k, l in ((0, c.M - 1), (c.M - 1, 0), (1, 2)):
            moved = occ.clone()
            moved[:, k] -= 1
            moved[:, l] += 1
            idx = sp.rank(moved).cpu().numpy()           # rows with n_k = 0 become invalid -> -1
            assert (idx == got[:, k, l]).all()
    if _maps_fit(sp, mcb):
        sp.build_structure(mcb.MAP2)
        Wm = 64
        for b0 in (0, nc // 2 - 77, nc - Wm):
            assert (sp.map2_export(b0, Wm) == oracle.map2(c.N, c.M, b0, Wm)).all()
    sp.close()


def test_apply_host_matches_device_and_counts_launches(mcb):
    c, T, V, (C,) = workloads.make_inputs(1)
    sp = mcb.Space(c.N, c.M)
    sp.build_structure(mcb.FOCK_TABLE)
    dev = sp.hc_apply(T, V, torch.from_numpy(C).cuda()).cpu()
    host = sp.hc_apply_host(T, V, torch.from_numpy(C).pin_memory())
    assert torch.equal(dev, host)
    assert sp.last_apply_launches() in (1, 2, 3)
    sp.timing_enable(True)
    sp.hc_apply(T, V, torch.from_numpy(C).cuda())
    ms, la = sp.timing_read()
    assert len(la) == 1 and la[0] == sp.last_apply_launches() and (ms[0, :la[0]] > 0).all()
    sp.timing_enable(False)
    sp.close()


def test_error_paths(mcb):
    with pytest.raises(mcb.McbError):
        mcb.Space(0, 3)
    with pytest.raises(mcb.McbError):
        mcb.Space(3, 0)
    with pytest.raises(mcb.McbError):
        mcb.Space(60, 30)                       # nc overflows int32 -> MCB_ERANGE
    sp = mcb.Space(4, 3)
    C = torch.zeros(sp.nc, dtype=torch.complex128, device="cuda")
    T = np.zeros((3, 3), dtype=np.complex128)
    V = np.zeros((3,) * 4, dtype=np.complex128)
    with pytest.raises(mcb.McbError) as e:
        sp.hc_apply(T, V, C)                    # hashing table not built
    assert e.value.status == mcb.ENOTREADY
    sp.build_structure(mcb.FOCK_TABLE)
    with pytest.raises(mcb.McbError) as e:
        sp.hc_apply(T, V, C, mode=mcb.MAPS)     # maps not built
    assert e.value.status == mcb.ENOTREADY
    with pytest.raises(mcb.McbError) as e:
        sp.hc_apply(T, V, C, out=C)             # aliasing
    assert e.value.status == mcb.EINVAL
    big = mcb.Space(3, 14)
    big.build_structure(mcb.FOCK_TABLE)
    Cb = torch.zeros(big.nc, dtype=torch.complex128, device="cuda")
    with pytest.raises(mcb.McbError) as e:          # 12 < M <= 32: the generic path has no per-output (REHASH) variant
        big.hc_apply(np.zeros((14, 14), dtype=np.complex128), np.zeros((14,) * 4, dtype=np.complex128), Cb, mode=mcb.REHASH)
    assert e.value.status == mcb.EUNSUPPORTED
    out = big.hc_apply(np.zeros((14, 14), dtype=np.complex128), np.zeros((14,) * 4, dtype=np.complex128), Cb)
    assert float(out.abs().max()) == 0.0
    sp.close()
    big.close()


def test_error_paths_rho_and_lanczos(mcb):
    sp = mcb.Space(4, 3)
    C = torch.ones(sp.nc, dtype=torch.complex128, device="cuda")
    T = np.zeros((3, 3), dtype=np.complex128)
    V = np.zeros((3,) * 4, dtype=np.complex128)
    with pytest.raises(mcb.McbError) as e:
        sp.rho(C)                               # hashing table not built
    assert e.value.status == mcb.ENOTREADY
    with pytest.raises(mcb.McbError) as e:
        sp.lanczos(T, V, C, 4)                  # the apply inside needs the table
    assert e.value.status == mcb.ENOTREADY
    sp.build_structure(mcb.FOCK_TABLE)
    with pytest.raises(mcb.McbError) as e:
        sp.lanczos(T, V, C, -1)                 # kmax < 0 (0 asks for the paper's cap nc / 8)
    assert e.value.status == mcb.EINVAL
    assert sp.lanczos_steps(0) == max(1, sp.nc // 8) and sp.lanczos_steps(7) == 7
    with pytest.raises(mcb.McbError) as e:
        sp.lanczos(T, V, torch.zeros_like(C), 3)        # zero start vector
    assert e.value.status == mcb.EINVAL
    a, b = sp.lanczos(T, V, C, 5)               # H = 0: invariant subspace after one step
    assert len(a) == 1 and a[0] == 0.0 and b[0] == 0.0
    big = mcb.Space(3, 14)                      # many orbitals: the generic path serves AUTO / GEMM, and SPARSE has a run-time-M kernel
    big.build_structure(mcb.FOCK_TABLE)
    Tb, Vb = np.zeros((14, 14), dtype=np.complex128), np.zeros((14,) * 4, dtype=np.complex128)
    Cb = torch.ones(big.nc, dtype=torch.complex128, device="cuda")
    for mode in (mcb.REHASH, mcb.MAPS, mcb.RUNS):
        with pytest.raises(mcb.McbError) as e:
            big.hc_apply(Tb, Vb, Cb, mode=mode)
        assert e.value.status == mcb.EUNSUPPORTED
    assert big.resolve_mode(Tb, Vb) == mcb.SPARSE                       # H = 0 has no off-diagonal element at all
    assert float(big.hc_apply(Tb, Vb, Cb, mode=mcb.SPARSE).abs().max()) == 0.0
    Vd = np.ones((14,) * 4, dtype=np.complex128)                        # a full V: the dense generic path
    assert big.resolve_mode(Tb, Vd) == mcb.GEMM
    with pytest.raises(mcb.McbError) as e:
        big.hc_apply(Tb, Vd, Cb, mode=mcb.SPARSE)                       # 105 * 104 off-diagonal elements > 1024
    assert e.value.status == mcb.EUNSUPPORTED
    sp.close()
    big.close()


def _poison_scratch(sp):
    """The binding's cached device scratch of C still holds the previous call's vector: fill it (and the workspace, whose
    class planes and flags an identical previous apply left behind) with NaN bytes so that a kernel that gathered C before
    it arrived, or summed planes before they were written, cannot pass by reading stale but correct data."""
    for name in ("dC", "dHC", "ws"):
        t = sp._workspace.get(name)
        if t is not None:
            t.view(torch.uint8).fill_(0xFF)
    torch.cuda.synchronize()


def test_apply_host_pipelined_runs_path(mcb):
    # configs[2] resolves to MCB_RUNS: with pinned vectors mcb_hc_apply_host overlaps H2D, the kernel (which waits per segment
    # for the prefix of C it needs) and the zero-copy write-back of HC; unpinned vectors take the plain copy-apply-copy path
    c, T, V, (C, C2) = workloads.make_inputs(2, n_vectors=2)
    sp = mcb.Space(c.N, c.M)
    sp.build_structure(mcb.FOCK_TABLE)
    assert sp.resolve_mode(T, V) == mcb.RUNS
    dev = sp.hc_apply(T, V, torch.from_numpy(C).cuda()).cpu()
    dev2 = sp.hc_apply(T, V, torch.from_numpy(C2).cuda()).cpu()
    hC, hC2 = torch.from_numpy(C).pin_memory(), torch.from_numpy(C2).pin_memory()
    out = torch.empty_like(hC).pin_memory()
    for i in range(4):                                   # repeated calls reuse the scratch vectors, streams and flags
        out.zero_()
        _poison_scratch(sp)                              # stale-but-identical scratch must not be able to hide a premature gather
        src, want = (hC, dev) if i % 2 == 0 else (hC2, dev2)     # and a DIFFERENT vector goes through the same space
        host = sp.hc_apply_host(T, V, src, out_host=out)
        assert torch.equal(want, host)
    plain = sp.hc_apply_host(T, V, torch.from_numpy(C))  # pageable memory
    assert torch.equal(dev, plain)
    sp.close()


@pytest.mark.parametrize("N,M", [(2200, 2), (1500, 3), (64, 5), (7, 4)])
def test_apply_host_pipelined_other_shapes(mcb, N, M):
    # the prefix of C a segment needs (nc - N_c(N - j - 3, M) for top occupation j) for the other orbital counts MCB_RUNS
    # serves (mode given explicitly: MCB_AUTO takes MCB_RUNS only from 2^20 configurations on), many segments and a tiny space
    sp = mcb.Space(N, M)
    T, V, C = workloads.make_small_inputs(N, M, sp.nc, seed=77 + N + M)
    sp.build_structure(mcb.FOCK_TABLE)
    assert sp.resolve_mode(T, V, mcb.RUNS) == mcb.RUNS
    dev = sp.hc_apply(T, V, torch.from_numpy(C).cuda(), mode=mcb.RUNS).cpu()
    rows = workloads.sample_rows(sp.nc, 16, min(200, sp.nc), 5)
    ref, _ = oracle.hc_apply(N, M, T, V, C, rows=rows)
    t = max(tol(T, V, C), 64 * 2.0 ** -53 * np.abs(ref).max()) if N > 1000 else tol(T, V, C)
    assert np.abs(dev.numpy()[rows] - ref).max() <= t
    hC = torch.from_numpy(C).pin_memory()
    out = torch.empty_like(hC).pin_memory()
    for _ in range(2):
        out.zero_()
        _poison_scratch(sp)
        assert torch.equal(dev, sp.hc_apply_host(T, V, hC, out_host=out, mode=mcb.RUNS))
    sp.close()
