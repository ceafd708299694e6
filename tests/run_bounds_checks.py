#!/usr/bin/env python
"""Bounds-checked sweep of the CUDA path (stands in for compute-sanitizer memcheck, which is closed on this GPU pool).

    python tests/run_bounds_checks.py          # on a GPU box; rebuilds libmcb.so twice (debug, then release)

Builds libmcb.so with -DMCB_DEBUG_BOUNDS (every gather / scatter index of the apply, map and density kernels is checked on
the device, csrc/mcb_internal.cuh MCB_CHK), runs every hc_apply mode, the map builders, rho and Lanczos on small and
medium spaces with NaN-poisoned workspaces, compares with the CPU oracle, and requires that no space recorded a violation.
Poisoning plays the part of initcheck (a read of never-written workspace shows up as NaN in the result); bit-identical
repeats on a second stream play the part of racecheck for the flag-synchronised persistent kernel.
"""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def build(extra):
    env = dict(os.environ, MCB_NVCC_EXTRA=extra)
    subprocess.run([sys.executable, "-m", "paper_2005_13679_b200.build", "--force"], check=True, env=env, cwd=ROOT)


def sweep():
    import numpy as np
    import torch

    import oracle
    import paper_2005_13679_b200 as mcb
    import workloads

    oracle.build()
    spaces = [(10, 5), (2, 2), (3, 3), (6, 4), (33, 4), (17, 5), (200, 3), (2000, 2), (60, 4), (5, 7), (4, 12), (5, 10), (3, 13), (5, 14), (2, 20)]
    checked = 0
    for N, M in spaces:
        sp = mcb.Space(N, M)
        nc = sp.nc
        T, V, C = workloads.make_small_inputs(N, M, nc, seed=31 * N + M)
        ref, _ = oracle.hc_apply(N, M, T, V, C)
        t = 1e-12 * max(np.abs(T).max(), np.abs(V).max()) * np.abs(C).sum()
        if N > 1000:
            t = max(t, 64 * 2.0 ** -53 * float(np.abs(ref).max()))
        sp.build_structure(mcb.FOCK_TABLE)
        dC = torch.from_numpy(C).cuda()
        modes = [mcb.AUTO, mcb.GEMM]
        if M <= 12:
            modes += [mcb.REHASH] + ([mcb.SPARSE] if sp.P * sp.P <= 1024 else [])    # SPARSE: at most 1024 off-diagonal elements
            if 2 <= M <= 5:
                modes.append(mcb.RUNS)
            if M <= 8:
                sp.build_structure(mcb.MAP1); sp.build_structure(mcb.MAP2)
                modes.append(mcb.MAPS)
        for mode in modes:
            for rep in range(2):
                w = sp._workspace.get("ws")
                if w is not None:
                    w.fill_(0xFF)                                   # poison: stale planes / flags cannot help
                out = sp.hc_apply(T, V, dC, mode=mode)
                err = float(np.abs(out.cpu().numpy() - ref).max())
                assert err <= t, (N, M, mode, err, t)
        if M <= 12:
            sp.drop_structure(mcb.MAP1) if M <= 8 else None
            sp.drop_structure(mcb.MAP2) if M <= 8 else None
            sp.build_structure(mcb.MAP2C)
            out = sp.hc_apply(T, V, dC, mode=mcb.MAPS)
            assert float(np.abs(out.cpu().numpy() - ref).max()) <= t
            hC = torch.from_numpy(C).pin_memory()
            if 2 <= M <= 5:
                assert float(np.abs(sp.hc_apply_host(T, V, hC, mode=mcb.RUNS).numpy() - ref).max()) <= t
        if M > 12:                                                   # run-time-M MCB_SPARSE kernel: a Bose-Hubbard ring on M sites
            Tb, Vb, _ = workloads.make_small_inputs(N, M, nc, seed=31 * N + M, kind="bh")
            refb, _ = oracle.hc_apply(N, M, Tb, Vb, C)
            tb = 1e-12 * max(np.abs(Tb).max(), np.abs(Vb).max()) * np.abs(C).sum()
            for rep in range(2):
                assert float(np.abs(sp.hc_apply(Tb, Vb, dC, mode=mcb.SPARSE).cpu().numpy() - refb).max()) <= tb
        r1, r2 = sp.rho(dC)
        if M <= mcb.RHO_STATIC_MAX_M:                                # the allocation-free variant: same kernels, fixed scratch
            s1, s2 = sp.rho_static(dC)
            assert float((s1 - r1).abs().max()) <= 1e-12 * N * max(N - 1, 1) and float((s2 - r2).abs().max()) <= 1e-12 * N * max(N - 1, 1)
        sp.lanczos(T, V, dC, min(5, nc))
        compiled, site, idx = sp.debug_bounds()
        assert compiled, "libmcb.so was not built with -DMCB_DEBUG_BOUNDS"
        assert site == 0, f"out-of-range index {idx} at site {site} on space N={N}, M={M}"
        checked += 1
        sp.close()
    print(f"bounds checks: {checked} spaces, every hc_apply mode, maps, rho, lanczos: no out-of-range index; results within tolerance with poisoned workspaces")


if __name__ == "__main__":
    if "--sweep-only" in sys.argv:
        sweep()
        sys.exit(0)
    build("-DMCB_DEBUG_BOUNDS")
    try:
        subprocess.run([sys.executable, os.path.abspath(__file__), "--sweep-only"], check=True, cwd=ROOT)
    finally:
        build("")
