"""CPU-only checks of the host-side logic: the C ABI library exports every symbol include/mcb.h declares (no compute
calls without a GPU), the Python binding names them all, the product path fails loudly without CUDA, and bench.py's
multi-process plumbing (N independent replicas: barrier + max-over-ranks, world_size 2 on gloo)."""
import ctypes
import json
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "mcb.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mcb_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported_and_bound():
    import paper_2005_13679_b200 as mcb
    from paper_2005_13679_b200 import build
    build.build()
    names = _declared_functions()
    assert len(names) >= 20
    L = ctypes.CDLL(mcb.LIB_PATH)
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/mcb.h but not exported by libmcb.so"
    assert sorted(mcb.EXPORTS) == names
    # pure host entry points that need no device
    L.mcb_strerror.restype = ctypes.c_char_p
    assert L.mcb_strerror(0) == b"ok" and b"invalid" in L.mcb_strerror(-1)
    L.mcb_nc.restype = ctypes.c_longlong
    assert L.mcb_nc(None) == -1
    assert L.mcb_structure_bytes(None, 0) == -1


def test_tridiag_eigvals_host_solver():
    """mcb_tridiag_eigvals is host-only (the paper's LAPACK step): Sturm bisection against LAPACK's answer
    (numpy eigvalsh of the dense tridiagonal matrix), closed forms, and degenerate inputs."""
    import numpy as np
    import paper_2005_13679_b200 as mcb
    from paper_2005_13679_b200 import build
    build.build()
    rng = np.random.default_rng(7)
    for n in (1, 2, 3, 17, 200):
        a = rng.standard_normal(n) * 10.0
        b = np.abs(rng.standard_normal(max(n - 1, 0)))
        Tm = np.diag(a) + np.diag(b, 1) + np.diag(b, -1)
        ref = np.linalg.eigvalsh(Tm)
        got = mcb.tridiag_eigvals(a, b)
        assert got.shape == (n,) and (np.diff(got) >= 0).all()
        assert np.abs(got - ref).max() <= 1e-13 * max(1.0, np.abs(ref).max()), n
    # free chain: alpha = 0, beta = 1 -> 2 cos(k pi / (n + 1)); a zero off-diagonal splits the matrix; repeated eigenvalues
    n = 64
    got = mcb.tridiag_eigvals(np.zeros(n), np.ones(n - 1))
    assert np.abs(got - np.sort(2 * np.cos(np.arange(1, n + 1) * np.pi / (n + 1)))).max() < 1e-13
    assert np.allclose(mcb.tridiag_eigvals([3.0, 1.0, 2.0], [0.0, 0.0]), [1.0, 2.0, 3.0], rtol=0, atol=1e-15)
    assert np.allclose(mcb.tridiag_eigvals([5.0, 5.0, 5.0, 5.0], [0.0, 0.0, 0.0]), 5.0, rtol=0, atol=1e-14)
    tiny = mcb.tridiag_eigvals([0.0, 0.0], [1e-200])             # a coupling whose square underflows: finite, ordered, and
    assert np.isfinite(tiny).all() and tiny[0] <= tiny[1] and np.abs(tiny - [-1e-200, 1e-200]).max() <= 2e-200   # off by no more than the coupling
    with pytest.raises(mcb.McbError):
        mcb.lib().mcb_tridiag_eigvals.restype = ctypes.c_int
        mcb._check(mcb.lib().mcb_tridiag_eigvals(0, None, None, None), "mcb_tridiag_eigvals")


def test_product_path_fails_loudly_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    import paper_2005_13679_b200 as mcb
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        mcb.Space(3, 3)


def test_package_does_not_import_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2005_13679_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "mcb_oracle" not in txt and "mcbo_" not in txt, f
    otxt = open(os.path.join(ROOT, "oracle", "mcb_oracle.c")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "mcb.h" not in otxt and "import paper_2005_13679_b200" not in otxt and "libmcb.so" not in otxt


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch, bench
rank = int(os.environ["RANK"])
job = bench.Job(2, "gloo", torch.device("cpu"))
job.barrier()
ms = 2.0 if rank == 0 else 5.0            # the slower rank sets the job time
assert job.max_over_ranks(ms) == 5.0
v = job.whole_job_value(1000.0, ms)       # 2 replicas x 1000 units / 5 ms
assert abs(v - 2 * 1000.0 / 5e-3) < 1e-6, v
job.barrier()
job.close()
print("rank", rank, "ok")
"""


def test_replica_plumbing_world_size_2_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    port = 29500 + (os.getpid() % 2000)
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
    for r, p in enumerate(procs):
        out, _ = p.communicate(timeout=180)
        assert p.returncode == 0 and f"rank {r} ok" in out, out


def test_reference_arm_rank_gating_and_json_contract():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--cfg", "0", "--steps", "1", "--warmup", "3"],
                         env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0 and out.stdout.strip() == ""          # other ranks exit 0 without work
    env = dict(os.environ, RANK="0", WORLD_SIZE="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--cfg", "0", "--steps", "1", "--warmup", "3"],
                         env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert key in line, key
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["value"] == line["value"]
    assert "workload" in line["config"]


def test_term_counts_match_brute_force_enumeration():
    # bench.py's algorithmic term counts (roofline numerators) against explicit enumeration on a tiny space
    import bench
    from oracle import brute
    N, M = 5, 4
    confs = brute.enumerate_configs(N, M)
    nc = len(confs)
    nc1 = len(brute.enumerate_configs(N - 1, M))
    nc2 = len(brute.enumerate_configs(N - 2, M))
    tc = bench.term_counts(N, M, nc, nc1, nc2)
    one = sum(M for n in confs for k in range(M) if n[k] >= 1)
    pairs = sum(1 for n in confs for k in range(M) for s in range(k, M) if (n[k] >= 2 if k == s else (n[k] >= 1 and n[s] >= 1)))
    P = M * (M + 1) // 2
    assert tc["one_body_terms"] == one and tc["two_body_terms_packed"] == pairs * P and tc["P"] == P
