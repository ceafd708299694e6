#!/usr/bin/env python
"""bench.py -- H.C throughput of libmcb on B200, with the oracle timed beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--cfg 0..4] [--mode auto|gemm|rehash|maps] [--impl reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

A "step" is one pass of the whole hot path's steady state over one coefficient vector: one
`hc_apply(T, V, C) -> HC` (Eq. 12) through the C ABI (include/mcb.h), with the hashing table
(and the jump maps in MAPS mode) already built on the device -- they are built once per space
(PAPER.md:178-224); their build times are reported under "setup".  T and V are packed and uploaded inside
every step (they change every step in the paper's motivating use).

Headline workload = BASELINE.json configs[2] (N=400, M=4: the largest nc, which is what `metric` is quoted
on).  `value` = configurations/s = nc * applications/s, whole job (all ranks; the path does not shard by
north_star, so N>1 runs N independent replicas = weak scaling, no data-path collective).

Cold-cache rule: inputs are larger than L2 -- the step rotates through R distinct C vectors and R distinct HC
buffers whose total size (>= 3 * 2 * 16 * nc bytes) exceeds the 126 MB L2 several times over.

One JSON line is printed by rank 0.  `--impl reference` times the CPU oracle (oracle/, as it stands) on the
host cores on a bounded row sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "hc_apply_configurations_per_s"
UNIT = "configs/s"
FP64_FMA_PER_CLK_PER_SM = 64          # B200 SM = 4 sub-partitions x 16 FP64 lanes
N_SM = 148


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


def fp64_peak_tflops(sm_mhz: float) -> float:
    """Plain FP64 ALU peak: 148 SMs x 64 DFMA/clk x 2 flop x clock."""
    return N_SM * FP64_FMA_PER_CLK_PER_SM * 2 * sm_mhz * 1e6 / 1e12


def term_counts(N: int, M: int, nc: int, nc1: int, nc2: int):
    """Algorithmic term counts per apply: one-body M^2*nc1, two-body (packed) P^2*nc2."""
    P = M * (M + 1) // 2
    return {"one_body_terms": M * M * nc1, "two_body_terms_packed": P * P * nc2, "P": P}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md clocks line)."""

    def __init__(self, index: int, period_s: float = 0.005):
        self.index, self.period = index, period_s
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._thr = None
        self._nv = None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nv = None
        self._thr = threading.Thread(target=self._run, daemon=True)
        self._thr.start()

    def _run(self):
        nv = self._nv
        names = {}
        if nv is not None:
            for nm, key in (("nvmlClocksThrottleReasonHwSlowdown", "hw_slowdown"),
                            ("nvmlClocksThrottleReasonHwThermalSlowdown", "hw_thermal_slowdown"),
                            ("nvmlClocksThrottleReasonSwThermalSlowdown", "sw_thermal_slowdown"),
                            ("nvmlClocksThrottleReasonSwPowerCap", "sw_power_cap"),
                            ("nvmlClocksThrottleReasonHwPowerBrakeSlowdown", "hw_power_brake_slowdown")):
                if hasattr(nv, nm):
                    names[getattr(nv, nm)] = key
        while not self._stop.is_set():
            try:
                if nv is not None:
                    self.samples.append(float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
                    for bit, key in names.items():
                        if r & bit:
                            self.reasons.add(key)
                else:
                    import subprocess
                    out = subprocess.run(
                        ["nvidia-smi", "-i", str(self.index),
                         "--query-gpu=clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
                         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
                         "clocks_event_reasons.sw_power_cap", "--format=csv,noheader,nounits"],
                        capture_output=True, text=True, timeout=5).stdout.strip().split(",")
                    self.samples.append(float(out[0]))
                    self.max_mhz = float(out[1])
                    for v, key in zip(out[2:], ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")):
                        if v.strip().lower() == "active":
                            self.reasons.add(key)
            except Exception:
                pass
            self._stop.wait(self.period)

    def stop(self):
        self._stop.set()
        if self._thr is not None:
            self._thr.join(timeout=5)
        s = sorted(self.samples)
        med = s[len(s) // 2] if s else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(s)}


# ------------------------------------------------------------------------------------------------------------
# CPU oracle legs
# ------------------------------------------------------------------------------------------------------------
def oracle_sample_rate(c, T, V, C, target_s: float, nthreads: int = 0):
    """Time oracle.hc_apply on a bounded seeded row sample; returns (configs/s, threads, rows, seconds)."""
    import oracle
    probe = workloads.sample_rows(c.nc, 64, 1024, workloads.seed_for(c.cfg, 11))
    t0 = time.perf_counter()
    _, used = oracle.hc_apply(c.N, c.M, T, V, C, rows=probe, nthreads=nthreads)
    dt = max(time.perf_counter() - t0, 1e-6)
    rate = probe.size / dt
    nrows = int(min(c.nc, max(probe.size, rate * target_s)))
    if nrows >= c.nc:
        rows = None
        nrows = c.nc
    else:
        rows = workloads.sample_rows(c.nc, 1024, nrows, workloads.seed_for(c.cfg, 12))
        nrows = rows.size
    t0 = time.perf_counter()
    _, used = oracle.hc_apply(c.N, c.M, T, V, C, rows=rows, nthreads=nthreads)
    dt = time.perf_counter() - t0
    return nrows / dt, used, nrows, dt


def run_reference(args):
    """--impl reference: the oracle as it stands, on the host cores; rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    oracle.build()
    c, T, V, (C,) = workloads.make_inputs(args.cfg)
    per_step_s = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    rates, rows_used, used = [], 0, 1
    for i in range(args.warmup + args.steps):
        r, used, nrows, dt = oracle_sample_rate(c, T, V, C, per_step_s)
        if i >= args.warmup:
            rates.append((nrows, dt))
            rows_used = nrows
    tot_rows = sum(n for n, _ in rates)
    tot_s = sum(d for _, d in rates)
    value = tot_rows / tot_s
    sample = f"{rows_used} seeded rows of {c.nc} per step (rows of H.C are independent), all host threads"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * c.nc / value,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "complex128 (f64)",
        "data": "synthetic (seeded, workloads.py)",
        "config": config_dict(c, "oracle O6: ordered M^4 sums, literal Algorithm 1 per term"),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "note": "ms_per_step is the full-vector time extrapolated from the row sample",
    }
    print(json.dumps(line))
    return 0


def config_dict(c, variant: str):
    return {"workload": f"BASELINE.json configs[{c.cfg}] {c.name}: N={c.N} bosons, M={c.M} orbitals, nc={c.nc}, "
                        f"{'Lieb-Liniger T,V (g=10, L=1)' if c.kind == 'll' else 'dense random Hermitian T, symmetric random V'}, "
                        "random L2-normalised complex128 C",
            "N": c.N, "M": c.M, "nc": c.nc, "variant": variant}


# ------------------------------------------------------------------------------------------------------------
# multi-process plumbing: N independent replicas (the path does not shard); the only
# cross-rank operations are the barrier around the timed region and the max of the per-rank device times.
# ------------------------------------------------------------------------------------------------------------
class Job:
    def __init__(self, world: int, backend: str, device):
        self.world, self.device, self.dist = world, device, None
        if world > 1:
            import torch.distributed as dist
            kw = {"device_id": device} if backend == "nccl" else {}
            dist.init_process_group(backend, **kw)
            self.dist = dist

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()

    def max_over_ranks(self, x: float) -> float:
        if self.dist is None:
            return x
        import torch
        t = torch.tensor([x], dtype=torch.float64, device=self.device)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def whole_job_value(self, units_per_rank: float, ms_per_step_this_rank: float) -> float:
        """units all ranks processed / max-over-ranks time (weak scaling, replicas)."""
        ms = self.max_over_ranks(ms_per_step_this_rank)
        return self.world * units_per_rank / (ms * 1e-3)

    def close(self):
        if self.dist is not None:
            self.dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------------------
# GPU arm
# ------------------------------------------------------------------------------------------------------------
MODES = {"auto": 0, "maps": 1, "rehash": 2, "gemm": 3, "runs": 4, "sparse": 5}
MODE_NAMES = {1: "MAPS", 2: "REHASH", 3: "GEMM", 4: "RUNS", 5: "SPARSE"}
KERNELS = {1: ["k_hc_direct<M,maps>"], 2: ["k_hc_direct<M,rehash>"], 3: ["k_hc2_contract<M>", "k_hc2_reduce<M>"],
           4: ["k_hc2_runs<M>"], 5: ["k_hc_sparse<M>"]}


# dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel, per launch, from the committed `ncu --set full`
# captures (profiles/*.md name the commands); None where no capture of the current kernel exists.
NCU_TRAFFIC_BYTES = {
    (2, 4): (1.437949e9 + 1.193993e9, "profiles/r2_cfg2_runs_head.md"),
    (1, 5): (0.119572e9 + 0.048353e9, "profiles/r3_cfg1_sparse.md"),
    (4, 3): (0.452885e9 + 3.056407e9, "profiles/r2_gemm_final.md"),
    (3, 3): (0.612919e9 + 4.066090e9, "profiles/r2_gemm_final.md"),
    (2, 1): (5.121572e9 + 0.172730e9, "profiles/r2_cfg2_maps_final.md"),
}


def time_mode(sp, mcb, torch, T, V, dCs, dHCs, mode, steps, warmup, barrier):
    """Device time of `steps` applies (CUDA events on the launching stream), plus per-kernel times."""
    R = len(dCs)
    for i in range(warmup):
        sp.hc_apply(T, V, dCs[i % R], out=dHCs[i % R], mode=mode)
    torch.cuda.synchronize()
    barrier()
    sp.timing_enable(True)
    # one event per step boundary on the launching stream: the total is first-to-last, the per-step gaps give median and best
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    evs[0].record()
    for i in range(steps):
        sp.hc_apply(T, V, dCs[i % R], out=dHCs[i % R], mode=mode)
        evs[i + 1].record()
    torch.cuda.synchronize()
    barrier()
    ms_total = evs[0].elapsed_time(evs[steps])
    time_mode.per_step_ms = [evs[i].elapsed_time(evs[i + 1]) for i in range(steps)]
    kms, la = sp.timing_read(min(steps, 512))
    sp.timing_enable(False)
    launches = int(sp.last_apply_launches())
    return ms_total, kms, launches


def spread(ms_list):
    """median / best / worst of per-step device times (ms)."""
    s = sorted(ms_list)
    return {"median_ms": s[len(s) // 2], "best_ms": s[0], "worst_ms": s[-1], "n": len(s)} if s else None


def other_config(cfg, mcb, torch, peaks, fp64_measured, barrier, steps):
    """A short, driver-timed line for another BASELINE.json config: device-resident H.C (MCB_AUTO), its kernels, the roofline
    fraction of the dominant one, and the host-buffer e2e -- so that BASELINE.md's numbers for it are not the builder's alone."""
    R = 3
    c, T, V, Cs = workloads.make_inputs(cfg, n_vectors=R)
    sp = mcb.Space(c.N, c.M)
    try:
        sp.build_structure(mcb.FOCK_TABLE)
        mode = sp.resolve_mode(T, V, mcb.AUTO)
        nc, nc1, nc2 = sp.nc, sp.nc_removed(1), sp.nc_removed(2)
        tc = term_counts(c.N, c.M, nc, nc1, nc2)
        dCs = [torch.from_numpy(C).cuda() for C in Cs]
        dHCs = [torch.empty_like(d) for d in dCs]
        ms_total, kms, launches = time_mode(sp, mcb, torch, T, V, dCs, dHCs, mode, steps, 3, barrier)
        per = spread(time_mode.per_step_ms)
        kavg = kms.mean(axis=0) if len(kms) else np.zeros(3)
        dom = int(np.argmax(kavg)); dom_ms = float(kavg[dom])
        out = {"workload": f"BASELINE.json configs[{cfg}] N={c.N} M={c.M} nc={nc}", "mode": MODE_NAMES[mode], "steps": steps,
               "ms_per_step": ms_total / steps, "ms_per_step_median": per["median_ms"], "ms_per_step_best": per["best_ms"],
               "configs_per_s": nc / (ms_total / steps * 1e-3), "gpu_launches_per_step": launches,
               "kernel_ms": {KERNELS[mode][i]: float(kavg[i]) for i in range(len(KERNELS[mode]))}}
        if mode == mcb.SPARSE:
            alg = 32.0 * nc + 2.0 * c.M * nc
            out["roofline"] = {"bound": "hbm", "kernel": KERNELS[mode][dom], "achieved": alg / (dom_ms * 1e-3) / 1e9, "peak": peaks["hbm_gbs"],
                               "unit": "GB/s", "frac": alg / (dom_ms * 1e-3) / 1e9 / peaks["hbm_gbs"], "algorithmic_bytes_per_launch": alg}
        else:
            kflops = 8.0 * tc["two_body_terms_packed"] if mode in (mcb.GEMM, mcb.RUNS) else 8.0 * (tc["one_body_terms"] + tc["two_body_terms_packed"])
            pk = fp64_measured["dmma_tflops" if mode in (mcb.GEMM, mcb.RUNS) else "dfma_tflops"]
            out["roofline"] = {"bound": "alu", "kernel": KERNELS[mode][dom], "achieved": kflops / (dom_ms * 1e-3) / 1e12, "peak": pk,
                               "unit": "TFLOP/s", "frac": kflops / (dom_ms * 1e-3) / 1e12 / pk, "algorithmic_flops_per_launch": kflops,
                               "step_frac": 8.0 * (tc["one_body_terms"] + tc["two_body_terms_packed"]) / (ms_total / steps * 1e-3) / 1e12 / pk}
        hC = [torch.from_numpy(C).pin_memory() for C in Cs]
        hHC = [torch.empty_like(h).pin_memory() for h in hC]
        for i in range(2):
            sp.hc_apply_host(T, V, hC[i % R], out_host=hHC[i % R], mode=mode)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n_e2e = 4
        a.record()
        for i in range(n_e2e):
            sp.hc_apply_host(T, V, hC[i % R], out_host=hHC[i % R], mode=mode)
        b.record(); torch.cuda.synchronize()
        out["e2e"] = {"ms_per_step": a.elapsed_time(b) / n_e2e, "value": nc / (a.elapsed_time(b) / n_e2e * 1e-3), "unit": UNIT,
                      "h2d_bytes_per_step": 16 * nc + 16 * (c.M ** 2 + c.M ** 4), "d2h_bytes_per_step": 16 * nc}
        return out
    finally:
        sp.close()
        torch.cuda.empty_cache()


def run_gpu(args):
    import torch
    import paper_2005_13679_b200 as mcb

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libmcb has no CPU path")
    mcb.lib()
    torch.cuda.set_device(local)
    job = Job(world, "nccl", torch.device("cuda", local))
    barrier, max_over_ranks = job.barrier, job.max_over_ranks

    peaks = load_peaks()
    # FP64 throughput this GPU sustains, measured with register-only kernels (mcb_fp64_peak): plain DFMA chains, DMMA m8n8k4
    # chains, both interleaved -- the ALU roofline is quoted against the MEASURED figure of the pipe the mode uses
    fp64_measured = {"dfma_tflops": mcb.fp64_peak(0), "dmma_tflops": mcb.fp64_peak(1), "both_tflops": mcb.fp64_peak(2)}
    R = 3
    c, T, V, Cs = workloads.make_inputs(args.cfg, n_vectors=R)
    sp = mcb.Space(c.N, c.M)
    assert sp.nc == c.nc
    nc, nc1, nc2 = sp.nc, sp.nc_removed(1), sp.nc_removed(2)
    tc = term_counts(c.N, c.M, nc, nc1, nc2)

    # ---- setup (once per space): hashing table, and the maps if the mode needs them.  Every builder of the path (Algorithm
    #      1 / 2 over all nc configurations, hashing table, single- and double-jump map) is timed here,
    #      as GB/s of the bytes it must move against the measured HBM copy bandwidth: they are HBM-write bound by design ----
    setup = {"peak_GBps": peaks["hbm_gbs"]}
    def timed(fn, reps):
        for _ in range(3):                               # (three: rotating outputs are allocated by the first three calls)
            fn()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            fn()
        b.record(); torch.cuda.synchronize()
        return a.elapsed_time(b) / reps
    def record(name, ms, nbytes):
        setup[name] = {"ms": ms, "bytes": nbytes, "GBps": nbytes / (ms * 1e-3) / 1e9, "hbm_frac": nbytes / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"]}
    # builders write into ROTATING outputs (3 buffers, together larger than the 126 MB L2 for the big structures): rebuilding
    # into one buffer lets L2 absorb part of the writes and the "HBM" rate is then partly an L2 rate
    fbufs = [sp.build_structure(mcb.FOCK_TABLE) for _ in range(3)]
    fstate = {"i": 0}
    def build_fock():
        fstate["i"] += 1
        sp.build_structure(mcb.FOCK_TABLE, buf=fbufs[fstate["i"] % 3])
    record("fock_table", timed(build_fock, 6), sp.structure_bytes(mcb.FOCK_TABLE))
    fbuf = fbufs[0]
    sp.build_structure(mcb.FOCK_TABLE, buf=fbuf)         # the table the applies use
    del fbufs
    setup["builder_outputs"] = "3 rotating output buffers per builder"
    mode = sp.resolve_mode(T, V, MODES[args.mode])       # what MCB_AUTO resolves to for these matrix elements
    if rank == 0 and not args.no_setup_rates:
        from collections import deque
        idx_all = torch.arange(nc, dtype=torch.int32, device="cuda")
        alive = deque(maxlen=2)                          # the two latest outputs stay alive: each call writes a third block
        record("unrank_all", timed(lambda: alive.append(sp.unrank(idx_all)), 6), 4 * (c.M + 1) * nc)
        alive.clear()
        occ_all = sp.unrank(idx_all)
        record("rank_all", timed(lambda: alive.append(sp.rank(occ_all)), 6), 4 * (c.M + 1) * nc)
        alive.clear()
        del occ_all, idx_all
        free, _ = torch.cuda.mem_get_info()
        for which, name in ((mcb.MAP1, "map1"), (mcb.MAP2, "map2")) + (((mcb.MAP2C, "map2_compact"),) if hasattr(mcb, "MAP2C") and c.N >= 2 else ()):
            need = sp.structure_bytes(which)
            if need < 0.6 * free and need < 80e9:
                mbuf = sp.build_structure(which)
                record(name, timed(lambda: sp.build_structure(which, buf=mbuf), 3), need + 2 * c.M * nc)     # + the hashing table it reads
                del mbuf
                sp.drop_structure(which)
                torch.cuda.empty_cache()
            else:
                setup[name] = {"skipped": f"needs {need / 1e9:.1f} GB (PAPER.md:264: memory is the limit)"}
    map_bytes = 0
    maps_layout = None
    if mode == mcb.MAPS:
        # dense planes (the faster layout on this part) when they fit, else the paper's compact double-jump table (T inside V)
        free, _ = torch.cuda.mem_get_info()
        dense_fits = sp.structure_bytes(mcb.MAP1) + sp.structure_bytes(mcb.MAP2) < 0.8 * free
        if c.N >= 2 and (args.compact_maps or not dense_fits):
            sp.build_structure(mcb.MAP2C)
            map_bytes = 4 * tc["P"] ** 2 * nc2 + 8 * nc                   # every stride entry + the line offsets
            maps_layout = "compact (MCB_MAP2C, PAPER.md:212-224)"
        else:
            sp.build_structure(mcb.MAP1)
            sp.build_structure(mcb.MAP2)
            map_bytes = 4 * nc * (c.M * c.M - c.M) + 4 * nc * tc["P"] ** 2   # entries the kernel may read (upper bound)
            maps_layout = "dense planes (MCB_MAP1 + MCB_MAP2)"

    dCs = [torch.from_numpy(C).cuda() for C in Cs]
    dHCs = [torch.empty_like(d) for d in dCs]

    # ---- device-resident timing ----
    clocks = ClockSampler(local)
    clocks.start()
    ms_total, kms, launches = time_mode(sp, mcb, torch, T, V, dCs, dHCs, mode, args.steps, args.warmup, barrier)
    clk = clocks.stop()
    step_spread = spread(time_mode.per_step_ms)
    memops = sp.last_apply_memops()                       # counted by the library where the copies / memsets are issued
    ms_step = max_over_ranks(ms_total) / args.steps
    value = job.whole_job_value(nc, ms_total / args.steps)
    # hot-cache figure (SURVEY.md 8(d) reporting rule): ONE C and ONE HC buffer, whatever of them fits stays in the 126 MB L2
    hot_total, _, _ = time_mode(sp, mcb, torch, T, V, dCs[:1], dHCs[:1], mode, max(5, min(args.steps, 20)), 3, barrier)
    hot = {"ms_per_step": hot_total / max(5, min(args.steps, 20)), **spread(time_mode.per_step_ms),
           "note": "R = 1: the same C and HC every step (not the headline: inputs of the headline rotate through 3 + 3 buffers)"}

    # ---- end to end through the public API with HOST buffers (pinned), H2D + D2H inside the timed region ----
    hC = [torch.from_numpy(C).pin_memory() for C in Cs]
    hHC = [torch.empty_like(h).pin_memory() for h in hC]
    e2e_steps = max(3, min(args.steps, 10))
    for i in range(2):
        sp.hc_apply_host(T, V, hC[i % R], out_host=hHC[i % R], mode=mode)
    torch.cuda.synchronize(); barrier()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for i in range(e2e_steps):
        sp.hc_apply_host(T, V, hC[i % R], out_host=hHC[i % R], mode=mode)
    b.record(); torch.cuda.synchronize(); barrier()
    e2e_ms = max_over_ranks(a.elapsed_time(b)) / e2e_steps
    e2e_value = world * nc / (e2e_ms * 1e-3)

    # ---- roofline of the dominant kernel ----
    kavg = kms.mean(axis=0) if len(kms) else np.zeros(3)
    if mode == mcb.MAPS and maps_layout and maps_layout.startswith("compact"):
        KERNELS[mode] = ["k_hc_maps2c<M>"]
    if c.M > 12:
        KERNELS[mode] = ["k_big_contract", "k_big_reduce"]
    dom = int(np.argmax(kavg))
    dom_ms = float(kavg[dom])
    flops_step = 8.0 * (tc["one_body_terms"] + tc["two_body_terms_packed"])
    unique_bytes = 32.0 * nc
    fock_bytes = 2.0 * c.M * (nc + nc2)
    alu_peak = fp64_peak_tflops(peaks["sm_max_mhz"])
    if mode == mcb.SPARSE:
        # structured matrix elements: per output one 16-byte gather per non-zero element; the unique bytes are C, HC
        # and the hashing table of the N-particle space
        alg_bytes = unique_bytes + 2.0 * c.M * nc
        roofline = {"bound": "hbm", "kernel": KERNELS[mode][dom], "achieved": alg_bytes / (dom_ms * 1e-3) / 1e9,
                    "peak": peaks["hbm_gbs"], "unit": "GB/s", "peak_source": peaks["source"], "traffic": None,
                    "algorithmic_bytes_per_launch": alg_bytes}
    elif mode == mcb.MAPS:
        alg_bytes = unique_bytes + map_bytes + 2.0 * c.M * nc
        roofline = {"bound": "hbm", "kernel": KERNELS[mode][dom], "achieved": alg_bytes / (dom_ms * 1e-3) / 1e9,
                    "peak": peaks["hbm_gbs"], "unit": "GB/s", "peak_source": peaks["source"], "traffic": None,
                    "algorithmic_bytes_per_launch": alg_bytes}
    else:
        # contract kernel (GEMM mode) carries every two-body term + the folded one-body terms: 8 flop per packed term
        kflops = 8.0 * tc["two_body_terms_packed"] if mode in (mcb.GEMM, mcb.RUNS) else flops_step
        pipe = "dmma_tflops" if mode in (mcb.GEMM, mcb.RUNS) else "dfma_tflops"
        roofline = {"bound": "alu", "kernel": KERNELS[mode][dom], "achieved": kflops / (dom_ms * 1e-3) / 1e12,
                    "peak": fp64_measured[pipe], "unit": "TFLOP/s",
                    "peak_source": f"measured in this run: mcb_fp64_peak, {pipe.split('_')[0].upper()} chains (register-only kernel)",
                    "peak_measured_tflops": fp64_measured,
                    "peak_derived_tflops": alu_peak,
                    "peak_derived_source": f"148 SM x 64 FP64 FMA/clk x 2 x {peaks['sm_max_mhz']:.0f} MHz (DESIGN.md)",
                    "frac_of_derived": kflops / (dom_ms * 1e-3) / 1e12 / alu_peak,
                    "traffic": None, "algorithmic_flops_per_launch": kflops}
    if (args.cfg, mode) in NCU_TRAFFIC_BYTES and not (mode == mcb.MAPS and maps_layout and maps_layout.startswith("compact")):
        roofline["traffic"], roofline["traffic_source"] = NCU_TRAFFIC_BYTES[(args.cfg, mode)]
        roofline["traffic_unit"] = "bytes per launch (dram read + write, one ncu --set full capture)"
    roofline["frac"] = roofline["achieved"] / roofline["peak"]
    roofline["kernel_ms"] = dom_ms
    roofline["kernel_share_of_step"] = dom_ms / ms_step
    hbm_unique = {"bytes_per_step": unique_bytes, "achieved_GBps": unique_bytes / (ms_step * 1e-3) / 1e9,
                  "peak_GBps": peaks["hbm_gbs"], "frac": unique_bytes / (ms_step * 1e-3) / 1e9 / peaks["hbm_gbs"],
                  "note": "unique bytes of C and HC only (32*nc); with dense V the step is bound by FP64 / shared-memory "
                          "throughput and, in RUNS mode, by the class-plane round trip (roofline.traffic), see DESIGN.md"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "ms_per_step_median": step_spread["median_ms"], "ms_per_step_best": step_spread["best_ms"],
        "ms_per_step_worst": step_spread["worst_ms"], "hot_cache": hot,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "complex128 (f64)", "data": "synthetic (seeded, workloads.py)",
        "config": dict(config_dict(c, MODE_NAMES[mode] + (f", {maps_layout}" if maps_layout else "")),
                       l2="inputs larger than L2: 3 rotating C and 3 rotating HC buffers, 16*nc bytes each",
                       replicas="N>1 = independent replicas (path does not shard by north_star)"),
        "applications_per_s": world / (ms_step * 1e-3),
        "terms_per_s": world * (tc["one_body_terms"] + tc["two_body_terms_packed"]) / (ms_step * 1e-3),
        "gflop_per_step": flops_step / 1e9,
        "kernel_ms": {KERNELS[mode][i]: float(kavg[i]) for i in range(len(KERNELS[mode]))},
        "gpu_launches": launches * args.steps,
        # what each apply enqueues besides its kernels, counted by the library at the call sites (mcb_last_apply_memops): the H2D
        # copy of the packed T, V from a pinned ring; RUNS passes them as a kernel argument and clears its tickets with one memset
        "gpu_memops_per_step": {"memcpy_h2d": memops[0], "memset": memops[1], "source": "mcb_last_apply_memops"},
        "roofline": roofline, "hbm_unique": hbm_unique, "setup": setup, "clocks": clk,
        "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": e2e_ms, "steps": e2e_steps,
                "h2d_bytes_per_step": 16 * nc + 16 * (c.M ** 2 + c.M ** 4), "d2h_bytes_per_step": 16 * nc,
                "api": "mcb_hc_apply_host (pinned host C and HC)"},
    }

    # ---- the other variants, short (map-memory vs recompute trade-off) ----
    if args.variants and rank == 0 and world == 1:
        var = {}
        for name, m in (("REHASH", mcb.REHASH), ("GEMM", mcb.GEMM), ("RUNS", mcb.RUNS), ("MAPS_COMPACT", mcb.MAPS), ("MAPS_DENSE", mcb.MAPS),
                        ("SPARSE", mcb.SPARSE)):
            if m == mcb.SPARSE and sp.resolve_mode(T, V) != mcb.SPARSE:
                continue
            if (m == mode and m != mcb.MAPS) or (m in (mcb.GEMM, mcb.RUNS) and c.N < 2) or (m == mcb.RUNS and not 2 <= c.M <= 5):
                continue
            if m == mcb.MAPS and (mode == mcb.MAPS or (name == "MAPS_COMPACT" and c.N < 2)):
                continue
            built = []
            try:
                if m == mcb.MAPS:
                    which = (mcb.MAP2C,) if name == "MAPS_COMPACT" else (mcb.MAP1, mcb.MAP2)
                    need = sum(sp.structure_bytes(w) for w in which)
                    free, _ = torch.cuda.mem_get_info()
                    if need > 0.8 * free:
                        var[name] = {"skipped": f"maps need {need / 1e9:.1f} GB (PAPER.md:264: memory is the limit)"}
                        continue
                    for w in which:
                        sp.build_structure(w); built.append(w)
                ms, km, la = time_mode(sp, mcb, torch, T, V, dCs, dHCs, m, max(3, args.steps // 4), 3, barrier)
                st = max(3, args.steps // 4)
                var[name] = {"ms_per_step": ms / st, "configs_per_s": nc / (ms / st * 1e-3)}
                if m == mcb.MAPS:
                    mb = (4 * tc["P"] ** 2 * nc2 + 8 * nc) if name == "MAPS_COMPACT" else (4 * nc * (c.M * c.M - c.M) + 4 * nc * tc["P"] ** 2)
                    var[name]["map_bytes"] = mb
                    var[name]["map_stream_GBps"] = (mb + unique_bytes + 2.0 * c.M * nc) / (ms / st * 1e-3) / 1e9
                    var[name]["hbm_frac"] = var[name]["map_stream_GBps"] / peaks["hbm_gbs"]
            except Exception as ex:  # report, never hide
                var[name] = {"error": str(ex)}
            for w in built:
                sp.drop_structure(w)
            torch.cuda.empty_cache()
        line["variants"] = var
        # density matrices of the same state: one real SYRK (2P x 2P x nc2) on the DMMA path
        try:
            for _ in range(3):
                sp.rho(dCs[0])
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            reps = 10
            a.record()
            for i in range(reps):
                sp.rho(dCs[i % R])
            b.record(); torch.cuda.synchronize()
            rho_ms = a.elapsed_time(b) / reps
            syrk_flop = 2.0 * (2 * tc["P"]) ** 2 * nc2            # full 2P x 2P real product, 2 flop per MAC
            line["rho"] = {"ms": rho_ms, "configs_per_s": nc / (rho_ms * 1e-3), "launches": int(sp.last_apply_launches()),
                           "tflops_full_syrk": syrk_flop / (rho_ms * 1e-3) / 1e12,
                           "gather_GBps": 16.0 * tc["P"] * nc2 / (rho_ms * 1e-3) / 1e9}
        except Exception as ex:
            line["rho"] = {"error": str(ex)}
        # Lanczos with full re-orthogonalisation (NEXT-2): 16 steps from C, synchronous API
        try:
            import time
            ksteps = 16
            sp.lanczos(T, V, dCs[0], ksteps, mode=mode)                  # (same kmax: the basis workspace is allocated here)
            torch.cuda.synchronize(); t0 = time.perf_counter()
            al, be = sp.lanczos(T, V, dCs[0], ksteps, mode=mode)
            torch.cuda.synchronize(); dt = time.perf_counter() - t0
            line["lanczos"] = {"steps": int(len(al)), "ms_per_step": dt * 1e3 / max(1, len(al)), "alpha0": float(al[0]),
                               "note": "wall clock of the synchronous call: H.C + two Gram-Schmidt passes over all previous vectors + host read-backs per step"}
        except Exception as ex:
            line["lanczos"] = {"error": str(ex)}

    # ---- the other BASELINE.json configs, short (rank 0, N = 1): their numbers in BASELINE.md come from here ----
    if rank == 0 and world == 1 and not args.no_other_configs:
        others = {}
        for oc in (1, 2, 3, 4):
            if oc == args.cfg:
                continue
            try:
                others[f"configs[{oc}]"] = other_config(oc, mcb, torch, peaks, fp64_measured, barrier, 100 if oc == 4 else 10)
            except Exception as ex:  # report, never hide
                others[f"configs[{oc}]"] = {"error": str(ex)}
        line["other_configs"] = others

    # ---- the oracle beside it (rank 0, N=1 only) ----
    if rank == 0 and world == 1 and not args.no_cpu:
        import oracle
        oracle.build()
        v, used, nrows, dt = oracle_sample_rate(c, T, V, Cs[0], args.cpu_seconds)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": used, "kind": "oracle",
                                "sample": f"{nrows} seeded rows of {nc} (rows are independent), {dt:.1f} s, all host threads"}
        v1, used1, nrows1, dt1 = oracle_sample_rate(c, T, V, Cs[0], max(2.0, args.cpu_seconds / 4), nthreads=1)
        line["cpu_baseline_1thread"] = {"value": v1, "unit": UNIT, "cores": used1, "kind": "oracle",
                                        "sample": f"{nrows1} seeded rows, {dt1:.1f} s"}
    sp.close()
    if rank == 0:
        print(json.dumps(line))
    job.close()
    return 0


def run_sweep(args):
    """--sweep: the paper's two timing sweeps (M = 3 with N up to 1000; N = 5 with M up to 25), one
    hc_apply (MCB_AUTO) per point on dense random T, V, C; prints one JSON line.  Context for BASELINE.md, not the metric."""
    import torch
    import paper_2005_13679_b200 as mcb
    pts = [(N, 3) for N in (100, 200, 400, 700, 1000)] + [(5, M) for M in (5, 8, 11, 15, 21, 25)]
    out = []
    for N, M in pts:
        sp = mcb.Space(N, M)
        T, V, C = workloads.make_small_inputs(N, M, sp.nc, seed=2005 + 13 * N + M)
        sp.build_structure(mcb.FOCK_TABLE)
        mode = sp.resolve_mode(T, V)
        dC = torch.from_numpy(C).cuda()
        dH = torch.empty_like(dC)
        for _ in range(max(3, args.warmup)):
            sp.hc_apply(T, V, dC, out=dH)
        torch.cuda.synchronize()
        sp.timing_enable(True)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(args.steps):
            sp.hc_apply(T, V, dC, out=dH)
        b.record(); torch.cuda.synchronize()
        us = 1e3 * a.elapsed_time(b) / args.steps
        kms, _ = sp.timing_read(min(args.steps, 512))
        sp.timing_enable(False)
        k_us = 1e3 * float(kms.sum(axis=1).mean()) if len(kms) else None
        out.append({"N": N, "M": M, "nc": sp.nc, "mode": MODE_NAMES.get(mode, str(mode)) if M <= 12 else "GEMM (many-orbital path)",
                    "us_per_apply": us, "kernels_us": k_us, "configs_per_s": sp.nc / (us * 1e-6),
                    "note": "us_per_apply is back-to-back calls through the Python binding (host-bound below ~50 us); kernels_us = device time of the kernels alone"})
        sp.close()
    print(json.dumps({"sweep": "paper shapes (PAPER.md:184,260,289)", "steps": args.steps, "points": out}))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--cfg", type=int, default=2, choices=range(5))
    ap.add_argument("--mode", default="auto", choices=sorted(MODES))
    ap.add_argument("--impl", default="mcb", choices=["mcb", "reference"])
    ap.add_argument("--variants", action="store_true", help="also time the other hc_apply modes (short)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-setup-rates", action="store_true", help="skip the timing of the hash / map builders")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the short lines of the other BASELINE.json configs")
    ap.add_argument("--compact-maps", action="store_true", help="--mode maps: use the paper's compact table (MCB_MAP2C) even where the dense planes fit")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--sweep", action="store_true", help="time the paper's M = 3 and N = 5 sweeps instead of the metric (one JSON line)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)
    if args.sweep:
        return run_sweep(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
