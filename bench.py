#!/usr/bin/env python
"""bench.py — the hot path of arXiv:2203.17119 (Moebius DWF Dhop / Mpc^dag Mpc / red-black CG) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl dwf|reference] [--workload c4]

One STEP = one pass of the whole hot path on one seeded synthetic subdomain (BASELINE.json configs[3]:
32^4 x Ls=12 Moebius, the configuration the metric is quoted on): a fixed-length red-black CG segment
`dwf_cg(max_iter = --cg-iters)` on Mpc^dag Mpc in fp64 -- every iteration is Mpc (A, Dhop_eo, A Mee^-1,
Dhop_oe, Moo) + Mpc^dag + the fused axpy/norm kernels, plus the segment's |b|^2 and closing true residual.
`value` is the step's nominal GFLOP/s (flop convention in DESIGN.md §6: 1320 per 5-D site per Dhop, 3000 per
Mpc, 240 per iteration of BLAS-1), device-timed with inputs resident in HBM.  `e2e` is the same step through
dwf_cg_host with pinned HOST buffers (H2D/D2H copies and layout packing inside the timed region).
`roofline` is the dominant kernel (half-volume fp64 Dhop) timed per launch by CUDA events on the launching
stream inside the timed steps.  Extra keys report the Dhop / Mpc^dag Mpc sweeps and CG time-to-solution.

N > 1 (torchrun): replicas only -- every rank runs the same step on its own seeded
copy of the workload lattice (the paper's situation: one Dirichlet subdomain per GPU, solved with no communication,
PAPER.md:123); there is no data-path collective, timing is the max over ranks ("scaling": "weak").
--impl reference: the CPU oracle (oracle/), as it stands, on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "DWF Dhop/Mpc^dag Mpc red-black CG hot-path throughput (1320 flop per 5-D site per Dhop)"
UNIT = "GFLOP/s"
FLOP_DHOP = 1320            # per 5-D output site
FLOP_MPC = 2 * 1320 + 360   # per odd 5-D site (a5)
FLOP_BLAS_ITER = 240        # x+=ap, r-=az, |r|^2, p=r+bp, |q|^2 : 5 x 48


def segment_flops(n5h: int, iters: int) -> float:
    """nominal flops of one CG segment on n5h odd 5-D sites: |b|^2, `iters` iterations, closing true residual."""
    per_iter = 2 * FLOP_MPC + FLOP_BLAS_ITER
    closing = 2 * FLOP_MPC + 24 + 48      # A x, b - Ax, |.|^2
    return float(n5h) * (48 + iters * per_iter + closing)


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.t.join(timeout=2)
        sm, smax, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); smax.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def make_inputs(cfg, rank: int):
    from paper_2203_17119_b200 import inputs
    import dataclasses
    c = dataclasses.replace(cfg, gauge_seed=cfg.gauge_seed + 100 * rank, source_seed=cfg.source_seed + 100 * rank)
    U = inputs.make_gauge(c)
    b = inputs.source_half(c.dims, c.Ls, c.source_seed, parity=1)
    return U, b


# ------------------------------------------------------------------------------------------- reference arm
def host_cpu():
    """CPU model, physical cores and the threads the oracle's OpenMP loops use (SURVEY 8d "Oracle timing")."""
    model, phys = "unknown", set()
    try:
        pid = cid = None
        for ln in open("/proc/cpuinfo"):
            k, _, v = ln.partition(":")
            k, v = k.strip(), v.strip()
            if k == "model name":
                model = v
            elif k == "physical id":
                pid = v
            elif k == "core id":
                cid = v
            elif not k and pid is not None:
                phys.add((pid, cid))
                pid = cid = None
    except OSError:
        pass
    try:
        avail = len(os.sched_getaffinity(0))
    except AttributeError:
        avail = os.cpu_count() or 1
    threads = int(os.environ.get("OMP_NUM_THREADS", "0") or 0) or avail
    return {"cpu_model": model, "physical_cores": len(phys) or None, "logical_cpus": os.cpu_count(), "threads": threads}


def _timed(fn, warm, reps):
    for _ in range(warm):
        fn()
    t0 = time.perf_counter()
    for _ in range(reps):
        fn()
    return (time.perf_counter() - t0) / max(reps, 1)


def oracle_setup(cfg, dims, U=None, b=None):
    from oracle.dwf_oracle import Oracle
    from paper_2203_17119_b200 import inputs
    if U is None:
        U = inputs.gauge_weak(dims, cfg.eps, cfg.gauge_seed)
    if b is None:
        b = inputs.source_half(dims, cfg.Ls, cfg.source_seed, parity=1)
    orc = Oracle(dims, cfg.Ls, cfg.M5, cfg.mf, cfg.b5, cfg.c5, antiperiodic_t=cfg.antiperiodic_t, cut=cfg.cut).set_gauge(U)
    return orc, b


def oracle_workload_baseline(cfg, U, b, iters=1):
    """cpu_baseline of the own arm: the oracle, as it stands, on the WORKLOAD ITSELF (same lattice, gauge field and source
    the GPU step ran on): one Dhop (1 warm-up + 3 repetitions), one Mpc^dag Mpc (1 + 2) and one CG segment of `iters`
    iteration(s) with |b|^2 and the closing true residual (1 warm-up + 2 repetitions, each timed: the value is their mean,
    the two samples are reported beside it)."""
    from oracle.dwf_oracle import cg
    orc, b = oracle_setup(cfg, cfg.dims, U, b)
    n5h = b.shape[0] * cfg.Ls
    t_dhop = _timed(lambda: orc.dhop(b, 0, False), 1, 3)
    t_mdagm = _timed(lambda: orc.mdagm(b), 1, 2)
    cg(orc, b, 1e-300, iters)
    segs = [_timed(lambda: cg(orc, b, 1e-300, iters), 0, 1) for _ in range(2)]
    t_seg = sum(segs) / len(segs)
    return {"value": segment_flops(n5h, iters) / t_seg / 1e9, "unit": UNIT, "kind": "oracle", "s_per_step": t_seg,
            "s_per_step_samples": segs,
            "dhop_s": t_dhop, "dhop_gflops": FLOP_DHOP * n5h / t_dhop / 1e9,
            "mdagm_s": t_mdagm, "mdagm_gflops": 2 * FLOP_MPC * n5h / t_mdagm / 1e9,
            "sample": f"the workload itself ({'x'.join(map(str, cfg.dims))} x Ls={cfg.Ls}, the GPU step's gauge field and source): "
                      f"half-volume Dhop 1+3 repetitions, Mpc^dag Mpc 1+2, CG segment of {iters} iteration(s) + |b|^2 + closing "
                      f"true residual 1+2 (the GPU step runs 10 iterations per segment); oracle built -O3 -march=native -fno-fast-math"}


def run_reference(args, cfg):
    """--impl reference: the oracle on the host cores.  A step is the CG segment (`--ref-iters` iteration(s) + |b|^2 + closing
    true residual) on the workload's own lattice when (steps + warmup) such segments fit in ~4 minutes, else on the same
    lattice shortened in t (same parameters, seeds and recipe); one oracle Dhop on a 32^3 x 4 slab calibrates the choice."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle.dwf_oracle import cg
    cpu = host_cpu()
    if args.ref_dims:
        sample = tuple(args.ref_dims)
    else:
        cal = tuple(cfg.dims[:3]) + (4,)
        orc, b = oracle_setup(cfg, cal)
        t_cal = _timed(lambda: orc.dhop(b, 0, False), 1, 2)
        # a 1-iteration segment costs ~17 half-volume Dhops (2 Mpc^dag Mpc + numpy vector work); measured, DESIGN.md section 7
        per_t = 17.0 * t_cal / 4.0 * (args.ref_iters + 1) / 2.0
        lt = cfg.dims[3]
        while lt > 4 and (args.steps + args.warmup) * per_t * lt > 240.0:
            lt //= 2
        sample = tuple(cfg.dims[:3]) + (lt,)
        del orc, b
    orc, b = oracle_setup(cfg, sample)
    n5h = b.shape[0] * cfg.Ls
    dt = _timed(lambda: cg(orc, b, 1e-300, args.ref_iters), args.warmup, args.steps)
    val = segment_flops(n5h, args.ref_iters) / dt / 1e9
    desc = (f"oracle CG segment ({args.ref_iters} iteration(s) + |b|^2 + closing true residual) on "
            f"{'the workload lattice itself' if sample == tuple(cfg.dims) else 'a ' + 'x'.join(map(str, sample)) + ' sample of the workload lattice'}"
            f" ({'x'.join(map(str, sample))} x Ls={cfg.Ls}, same parameters, seeds and recipe); oracle built -O3 -march=native -fno-fast-math")
    base = {"value": val, "unit": UNIT, "cores": cpu["threads"], "kind": "oracle", "sample": desc, **cpu}
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(cfg), "sample": desc},
            "cpu_baseline": base,
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def workload_name(cfg):
    return (f"{cfg.name}: {'x'.join(map(str, cfg.dims))} x Ls={cfg.Ls} Moebius b5={cfg.b5} c5={cfg.c5} M5={cfg.M5} "
            f"mf={cfg.mf}, gauge exp(i*{cfg.eps}*H) seeded SU(3), 2-row compressed links (BASELINE.json configs[3])")


# ------------------------------------------------------------------------------------------------ own arm
HBM_NOMINAL_GBS = 8000.0          # B200 data sheet (SURVEY 8d asks for the fraction against both HBM figures)
# Arithmetic instructions of the plain Dhop kernel per 5-D site, from the SASS histogram profiles/r02_sass_hist.md:
# fp64 2 lanes x 432 DFMA/DADD/DMUL per site-slice, fp32 870 FFMA/FADD/FMUL per site-slice; 1320 flop per site.
ALU_INST_PER_SITE = {"f64": 864.0, "f32": 870.0}
ALU_LANES_PER_SM = {"f64": 64, "f32": 128}         # FP64 / FP32 FMA lanes per SM per clock on sm_100
LIMITER_NOTE = ("sm_latency: the launch time follows the SM clock (ncu at 1.80 GHz against the power-capped clock of the step, "
                "DESIGN.md 5.1); neither HBM (frac) nor the arithmetic pipe (alu.frac_issue) is saturated")


def alu_block(sites, launch_ms, sm_mhz, prec, g):
    """The ALU side of the roofline ('HBM first, with the plain FP32/FP64 ALUs a close second') at the SM clock
    sampled during the timed region: frac_issue = arithmetic instructions issued per second / (SMs x lanes x clock),
    frac_flops = useful flop/s / (SMs x lanes x 2 x clock)."""
    if not sm_mhz or launch_ms <= 0:
        return None
    import torch
    sms = torch.cuda.get_device_properties(g.device).multi_processor_count
    lanes = ALU_LANES_PER_SM[prec]
    t = launch_ms * 1e-3
    inst_peak = sms * lanes * sm_mhz * 1e6
    return {"sm_count": sms, "lanes_per_sm": lanes, "inst_per_site": ALU_INST_PER_SITE[prec],
            "peak_gflops_at_clock": 2 * inst_peak / 1e9, "frac_issue": ALU_INST_PER_SITE[prec] * sites / t / inst_peak,
            "frac_flops": FLOP_DHOP * sites / t / (2 * inst_peak)}


def ev_median(torch, fn, warm=10, min_reps=100, min_s=1.0, max_reps=2000):
    """SURVEY 8d 'GPU timing': >= 10 warm-ups, then one CUDA-event pair per repetition until >= 100 repetitions or >= 1 s of
    kernel time; returns (median ms, first-repetition ms after the warm-ups, repetitions)."""
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    times, total = [], 0.0
    while len(times) < max_reps and (len(times) < min_reps and total < min_s * 1e3):
        batch = []
        for _ in range(10):
            s, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            s.record()
            fn()
            e.record()
            batch.append((s, e))
        torch.cuda.synchronize()
        for s, e in batch:
            t = s.elapsed_time(e)
            times.append(t)
            total += t
    st = sorted(times)
    return st[len(st) // 2], times[0], len(times)


def ev_time(torch, fn, reps):
    s, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    s.record()
    for _ in range(reps):
        fn()
    e.record()
    torch.cuda.synchronize()
    return s.elapsed_time(e) / reps


def run_dwf(args, cfg):
    import torch
    import torch.distributed as dist
    from paper_2203_17119_b200 import api

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    hbm_peak, peak_src = peaks()

    U, b_np = make_inputs(cfg, rank)
    g = api.from_config(cfg, device=f"cuda:{local}")
    g.set_gauge(U)
    if rank != 0 or world != 1 or args.no_cpu:
        U = None                       # rank 0 at N = 1 keeps the host copy for the cpu_baseline leg
    A = api
    b = g.pack(b_np, A.F64, A.ODD)
    x = g.new_native(A.F64, A.ODD)
    n5h = (cfg.V4 // 2) * cfg.Ls
    iters = args.cg_iters

    def step():
        g.cg(b, 1e-300, iters, A.CG_F64, x=x, use_guess=False)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    # ---- timed region: K steps, device-timed, per-launch Dhop events on the ctx stream
    sampler = ClockSampler(local)
    sampler.start()
    g.set_option("time_dhop", 1)
    l0 = g.launch_count()
    barrier()
    s, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s.record()
    for _ in range(args.steps):
        step()
    e.record()
    barrier()
    ms = s.elapsed_time(e)
    dhop_ms, dhop_n, dhop_bytes_total = g.get_option("dhop_ms"), g.get_option("dhop_timed"), g.get_option("dhop_bytes")
    launches = g.launch_count() - l0
    g.set_option("time_dhop", 0)
    clocks = sampler.stop()
    if world > 1:
        t = torch.tensor([ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    ms_step = ms / args.steps
    value = world * segment_flops(n5h, iters) / (ms_step * 1e-3) / 1e9

    # ---- roofline of the dominant kernel: the half-volume fp64 Dhop kernel.  Per launch the library
    # sums the ALGORITHMIC bytes (field in + field out + 12-real links, + the Mee operand for the launch that carries
    # the fused epilogue) next to the event pair it records on its stream.
    dhop_avg_ms = dhop_ms / max(dhop_n, 1)
    dhop_bytes = dhop_bytes_total / max(dhop_n, 1)
    achieved = dhop_bytes / (dhop_avg_ms * 1e-3) / 1e9
    traffic64, traffic_src, stale64 = static_traffic("dhop_f64")
    sm_mhz = (clocks or {}).get("sm_mhz") or None
    sites = n5h                                            # 5-D sites one half-volume launch writes
    roofline = {"bound": "hbm", "dtype": "f64",
                "kernel": "dhop_tma_kernel<double> (half-volume, 12-real links; per CG iteration 3 plain launches + 1 with the fused Mee epilogue)",
                "achieved": achieved, "peak": hbm_peak, "peak_source": peak_src, "unit": "GB/s", "frac": achieved / hbm_peak,
                "traffic": traffic64, "traffic_source": traffic_src, "algorithmic_bytes_per_launch": dhop_bytes,
                "avg_launch_ms": dhop_avg_ms, "launches_timed": int(dhop_n), "share_of_step": dhop_ms / ms if ms > 0 else None,
                "gflops": FLOP_DHOP * n5h / (dhop_avg_ms * 1e-3) / 1e9,
                "traffic_stale": stale64, "frac_nominal": achieved / HBM_NOMINAL_GBS, "peak_nominal": HBM_NOMINAL_GBS,
                "sm_mhz": sm_mhz, "alu": alu_block(sites, dhop_avg_ms, sm_mhz, "f64", g),
                "limiter": LIMITER_NOTE}

    # ---- the same per-launch event timing for the fp32 kernel, inside a long fp32 step with the CG's launch mix (3 plain
    # + 1 fused Dhop per Mpc^dag Mpc): Chebyshev recurrences of Mpc^dag Mpc in fp32 (dwf_chebyshev, order = 2 x cg-iters)
    src32 = g.convert(b, A.F64, A.F32, A.ODD)
    out32 = g.new_native(A.F32, A.ODD)
    for _ in range(3):
        g.chebyshev(src32, 0.0, 5000.0, 2 * iters, A.F32, out=out32)
    g.set_option("time_dhop", 1)
    torch.cuda.synchronize()
    for _ in range(args.steps):
        g.chebyshev(src32, 0.0, 5000.0, 2 * iters, A.F32, out=out32)
    ms32, n32, by32 = g.get_option("dhop_ms"), g.get_option("dhop_timed"), g.get_option("dhop_bytes")
    g.set_option("time_dhop", 0)
    del src32, out32
    avg32, b32 = ms32 / max(n32, 1), by32 / max(n32, 1)
    traffic32, traffic32_src, stale32 = static_traffic("dhop_f32")
    roofline_f32 = {"bound": "hbm", "dtype": "f32", "kernel": "dhop_tma_kernel<float> (same launch mix, inside fp32 Chebyshev steps of Mpc^dag Mpc)",
                    "achieved": b32 / (avg32 * 1e-3) / 1e9, "peak": hbm_peak, "peak_source": peak_src, "unit": "GB/s",
                    "frac": b32 / (avg32 * 1e-3) / 1e9 / hbm_peak, "traffic": traffic32, "traffic_source": traffic32_src,
                    "algorithmic_bytes_per_launch": b32, "avg_launch_ms": avg32, "launches_timed": int(n32),
                    "gflops": FLOP_DHOP * n5h / (avg32 * 1e-3) / 1e9,
                    "traffic_stale": stale32, "frac_nominal": b32 / (avg32 * 1e-3) / 1e9 / HBM_NOMINAL_GBS,
                    "peak_nominal": HBM_NOMINAL_GBS, "sm_mhz": sm_mhz, "alu": alu_block(sites, avg32, sm_mhz, "f32", g),
                    "limiter": LIMITER_NOTE}

    # ---- e2e: the same step through the C ABI with pinned HOST buffers
    b_host = torch.from_numpy(np.ascontiguousarray(b_np).view(np.float64).reshape(-1)).pin_memory()
    x_host = torch.empty_like(b_host).pin_memory()
    g.cg_host(x_host, b_host, 1e-300, iters)
    barrier()
    t0 = time.perf_counter()
    e2e_steps = max(1, min(args.steps, 5))
    for _ in range(e2e_steps):
        g.cg_host(x_host, b_host, 1e-300, iters)
    barrier()
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    if world > 1:
        t = torch.tensor([e2e_s], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    hb = b_host.numel() * 8
    e2e = {"value": world * segment_flops(n5h, iters) / e2e_s / 1e9, "unit": UNIT, "h2d_bytes_per_step": hb,
           "d2h_bytes_per_step": hb, "ms_per_step": e2e_s * 1e3, "call": "dwf_cg_host (pinned canonical fp64 buffers)"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "impl": "dwf",
            "config": {"workload": workload_name(cfg), "step": f"dwf_cg fp64 segment: {iters} iterations + |b|^2 + closing true residual",
                       "l2": "inputs_larger_than_L2 (each half field 1.2 GB, gauge 0.4 GB per parity)", "parallelism": f"replicas x{world}: one seeded {cfg.name} subdomain per GPU, no data-path collective"},
            "clocks": clocks, "gpu_launches": int(launches), "roofline": roofline, "roofline_f32": roofline_f32, "e2e": e2e}

    cpu_leg = rank == 0 and world == 1 and not args.no_cpu
    xs = {} if cpu_leg else None
    if rank == 0 and not args.no_extras:
        line["sweeps"] = sweeps(torch, g, A, cfg, hbm_peak)
        line["cg"] = cg_solutions(g, A, b, cfg, args, keep=xs)
    if cpu_leg:
        cpu = host_cpu()
        line["cpu_baseline"] = {**oracle_workload_baseline(cfg, U, b_np, args.ref_iters), "cores": cpu["threads"], **cpu}
        if xs:                                                              # the converged solves, certified by the oracle
            for name, res in oracle_residuals(cfg, U, b_np, xs).items():
                line["cg"][name]["resid_true_oracle"] = res
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line), flush=True)


def kernel_source_sha():
    """sha256 (first 16 hex digits) of csrc/dwf_dhop_tma.cu with // comments and blank lines removed: the fingerprint
    profiles/dhop_traffic.csv stores for the kernel source its ncu capture was taken from (there is no .git on the GPU box)."""
    import hashlib
    import re
    txt = open(os.path.join(ROOT, "paper_2203_17119_b200", "csrc", "dwf_dhop_tma.cu")).read()
    lines = [re.sub(r"//.*$", "", ln).rstrip() for ln in txt.splitlines()]
    return hashlib.sha256("\n".join(ln for ln in lines if ln.strip()).encode()).hexdigest()[:16]


def static_traffic(kernel):
    """ncu DRAM bytes per launch of the Dhop kernels: NOT measured in this run -- read from the committed ncu summary
    (profiles/dhop_traffic.csv names the capture and the fingerprint of the kernel source it was taken from); null when the
    file has no row.  Returns (bytes, source description, stale): stale = the kernel source has changed since the capture."""
    tp = os.path.join(ROOT, "profiles", "dhop_traffic.csv")
    if os.path.exists(tp):
        import csv
        for row in csv.DictReader(open(tp)):
            if row["kernel"] == kernel:
                stale = row.get("source_sha", "") != kernel_source_sha()
                return (float(row["dram_bytes_per_launch"]),
                        f"static: profiles/dhop_traffic.csv ({row.get('capture', 'ncu --set full')}; kernel source {row.get('source_sha', '?')})", stale)
    return None, "none", None


def sweeps(torch, g, A, cfg, hbm_peak):
    """Kernel-alone sweeps (CUDA events, >= 10 warm-ups, >= 100 repetitions or >= 1 s, median): full-volume Dhop
    and Mpc^dag Mpc in fp32 and fp64."""
    out = {}
    n5h = (cfg.V4 // 2) * cfg.Ls
    for prec, name, B in ((A.F32, "f32", 4), (A.F64, "f64", 8)):
        src = g.new_native(prec, A.FULL).normal_()
        dst = g.new_native(prec, A.FULL)
        ms, first, reps = ev_median(torch, lambda: g.dhop(src, A.FULL, False, prec, out=dst))
        by = 2 * (n5h * 48 * B + (cfg.V4 // 2) * 8 * 12 * B)
        out[f"dhop_{name}"] = {"ms_full_volume": ms, "gflops": FLOP_DHOP * 2 * n5h / ms / 1e6, "gbs": by / ms / 1e6,
                               "frac_hbm": by / ms / 1e6 / hbm_peak, "frac_hbm_nominal": by / ms / 1e6 / HBM_NOMINAL_GBS,
                               "timing": f"median of {reps} repetitions after 10 warm-ups", "ms_first_repetition": first}
        so, do = src[: src.numel() // 2], dst[: dst.numel() // 2]
        ms, first, reps = ev_median(torch, lambda: g.mdagm(so, prec, out=do))
        by = 2 * (5 * n5h * 24 * B + 2 * (cfg.V4 // 2) * 8 * 12 * B)      # fused minimum 5 S_h + 2 G_h per Mpc
        out[f"mdagm_{name}"] = {"ms": ms, "gflops": 2 * FLOP_MPC * n5h / ms / 1e6, "gbs_fused_minimum": by / ms / 1e6,
                                "frac_hbm_fused_minimum": by / ms / 1e6 / hbm_peak,
                                "timing": f"median of {reps} repetitions after 10 warm-ups", "ms_first_repetition": first}
        del src, dst
    return out


def cg_solutions(g, A, b, cfg, args, keep=None):
    """red-black CG time-to-solution on the workload (fp64 and fp32-inner/fp64-outer), once each.  keep: dict that receives
    the canonical host copy of each solution (for the CPU leg's residual recompute)."""
    out = {}
    for mode, name in ((A.CG_F64, "f64"), (A.CG_MIXED, "mixed")):
        x, info, st = g.cg(b, cfg.tol, args.max_iter, mode)
        out[name] = {"tol": cfg.tol, "status": int(st), "iters": info["iters_total"], "restarts": info["restarts"],
                     "resid_true": info["resid_true"], "time_to_solution_s": info["seconds"], "launches": info["launches"]}
        if keep is not None:
            keep[name] = g.unpack(x, A.F64, A.ODD)
        del x
    return out


def oracle_residuals(cfg, U, b, xs):
    """CPU leg (SURVEY 8d reading (3)): the oracle recomputes |b - Mpc^dag Mpc x| / |b| of the GPU's converged solutions with
    one application of its own operator each."""
    orc, b = oracle_setup(cfg, cfg.dims, U, b)
    bn2 = orc.norm2(b)
    return {name: float(np.sqrt(orc.norm2(b - orc.mdagm(x)) / bn2)) for name, x in xs.items()}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="dwf", choices=["dwf", "reference"])
    ap.add_argument("--workload", default="c4")
    ap.add_argument("--cg-iters", type=int, default=10)
    ap.add_argument("--max-iter", type=int, default=20000)
    ap.add_argument("--ref-dims", type=int, nargs=4, default=None,
                    help="reference arm: sample lattice (default: the workload lattice, shortened in t to fit ~4 minutes)")
    ap.add_argument("--ref-iters", type=int, default=1)
    ap.add_argument("--no-extras", action="store_true", help="skip the kernel sweeps and CG time-to-solution")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    args = ap.parse_args()
    from paper_2203_17119_b200 import inputs
    cfg = inputs.CONFIGS[args.workload]
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_dwf(args, cfg)


if __name__ == "__main__":
    main()
