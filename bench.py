#!/usr/bin/env python
"""bench.py -- the headline measurement: one step = one 3D R2C + C2R pair (all hot-path passes)
on the 1024^3 fp32 grid of BASELINE.json configs[2], inputs resident in HBM.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--size 1024] [--slabs 8]

Prints ONE JSON line (rank 0).  `value` = GFLOP/s by BASELINE.json's convention
(2.5 N^3 log2 N^3 per real transform, 5 per pair; the paper's convention, is 2x).
Multi-GPU (torchrun): the ONE grid is slab-decomposed over the N ranks -- the paper's method
(paper_2202_12756_b200/dist.py) -- so the scaling is strong; `--exchange unified`
(the y pass stores straight into the peers' memory over NVLink; what `auto`, the default, picks wherever the
VMM peer mapping can work) or `chunks` (all-to-all over NCCL between the stages); the line carries both
back-ends' T_comm.  `--gpus N` must match the launcher's WORLD_SIZE (N > 1: torchrun), else the run exits non-zero.
The default single-GPU run also times a few pairs of the other BASELINE.json configs (1536^3 and 2048^3 fp32,
1024^3 fp64) into `config.other_configs`.  `--impl reference` times the fp64 CPU oracle on a bounded sample (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "GFLOP/s per 3D R2C+C2R pair (5*N^3*log2(N^3) flop per pair), fp32"
FALLBACK_HBM_GBS = 6650.0        # /opt/skills/guides/B200_PROFILING.md fallback


def flops_pair(shape):
    n = shape[0] * shape[1] * shape[2]
    return 5.0 * n * math.log2(n)


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def stored_traffic(kernel_name, n, dtype):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of a kernel from the committed ncu --set full
    captures (profiles/traffic.csv: kernel,N,dtype,dram_bytes_per_launch,source).  None when no capture exists
    for the configuration being run: a stored number is never stretched over another size."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as fh:
            for line in fh:
                parts = line.strip().split(",")
                if len(parts) >= 5 and parts[0] == kernel_name and parts[1] == str(n) and parts[2] == dtype:
                    return {"dram_bytes_per_launch": float(parts[3]), "source": parts[4],
                            "kind": "stored ncu capture, not measured by this run"}
    except Exception:
        pass
    return None


def workload_for(n):
    """The BASELINE.json config a cubic size belongs to: (label, generator name, default virtual_slabs)."""
    if n == 1024:
        return "configs[2]: 1024^3 fp32 turbulence-like field (128 random-phase modes, |u|^2 ~ k^-5/3, DESIGN.md R16)", "turbulence", 8
    if n == 1536:
        return "configs[3]: 1536^3 fp32 i.i.d. N(0,1)", "normal", 16
    if n == 2048:
        return "configs[4]: 2048^3 fp32 i.i.d. uniform[-1,1)", "uniform", 128
    return "%d^3 fp32 i.i.d. uniform[-1,1) (not a BASELINE.json config)" % n, "uniform", 8


def make_field(kind, shape, seed, device, x_range=None):
    import torch
    from paper_2202_12756_b200 import inputs
    if kind == "turbulence":
        return inputs.turbulence_grid(shape, torch.float32, seed=seed, device=device, x_range=x_range)[0]
    if kind == "normal":
        return inputs.normal_grid(shape, torch.float32, seed=seed, device=device, x_range=x_range)
    return inputs.uniform_grid(shape, torch.float32, seed=seed, device=device, x_range=x_range)


class ClockSampler:
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(gpu_index), "--query-gpu=" + self.QUERY,
                 "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=self.tmp, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()
        try:
            self.tmp.flush()
            self.tmp.seek(0)
            sm, mx, reasons = [], [], set()
            names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
            for line in self.tmp.read().splitlines():
                parts = [p.strip() for p in line.split(",")]
                if len(parts) < 7:
                    continue
                try:
                    sm.append(float(parts[0]))
                    mx.append(float(parts[1]))
                except ValueError:
                    continue
                for nm, val in zip(names, parts[3:7]):
                    if val.lower().startswith("active"):
                        reasons.add(nm)
            if sm:
                out = {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx),
                       "reasons": sorted(reasons), "samples": len(sm)}
        finally:
            self.tmp.close()
            try:
                os.unlink(self.tmp.name)
            except OSError:
                pass
        return out


# ------------------------------------------------------------------------------------------
# reference arm: the oracle, as it stands, on the host cores
# ------------------------------------------------------------------------------------------
def oracle_sample_cube(budget_s, cores):
    """Largest power-of-two cube whose oracle pair is expected to fit the per-step budget,
    calibrated by one 64^3 pair (the oracle is O(n log n) per line)."""
    import numpy as np
    import oracle
    f = np.random.Generator(np.random.PCG64(0)).uniform(-1, 1, (64, 64, 64))
    t0 = time.perf_counter()
    oracle.c2r(oracle.r2c(f, nthreads=cores), 64, nthreads=cores)
    t64 = max(time.perf_counter() - t0, 1e-4)
    best = 64
    for n in (128, 256, 512):
        est = t64 * flops_pair((n, n, n)) / flops_pair((64, 64, 64)) * 1.5
        if est <= budget_s:
            best = n
    return best


def time_oracle(sample_n, field, steps, warmup, cores):
    """Oracle R2C + C2R on the [0:sample_n]^3 corner of `field` (fp32 values promoted to fp64)."""
    import numpy as np
    import oracle
    sub = np.ascontiguousarray(field[:sample_n, :sample_n, :sample_n]).astype(np.float64)
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        F = oracle.r2c(sub, nthreads=cores)
        oracle.c2r(F, sample_n, nthreads=cores)
        dt = time.perf_counter() - t0
        if it >= warmup:
            times.append(dt)
    t = sum(times) / len(times)
    return flops_pair((sample_n,) * 3) / t / 1e9, t


def run_reference(args):
    _world, rank, _local = dist_env()
    if rank != 0:                                   # rank 0 alone runs and prints the reference arm
        return
    import numpy as np
    import oracle
    from paper_2202_12756_b200 import inputs
    import torch
    oracle.build_oracle()
    cores = oracle.max_threads()
    n = args.n
    total = max(1, args.steps + args.warmup)
    sample_n = min(n, oracle_sample_cube(150.0 / total, cores))
    # the same kind of field as the CUDA arm, generated at the sample size on the host
    field, _ = inputs.turbulence_grid((sample_n,) * 3, torch.float32, seed=0, device="cpu")
    gf, t = time_oracle(sample_n, field.numpy(), args.steps, args.warmup, cores)
    sample = ("oracle R2C+C2R on a %d^3 grid of the same field family (fp64), rate by the same flop formula; "
              "the full %d^3 pair would take ~%.0f s at this rate" % (sample_n, n, flops_pair((n,) * 3) / (gf * 1e9)))
    line = {
        "impl": "reference", "metric": METRIC, "value": gf, "unit": "GFLOP/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": t * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": "%s, R2C+C2R pair" % workload_for(n)[0],
                   "sample": sample},
        "cpu_baseline": {"value": gf, "unit": "GFLOP/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": gf, "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------
# multi-process plumbing (one process per GPU; replicas, no data-path collective -- DESIGN.md 8)
# ------------------------------------------------------------------------------------------
def dist_env():
    return (int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")),
            int(os.environ.get("LOCAL_RANK", "0")))


def dist_init(world, backend, device=None):
    """torch.distributed process group for world > 1 (rendezvous from MASTER_ADDR/PORT), else None."""
    if world <= 1:
        return None
    import torch.distributed as dist
    if device is not None:
        dist.init_process_group(backend, device_id=device)
    else:
        dist.init_process_group(backend)
    return dist


def max_over_ranks(x, dist, device="cpu"):
    """The slowest rank's time: a job of replicas is as slow as its slowest member."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_gflops(shape, seconds_per_step):
    """Whole-job rate: ONE grid of `shape`, slab-decomposed over all ranks, transformed in the (max-over-ranks) time."""
    return flops_pair(shape) / seconds_per_step / 1e9


# ------------------------------------------------------------------------------------------
# the oracle timed beside the CUDA arm (rank 0, N = 1 only): SURVEY.md 8(d), PAPER.md:103 protocol
# ------------------------------------------------------------------------------------------
def cpu_baseline_leg(field_dev, n, gpu_spec_natural=None):
    """The fp64 oracle, as it stands (gcc -O2 -fopenmp, no tuning), on the GPU box's host cores:
    all cores on the WHOLE n^3 grid of the bench workload when host memory allows (else on the largest
    power-of-two corner that does, named as such), and single-threaded on the 256^3 and 64^3 corners.
    When the whole grid was transformed, the oracle's spectrum also checks the timed CUDA result entry by entry."""
    import numpy as np
    import oracle
    oracle.build_oracle()
    cores = oracle.max_threads()
    try:
        import psutil
        avail = psutil.virtual_memory().available
    except Exception:
        avail = 0
    full_n = n if (n <= 1024 and avail >= 6 * 8 * n ** 3) else min(n, 512)
    w = np.random.Generator(np.random.PCG64(0)).uniform(-1, 1, (64, 64, 64))
    oracle.c2r(oracle.r2c(w, nthreads=cores), 64, nthreads=cores)          # warm-up: library load, thread pool
    sub = field_dev[:full_n, :full_n, :full_n].contiguous().cpu().numpy().astype(np.float64)
    t0 = time.perf_counter()
    F = oracle.r2c(sub, nthreads=cores)
    t1 = time.perf_counter()
    back = oracle.c2r(F, full_n, nthreads=cores)
    t2 = time.perf_counter()
    del back
    out = {"value": flops_pair((full_n,) * 3) / (t2 - t0) / 1e9, "unit": "GFLOP/s", "cores": cores, "kind": "oracle",
           "sample": ("oracle R2C+C2R (fp64) on the %s, all %d cores: forward %.1f s + inverse %.1f s; rate by the "
                      "same flop formula" % ("WHOLE %d^3 grid" % n if full_n == n else "[0:%d]^3 corner of the %d^3 grid"
                                             % (full_n, n), cores, t1 - t0, t2 - t1)),
           "seconds_per_pair": t2 - t0, "grid": full_n, "build": "gcc -O2 -std=c11 -fopenmp -ffp-contract=off"}
    if gpu_spec_natural is not None and full_n == n:
        num = den = 0.0
        for x0 in range(0, n, 64):
            d = gpu_spec_natural[x0:x0 + 64].cpu().numpy().astype(np.complex128) - F[x0:x0 + 64]
            num += float(np.sum(d.real ** 2 + d.imag ** 2))
            den += float(np.sum(F[x0:x0 + 64].real ** 2 + F[x0:x0 + 64].imag ** 2))
        out["gpu_vs_oracle_rel_l2"] = math.sqrt(num / den)
        out["gpu_vs_oracle_bound"] = 2e-6 * math.log2(n ** 3)
    del F, sub
    single = {}
    for m in (64, 256):
        if m > n:
            continue
        c = field_dev[:m, :m, :m].contiguous().cpu().numpy().astype(np.float64)
        t0 = time.perf_counter()
        oracle.c2r(oracle.r2c(c, nthreads=1), m, nthreads=1)
        dt = time.perf_counter() - t0
        single["%d^3" % m] = {"seconds_per_pair": dt, "gflops": flops_pair((m,) * 3) / dt / 1e9}
    out["single_thread"] = single
    return out


# ------------------------------------------------------------------------------------------
# CUDA arm
# ------------------------------------------------------------------------------------------
def alg_bytes_per_launch(plan_real_bytes):
    """Algorithmic bytes of one launch of each full-array kernel: one read + one write of the array;
    the packed intermediate [Nx][Ny][Nz/2] complex has the real array's size.  The fused z+y kernels exchange the
    plane through an L2-resident ring: HBM sees one read + one write for the two passes together."""
    b = 2 * plan_real_bytes
    return {k: b for k in ("z_r2c", "y_c2c_fwd", "x_c2c_fwd", "x_c2c_inv", "y_c2c_inv", "z_c2r", "zy_r2c_fused", "yz_c2r_fused")}


OTHER_CONFIGS = (   # (n, dtype name, generator, virtual_slabs, label): the BASELINE.json configs beside the headline
    (1536, "f32", "normal", 16, "configs[3]: 1536^3 fp32 i.i.d. N(0,1)"),
    (2048, "f32", "uniform", 128, "configs[4]: 2048^3 fp32 i.i.d. uniform[-1,1)"),
    (1024, "f64", "uniform", 128, "configs[4]: 1024^3 fp64 i.i.d. uniform[-1,1)"),
)


def other_config_leg(pkg, n, dname, kind, p, label, dev, local_rank, steps=3, warmup=2):
    """A few R2C+C2R pairs of another BASELINE.json config, timed like the headline (CUDA events around `steps` pairs
    after `warmup`, clocks sampled during them), plus the per-kernel durations and the round trip.  Device timed only."""
    import torch
    from paper_2202_12756_b200 import inputs
    dtype = torch.float32 if dname == "f32" else torch.float64
    shape = (n, n, n)
    free, _tot = torch.cuda.mem_get_info(dev)
    esize = 4 if dname == "f32" else 8
    need = 4.1 * n ** 3 * esize
    if free < need:
        return {"workload": label, "dtype": dname, "skipped": "needs %.0f GiB of free HBM, %.0f free" % (need / 2 ** 30, free / 2 ** 30)}
    plan = pkg.Plan(*shape, dtype=dtype, virtual_slabs=p)
    gen = inputs.normal_grid if kind == "normal" else inputs.uniform_grid
    field = gen(shape, dtype, seed=0, device=dev)
    spec, back, work = plan.empty_complex(dev), plan.empty_real(dev), plan.empty_workspace(dev)
    stream = torch.cuda.current_stream(dev)

    def step():
        plan.r2c(field, spec, work, stream)
        plan.c2r(spec, back, work, stream)

    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(local_rank)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        step()
    e1.record(stream)
    torch.cuda.synchronize()
    ms_step = e0.elapsed_time(e1) / steps
    clocks = sampler.stop()
    plan.timing_enable(steps)
    for _ in range(steps):
        step()
    torch.cuda.synchronize()
    per_kernel = {}
    for which in (0, 1):
        t, calls = plan.timing_read(which)
        for k, v in t.items():
            per_kernel[k] = v / max(1, calls)
    plan.timing_enable(0)
    rt = max((back[i] - field[i]).abs().max().item() for i in range(n)) / max(field[i].abs().max().item() for i in range(n))
    peak, _src = measured_peak()
    alg = {k: v for k, v in alg_bytes_per_launch(plan.real_bytes).items() if k in per_kernel}
    impls = dict(zip(plan.launch_names(0) + plan.launch_names(1), plan.launch_impls(0) + plan.launch_impls(1)))
    out = {"workload": "%s, R2C+C2R pair, virtual_slabs=%d" % (label, p), "dtype": dname, "steps": steps, "warmup": warmup,
           "ms_per_step": ms_step, "value_gflops": job_gflops(shape, ms_step * 1e-3),
           "all_kernels_ms": per_kernel, "all_kernels_impl": impls,
           "all_kernels_frac_of_hbm_peak": {k: alg[k] / (per_kernel[k] * 1e-3) / 1e9 / peak for k in alg},
           "array_passes_per_pair": len(alg),
           "pair_frac_of_pass_roofline": (sum(alg.values()) / peak / 1e9) / (ms_step * 1e-3),
           "pair_frac_of_one_read_one_write": (2 * 2 * plan.real_bytes / peak / 1e9) / (ms_step * 1e-3),
           "round_trip_rel_err": rt, "round_trip_bound": (2e-6 if dname == "f32" else 1e-13) * math.log2(n ** 3),
           "clocks": clocks}
    plan.close()
    del field, spec, back, work
    torch.cuda.empty_cache()
    return out


def run_cuda(args):
    import torch
    import paper_2202_12756_b200 as pkg

    world, rank, local_rank = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the FFT path has no CPU fallback")
    if world > 1 or args.dist:
        return run_cuda_dist(args)
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)

    n = args.n
    label, kind, p_default = workload_for(n)
    p = args.slabs if args.slabs > 0 else p_default
    shape = (n, n, n)
    plan = pkg.Plan(*shape, dtype=torch.float32, virtual_slabs=p)
    field = make_field(kind, shape, 0, dev)
    spec = plan.empty_complex(dev)
    back = plan.empty_real(dev)
    work = plan.empty_workspace(dev)
    stream = torch.cuda.current_stream(dev)

    def step():
        plan.r2c(field, spec, work, stream)
        plan.c2r(spec, back, work, stream)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    # ---- the headline: K steps between two events, nothing else on the stream ----
    sampler = ClockSampler(local_rank)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    torch.cuda.synchronize()
    ms_step = e0.elapsed_time(e1) / args.steps
    clocks = sampler.stop()
    value = job_gflops(shape, ms_step * 1e-3)
    # ---- per-kernel durations: a second loop with CUDA events between the launches (fft3d_timing_*) ----
    plan.timing_enable(args.steps)
    for _ in range(args.steps):
        step()
    torch.cuda.synchronize()
    t_fwd, c_fwd = plan.timing_read(0)
    t_inv, c_inv = plan.timing_read(1)
    plan.timing_enable(0)

    # sanity: the timed result is a real transform pair (round trip recovers the field)
    # plane by plane: no array-sized temporaries (2048^3 leaves ~18 GiB free)
    rt_num = max((back[i] - field[i]).abs().max().item() for i in range(n))
    rt_err = rt_num / max(field[i].abs().max().item() for i in range(n))
    tol = 2e-6 * math.log2(n ** 3)

    # ---- roofline of the dominant kernel ----
    per_kernel = {}
    for d, calls in ((t_fwd, c_fwd), (t_inv, c_inv)):
        for k, v in d.items():
            per_kernel[k] = v / max(1, calls)
    real_b, cplx_b = plan.real_bytes, plan.complex_bytes
    alg_bytes = {k: v for k, v in alg_bytes_per_launch(real_b).items() if k in per_kernel}
    big = {k: per_kernel[k] for k in alg_bytes}
    dom = max(big, key=big.get)
    peak, peak_src = measured_peak()
    achieved = alg_bytes[dom] / (big[dom] * 1e-3) / 1e9
    n_pass = len(alg_bytes)
    stored = stored_traffic(dom, n, "f32")
    impls = dict(zip(plan.launch_names(0) + plan.launch_names(1), plan.launch_impls(0) + plan.launch_impls(1)))
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": stored["dram_bytes_per_launch"] if stored else None,
                "traffic_source": stored, "peak_source": peak_src,
                "algorithmic_bytes": alg_bytes[dom], "ms_per_launch": big[dom],
                "all_kernels_ms": per_kernel, "all_kernels_impl": impls,
                "all_kernels_gbs": {k: alg_bytes[k] / (per_kernel[k] * 1e-3) / 1e9 for k in alg_bytes},
                "per_kernel_ms_sum": sum(per_kernel.values()),
                "array_passes_per_pair": n_pass,
                "pair_bytes_all_passes": sum(alg_bytes.values()),
                "pair_frac_of_pass_roofline": (sum(alg_bytes.values()) / peak / 1e9) / (ms_step * 1e-3),
                "pair_frac_of_6pass_roofline": (6 * 2 * real_b / peak / 1e9) / (ms_step * 1e-3),
                "pair_frac_of_one_read_one_write": (2 * 2 * real_b / peak / 1e9) / (ms_step * 1e-3)}

    # ---- the oracle timed beside it, and checking the timed spectrum ----
    cpu_baseline = None
    if not args.no_cpu_baseline:
        nat = plan.to_natural(spec).contiguous() if n <= 1024 else None
        cpu_baseline = cpu_baseline_leg(field, n, nat)
        del nat

    # ---- end to end through the host entry points (pinned host buffers, copies timed) ----
    e2e = None
    if not args.no_e2e:
        h_in = torch.empty(shape, dtype=torch.float32).pin_memory()
        h_spec = torch.empty(plan.n_complex, dtype=torch.complex64).pin_memory()
        h_back = torch.empty(shape, dtype=torch.float32).pin_memory()
        h_in.copy_(field)
        # free the device-resident bench buffers first: the host entry points own their own
        spec = back = work = None
        torch.cuda.empty_cache()
        plan.r2c_host(h_in, h_spec)                     # warm-up (allocates the plan's buffers)
        plan.c2r_host(h_spec, h_back)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            plan.r2c_host(h_in, h_spec)
            plan.c2r_host(h_spec, h_back)
        torch.cuda.synchronize()
        dt = (time.perf_counter() - t0) / args.e2e_steps
        e2e_rt = (h_back - h_in).abs().max().item() / h_in.abs().max().item()
        e2e = {"value": job_gflops(shape, dt), "unit": "GFLOP/s", "ms_per_step": dt * 1e3,
               "h2d_bytes_per_step": real_b + cplx_b, "d2h_bytes_per_step": cplx_b + real_b,
               "round_trip_rel_err": e2e_rt}

    # ---- the other BASELINE.json configs, a few pairs each, after the headline has released its buffers ----
    n_launches = args.steps * (plan.launches(0) + plan.launches(1))
    other = None
    if n == 1024 and not args.no_other_configs:
        plan.close()                                    # also frees the host entry points' device buffers
        field = spec = back = work = None
        torch.cuda.empty_cache()
        other = [other_config_leg(pkg, *cfg, dev, local_rank) for cfg in OTHER_CONFIGS]

    line = {
        "metric": METRIC, "value": value, "unit": "GFLOP/s", "n_gpus": 1,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step,
        "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": "%s, R2C+C2R pair, virtual_slabs=%d" % (label, p),
                   "l2": "inputs (%.1f GiB per array) are far larger than the 126 MB L2; no flush needed"
                         % (real_b / 2 ** 30),
                   "parallelism": "1 GPU",
                   "gflops_paper_convention": 2 * value,
                   "round_trip_rel_err": rt_err, "round_trip_bound": tol,
                   "other_configs": other},
        "clocks": clocks, "e2e": e2e,
        "gpu_launches": n_launches,
        "roofline": roofline, "cpu_baseline": cpu_baseline,
    }
    print(json.dumps(line), flush=True)
    if not (rt_err <= tol):
        raise SystemExit("round trip error %.3e exceeds %.3e: the timed path is wrong" % (rt_err, tol))
    if cpu_baseline and cpu_baseline.get("gpu_vs_oracle_rel_l2", 0.0) > tol:
        raise SystemExit("the timed spectrum is off the oracle by %.3e (bound %.3e)" % (cpu_baseline["gpu_vs_oracle_rel_l2"], tol))


def dist_launches_per_pair(plan):
    """Kernels one rank launches per R2C+C2R pair: the stages of the plan's current variant (fft3d_launches counts the
    z/y/x passes and the Nyquist fix-ups of both directions) plus the two plane-extraction kernels of the distributed
    bookkeeping (fft3d_dist_fwd_col0, fft3d_dist_inv_planes)."""
    lib = plan._lib
    return int(lib.fft3d_launches(plan._h, 0)) + int(lib.fft3d_launches(plan._h, 1)) + 2


def choose_exchange(asked, D, dist, dev, n, world, rank):
    """'unified' (the y pass stores into / loads from the peers' memory over a CUDA-VMM mapping) where it
    can work, else 'chunks' (NCCL all-to-all).  It needs: a part size that is a multiple of the VMM granularity, peer
    access from this GPU to every other rank's GPU, and all ranks on one host.  Every rank takes the same decision (MIN
    over the ranks).  Returns (exchange, reason)."""
    import torch
    if asked in ("chunks", "unified"):
        return asked, "asked for"
    part = 8 * n * (n // world) * (n // 2)              # [Nx][Ny/G][Nz/2] complex64
    ok, why = True, "VMM peer mapping usable"
    if not D.UnifiedExchange.usable(part):
        ok, why = False, "part size %d is not a multiple of the VMM granularity" % part
    elif world > 1:
        me = dev.index
        peers = [g for g in range(torch.cuda.device_count()) if g != me][:world - 1]
        if len(peers) < world - 1 or not all(torch.cuda.can_device_access_peer(me, g) for g in peers):
            ok, why = False, "no peer access between the ranks' GPUs"
    if world > 1:
        t = torch.tensor([1.0 if ok else 0.0], device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MIN)
        if ok and t.item() < 1.0:
            ok, why = False, "another rank cannot use the VMM peer mapping"
    return ("unified" if ok else "chunks"), ("auto: " + why)


def run_cuda_dist(args):
    """N > 1: ONE n^3 grid slab-decomposed over the N ranks (strong scaling), the paper's method: x-slabs, z+y
    transforms local, exchange, x transform on y-slabs; inverse the reverse."""
    import torch
    from paper_2202_12756_b200 import dist as D

    world, rank, local_rank = dist_env()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world == 1:                                  # --dist on one rank: a one-member group
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29531")
        import torch.distributed as dist
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=dev)
    else:
        dist = dist_init(world, "nccl", dev)
    n = args.n
    label, kind, _p = workload_for(n)
    shape = (n, n, n)
    Nxl = n // world
    exchange, why = choose_exchange(args.exchange, D, dist, dev, n, world, rank)
    fft = D.SlabFFT.create(n, n, n, torch.float32, dist, dev, exchange=exchange)
    plan = fft.plan
    field = make_field(kind, shape, 0, dev, x_range=(rank * Nxl, (rank + 1) * Nxl))
    spec = plan.empty_spec_part(dev)
    back = plan.empty_real_slab(dev)
    stream = torch.cuda.current_stream(dev)

    def barrier():
        dist.barrier()
        torch.cuda.synchronize()

    def step():
        fft.forward(field, spec)
        fft.inverse(spec, back)

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    barrier()
    ms_step = max_over_ranks(e0.elapsed_time(e1) / args.steps, dist, dev)
    clocks = sampler.stop() if sampler is not None else None
    # T_comp / T_comm as the paper's Table 2: a second loop with events between the phases
    fft.timed = True
    for _ in range(args.steps):
        step()
    barrier()
    fft.collect_times()
    fft.timed = False
    t_comp = max_over_ranks(fft.times["comp"] / args.steps, dist, dev)
    t_comm = max_over_ranks(fft.times["comm"] / args.steps, dist, dev)
    # the other exchange back-end, a few steps, for its T_comm beside the timed one's (same kernels, same buffers)
    t_comm_other, other = None, ("chunks" if exchange == "unified" else "unified")
    if other == "chunks" or choose_exchange("auto", D, dist, dev, n, world, rank)[0] == "unified":
        fft2 = D.SlabFFT.create(n, n, n, torch.float32, dist, dev, exchange=other)
        for k in range(1 + args.steps):
            fft2.timed = k > 0
            fft2.forward(field, spec)
            fft2.inverse(spec, back)
        barrier()
        fft2.collect_times()
        t_comm_other = max_over_ranks(fft2.times["comm"] / args.steps, dist, dev)
        fft2.close()
    rt_num = max_over_ranks((back - field).abs().max().item(), dist, dev)
    rt_den = max_over_ranks(field.abs().max().item(), dist, dev)
    rt_err = rt_num / rt_den
    tol = 2e-6 * math.log2(n ** 3)
    value = job_gflops(shape, ms_step * 1e-3)

    # end to end: every rank's slab comes from pinned host memory and its results go back each step
    e2e = None
    if not args.no_e2e:
        h_in = torch.empty(field.shape, dtype=torch.float32).pin_memory()
        h_spec = torch.empty(spec.shape, dtype=torch.complex64).pin_memory()
        h_back = torch.empty(field.shape, dtype=torch.float32).pin_memory()
        h_in.copy_(field)
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            field.copy_(h_in, non_blocking=True)
            fft.forward(field, spec)
            h_spec.copy_(spec, non_blocking=True)
            spec.copy_(h_spec, non_blocking=True)
            fft.inverse(spec, back)
            h_back.copy_(back, non_blocking=True)
        barrier()
        dt = max_over_ranks((time.perf_counter() - t0) / args.e2e_steps, dist, dev)
        sb, rb = spec.numel() * 8, field.numel() * 4
        e2e = {"value": job_gflops(shape, dt), "unit": "GFLOP/s", "ms_per_step": dt * 1e3,
               "h2d_bytes_per_step": world * (rb + sb), "d2h_bytes_per_step": world * (sb + rb),
               "round_trip_rel_err": (h_back - h_in).abs().max().item() / h_in.abs().max().item()}

    if rank == 0:
        peak, peak_src = measured_peak()
        arr = 2 * 4 * n ** 3                         # one read + one write of the (global) real-sized array
        line = {
            "metric": METRIC, "value": value, "unit": "GFLOP/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step,
            "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": "%s, R2C+C2R pair, slab-decomposed over %d GPUs" % (label, world),
                       "l2": "per-rank arrays are %.2f GiB; inputs are not re-used between steps" % (4 * n ** 3 / world / 2 ** 30),
                       "parallelism": "slab decomposition x%d (PAPER.md:54), exchange=%s (%s)" % (world, exchange, why),
                       "t_comm_ms_by_exchange": {exchange: t_comm, other: t_comm_other},
                       "gflops_paper_convention": 2 * value,
                       "t_comp_ms": t_comp, "t_comm_ms": t_comm, "comm_fraction_r": t_comm / max(1e-9, t_comp + t_comm),
                       "chunk_bytes": 8 * (n // world) * (n // world) * (n // 2),
                       "round_trip_rel_err": rt_err, "round_trip_bound": tol},
            "clocks": clocks, "e2e": e2e,
            "gpu_launches": args.steps * dist_launches_per_pair(plan),
            "roofline": {"bound": "hbm", "kernel": "pair", "achieved": 6 * arr / world / (ms_step * 1e-3) / 1e9,
                         "peak": peak, "unit": "GB/s", "frac": 6 * arr / world / (ms_step * 1e-3) / 1e9 / peak,
                         "traffic": None, "peak_source": peak_src,
                         "note": "per-GPU share of the 6-pass design bytes over the whole step (exchange included)"},
            "cpu_baseline": None,
        }
        print(json.dumps(line), flush=True)
        if not (rt_err <= tol):
            raise SystemExit("round trip error %.3e exceeds %.3e: the timed path is wrong" % (rt_err, tol))
    fft.close()
    dist.destroy_process_group()


# ------------------------------------------------------------------------------------------
# CUDA arm, 3D C2C transform (--transform c2c; single GPU, the widening row SURVEY.md 8(f)-3)
# ------------------------------------------------------------------------------------------
def run_cuda_c2c(args):
    import torch
    import paper_2202_12756_b200 as pkg
    from paper_2202_12756_b200 import inputs

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the FFT path has no CPU fallback")
    torch.cuda.set_device(0)
    n, p = args.n, (args.slabs if args.slabs > 0 else 8)
    shape = (n, n, n)
    plan = pkg.PlanC2C(*shape, dtype=torch.float32, virtual_slabs=p)
    f = inputs.complex_grid(shape, torch.complex64, seed=0, device="cuda").reshape(-1)
    spec, back, work = plan.empty_complex("cuda"), plan.empty_complex("cuda"), plan.empty_workspace("cuda")
    stream = torch.cuda.current_stream()

    def step():
        plan.c2c(f, -1, spec, work, stream)
        plan.c2c(spec, +1, back, work, stream)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    plan.timing_enable(args.steps)
    sampler = ClockSampler(0)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    torch.cuda.synchronize()
    ms_step = e0.elapsed_time(e1) / args.steps
    clocks = sampler.stop()
    per_kernel = {}
    for which in (0, 1):
        d, calls = plan.timing_read(which)
        per_kernel.update({k: v / max(1, calls) for k, v in d.items()})
    plan.timing_enable(0)
    rt_err = max((back[i:i + (1 << 26)] - f[i:i + (1 << 26)]).abs().max().item() for i in range(0, n ** 3, 1 << 26))
    fmax = max(f[i:i + (1 << 26)].abs().max().item() for i in range(0, n ** 3, 1 << 26))
    rt_err = rt_err / fmax                         # round-trip max-abs error relative to max|f|
    tol = 2e-6 * math.log2(n ** 3)
    pass_b = 2 * plan.complex_bytes              # one read + one write of the complex array
    dom = max(per_kernel, key=per_kernel.get)
    peak, peak_src = measured_peak()
    achieved = pass_b / (per_kernel[dom] * 1e-3) / 1e9
    flops = 2 * 5.0 * n ** 3 * math.log2(n ** 3)  # 5 N log2 N per complex transform, two transforms
    line = {
        "metric": "GFLOP/s per 3D C2C forward+inverse pair (10*N^3*log2(N^3) flop per pair), fp32",
        "value": flops / (ms_step * 1e-3) / 1e9, "unit": "GFLOP/s", "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": "%d^3 complex64 grid, re/im i.i.d. uniform[-1,1), C2C forward+inverse pair, "
                               "virtual_slabs=%d" % (n, p),
                   "l2": "arrays (%.1f GiB each) are far larger than the 126 MB L2; no flush needed"
                         % (plan.complex_bytes / 2 ** 30),
                   "round_trip_rel_err": rt_err, "round_trip_bound": tol},
        "clocks": clocks, "e2e": None,
        "gpu_launches": args.steps * (plan.launches(0) + plan.launches(1)),
        "roofline": {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": (stored_traffic("c2c:" + dom, n, "f32") or {}).get("dram_bytes_per_launch"),
                     "peak_source": peak_src,
                     "algorithmic_bytes": pass_b, "ms_per_launch": per_kernel[dom], "all_kernels_ms": per_kernel,
                     "array_passes_per_pair": len(per_kernel),
                     "pair_frac_of_pass_roofline": (len(per_kernel) * pass_b / peak / 1e9) / (ms_step * 1e-3),
                     "pair_frac_of_6pass_roofline": (6 * pass_b / peak / 1e9) / (ms_step * 1e-3)},
        "cpu_baseline": None,
    }
    print(json.dumps(line), flush=True)
    if not (rt_err <= tol):
        raise SystemExit("round trip error %.3e exceeds %.3e: the timed path is wrong" % (rt_err, tol))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--size", "--n", dest="n", type=int, default=1024)
    ap.add_argument("--slabs", type=int, default=0, help="virtual_slabs (0: the value BASELINE.json gives for the size)")
    ap.add_argument("--dist", action="store_true", help="run the slab-decomposed driver even with one rank")
    ap.add_argument("--exchange", default="auto", choices=["auto", "chunks", "unified"],
                    help="N > 1: stores straight into the peers' memory (VMM mapping; auto picks it where it can work), "
                         "or an all-to-all of chunks over NCCL; the other one's T_comm is reported beside the timed one's")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true",
                    help="default run only: skip the few pairs of 1536^3 / 2048^3 fp32 and 1024^3 fp64 reported in config.other_configs")
    ap.add_argument("--transform", default="r2c", choices=["r2c", "c2c"],
                    help="r2c (default): the headline R2C+C2R pair; c2c: the 3D C2C pair (single GPU, no e2e leg)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "cuda" and args.gpus != world:
        # never print an n_gpus = 1 line for an N-GPU request (or the reverse): the launcher decides the world size
        raise SystemExit("bench.py --gpus %d was started with WORLD_SIZE=%d: launch it as `python -m torch.distributed.run "
                         "--nnodes=1 --nproc-per-node %d --master-addr 127.0.0.1 --master-port P bench.py --gpus %d ...`"
                         % (args.gpus, world, args.gpus, args.gpus))
    if args.impl == "reference":
        run_reference(args)
    elif args.transform == "c2c":
        run_cuda_c2c(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
