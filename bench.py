#!/usr/bin/env python
"""bench.py -- GLUPS of the two-component Shan-Chen D3Q19 step on B200, against the HBM roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config2|config1|...|all]
                    [--tau-r T --tau-b T --G g]   # general-tau variant of the same workload
    python bench.py --impl reference ...        # the CPU oracle, as it stands, on host cores

`--workload all` prints one JSON line per BASELINE config (0-4), each at the config's own dtype.

One "step" is one pass of the whole hot path (moments, force, collide, bounce-back, stream)
over the whole box: one lb_step(1).  `value` is GLUPS = N_nodes * K / t / 1e9 (PAPER.md:166-171
Eq. 4) with the state resident in HBM, timed with CUDA events on the stream the kernels are
launched on.  `e2e` is the same metric through the C ABI with HOST buffers: lb_set_fields
(H2D) + lb_step(K) + lb_get_moments (D2H) inside one timed region.

The path does not shard (north_star: one GPU, no inter-GPU traffic): --gpus N runs N
independent replicas, one process per GPU, barrier + max-over-ranks timing ("replicas only",
DESIGN.md §Multi-GPU).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2112_08264_b200 import workloads as W  # noqa: E402

METRIC = "GLUPS (fp64 two-component D3Q19) on 1 B200; achieved HBM GB/s vs peak"
WORKLOADS = {f"config{i}": c for i, c in enumerate(W.CONFIGS)}
ALG_BYTES = {"f64": 608, "f32": 304}     # populations read + written per node per step


# ---------------------------------------------------------------------------------------------
# helpers
# ---------------------------------------------------------------------------------------------
def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def aggregate_over_ranks(ms_local: float, units_local: float, world: int, device=None):
    """(max time over ranks, total units over ranks).  Works on any torch.distributed backend."""
    if world == 1:
        return ms_local, units_local
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    u = torch.tensor([units_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={gpu_index}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            pass

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
            out, _ = self.p.communicate()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in out.splitlines():
            c = [v.strip() for v in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])), mx.append(float(c[2]))
            except ValueError:
                continue
            for nm, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def committed_traffic(workload: str, kernel: str):
    """(dram bytes per launch, where from) of the dominant kernel from the committed ncu capture
    (profiles/traffic.csv; the LAST matching row = the newest capture), if any."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    found = (None, None)
    if not os.path.exists(p):
        return found
    try:
        import csv
        for row in csv.DictReader(open(p)):
            if row["workload"] == workload and row["kernel"] == kernel:
                found = (float(row["dram_bytes_per_launch"]), row.get("source", "profiles/traffic.csv"))
    except (ValueError, OSError, KeyError):
        pass
    return found


def cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def with_overrides(cfg, args):
    """The workload with --tau-r / --tau-b / --G replaced (the general-tau bench variants of SURVEY 8(d) 'rules')."""
    import dataclasses
    kw = {}
    if getattr(args, "f32", False) and cfg.dtype != "f32":
        kw["dtype"] = "f32"
        kw["name"] = cfg.name.replace("f64", "f32")
    if args.tau_r is not None:
        kw["tau_r"] = args.tau_r
    if args.tau_b is not None:
        kw["tau_b"] = args.tau_b
    if args.G is not None:
        kw["G"] = args.G
    return dataclasses.replace(cfg, **kw) if kw else cfg


def time_oracle(cfg, sub, steps, warmup=0):
    """The oracle, as it stands, single-threaded on a periodic sub-box of the workload's fields."""
    from oracle import ora
    sx, sy, sz = sub
    rr, rb = W.mixture_fields(cfg.nx, cfg.ny, cfg.nz, cfg.seed, chunk=1 << 22) if cfg.n_nodes <= (1 << 24) else (None, None)
    if rr is None:      # 512^3: generate only the slab we need (same counters, same values)
        n = np.arange(sz * cfg.ny * cfg.nx, dtype=np.uint64)
        rr = 1.0 + 0.01 * (2.0 * W.u01(cfg.seed, np.uint64(2) * n) - 1.0)
        rb = 1.0 + 0.01 * (2.0 * W.u01(cfg.seed, np.uint64(2) * n + np.uint64(1)) - 1.0)
        rr = rr.reshape(sz, cfg.ny, cfg.nx)[:, :sy, :sx]
        rb = rb.reshape(sz, cfg.ny, cfg.nx)[:, :sy, :sx]
    else:
        rr = rr.reshape(cfg.nz, cfg.ny, cfg.nx)[:sz, :sy, :sx]
        rb = rb.reshape(cfg.nz, cfg.ny, cfg.nx)[:sz, :sy, :sx]
    o = ora.Oracle(sx, sy, sz, cfg.tau_r, cfg.tau_b, cfg.G)
    if cfg.n_spheres:
        o.set_solid_mask(cfg.solid_mask().reshape(cfg.nz, cfg.ny, cfg.nx)[:sz, :sy, :sx])
    o.set_fields(np.ascontiguousarray(rr), np.ascontiguousarray(rb))
    if warmup:
        o.step(warmup)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    return sx * sy * sz * steps / dt / 1e9, dt


# ---------------------------------------------------------------------------------------------
# reference arm: the CPU oracle
# ---------------------------------------------------------------------------------------------
def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    cfg = with_overrides(WORKLOADS["config2" if args.workload == "all" or args.workload in SINGLE else args.workload], args)
    sub = (min(cfg.nx, 64), min(cfg.ny, 32), min(cfg.nz, 32))
    glups, dt = time_oracle(cfg, sub, args.steps, args.warmup)
    sample = (f"periodic {sub[0]}x{sub[1]}x{sub[2]} corner of {cfg.name}'s seeded fields, "
              f"{args.steps} steps after {args.warmup} warm-up")
    line = {
        "impl": "reference", "metric": METRIC, "value": glups, "unit": "GLUPS", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "box": [cfg.nx, cfg.ny, cfg.nz], "tau": [cfg.tau_r, cfg.tau_b], "G": cfg.G,
                   "note": "CPU oracle (oracle/lb_oracle.cpp, g++ -O2 -ffp-contract=off) on a bounded sample"},
        "cpu_baseline": {"value": glups, "unit": "GLUPS", "cores": 1, "kind": "oracle", "sample": sample, "cpu": cpu_model()},
        "e2e": {"value": glups, "unit": "GLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    from paper_2112_08264_b200 import binding as B
    from paper_2112_08264_b200.build import build_lib

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; this library has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    if rank == 0:
        build_lib()
    if world > 1:
        dist.barrier()
    B.lib()
    names = sorted(WORKLOADS) + sorted(SINGLE) if args.workload == "all" else [args.workload]
    for i, name in enumerate(names):
        if name in SINGLE:
            run_single(args, name, B, torch, dev, rank, local_rank, world)
            continue
        if args.decomposition == "slab":
            run_slab(args, with_overrides(WORKLOADS[name], args), B, torch, dev, rank, local_rank, world)
            continue
        # `all`: the CPU oracle is timed once (on the headline workload), not five times
        cpu = not args.no_cpu_baseline and (args.workload != "all" or name == "config2")
        run_one(args, with_overrides(WORKLOADS[name], args), B, torch, dev, rank, local_rank, world, cpu)
    import torch.distributed as dist_
    if dist_.is_initialized():
        dist_.destroy_process_group()
    return 0


SINGLE = {"single128_f32": (128, "f32"), "single256_f32": (256, "f32"), "single256_f64": (256, "f64"), "single512_f32": (512, "f32")}


def run_single(args, name, B, torch, dev, rank, local_rank, world):
    """The single-fluid calibration workload (the paper's case 1, Table 1):
    one BGK fluid, fused collide + stream, 304 / 152 algorithmic bytes per node.  rho = 1 + 1 % seeded noise, u = 0."""
    n, dt = SINGLE[name]
    N = n * n * n
    tau = args.tau_r if args.tau_r is not None else 1.0
    steps, warmup = args.steps, max(args.warmup, 3)
    rho, _ = W.mixture_fields(n, n, n, 2112082645)
    pin = torch.empty(N, dtype=torch.float64).pin_memory()
    pin.numpy()[:] = rho
    out = torch.empty(N, dtype=torch.float64).pin_memory()
    stream = torch.cuda.Stream(device=dev)
    box = B.SingleBox(n, n, n, tau, dtype=B.LB_F64 if dt == "f64" else B.LB_F32, cuda_stream=stream.cuda_stream)
    box.set_fields(pin.numpy())
    box.step(warmup)
    box.sync()
    torch.cuda.synchronize(dev)
    sampler = ClockSampler(local_rank)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = box.launch_count()
    e0.record(stream)
    box.step(steps)
    e1.record(stream)
    e1.synchronize()
    launches = box.launch_count() - l0
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    ms_max, units = aggregate_over_ranks(ms, float(N) * steps, world, dev)
    glups = units / (ms_max * 1e-3) / 1e9
    t0 = time.perf_counter()
    box.set_fields(pin.numpy())
    box.step(steps)
    B._chk(B.lib().lbs_get_moments(box.h, B._d(out.numpy()), None, None, None))
    e2e_s = time.perf_counter() - t0
    box.close()
    if rank != 0:
        return
    peak, peak_src = measured_peak()
    alg = ALG_BYTES[dt] // 2
    achieved = alg * N / (ms / steps * 1e-3) / 1e9
    es = 8 if dt == "f64" else 4
    line = {
        "metric": "GLUPS (single-fluid D3Q19 BGK, fused collide + stream) on 1 B200; achieved HBM GB/s vs peak", "value": glups, "unit": "GLUPS",
        "n_gpus": world, "steps": steps, "warmup": warmup, "ms_per_step": ms_max / steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": dt, "data": "synthetic",
        "config": {"workload": name, "box": [n, n, n], "tau": [tau], "kernel": "single", "launches_per_step": launches / steps,
                   "l2": f"state {2 * 19 * N * es / 2**30:.1f} GiB vs 126 MB L2",
                   "context": "paper Table 1 (PAPER.md:175-194): 2.011 GLUPS fused at 256^3 fp32 on 1 V100; 3.406 quoted as state of the art (PAPER.md:192)"},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                     "peak_source": peak_src, "algorithmic_bytes_per_node": alg, "kernel_ms": ms / steps, "kernel": "k_single_step"},
        "e2e": {"value": N * steps / e2e_s / 1e9, "unit": "GLUPS", "h2d_bytes_per_step": N * 8 / steps, "d2h_bytes_per_step": N * 8 / steps,
                "seconds": e2e_s, "calls": "lbs_set_fields(host) + lbs_step(K) + lbs_get_moments(host rho)"},
        "gpu_launches": launches, "clocks": clocks,
    }
    print(json.dumps(line), flush=True)


def run_slab(args, cfg, B, torch, dev, rank, local_rank, world):
    """--decomposition slab: ONE global box split into z slabs, one per rank, two ghost planes exchanged with the ring
    neighbours before every step over torch.distributed (NCCL / NVLink): strong scaling.  General two-pass kernels."""
    from paper_2112_08264_b200 import slab as S
    import torch.distributed as dist
    if world == 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1"); os.environ.setdefault("MASTER_PORT", "29531")
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=dev)
    dtype = B.LB_F64 if cfg.dtype == "f64" else B.LB_F32
    stream = torch.cuda.current_stream(dev)
    kernel = {"auto": None, "twopass": B.LB_KERNEL_TWOPASS, "onepass": B.LB_KERNEL_ONEPASS, "tma": B.LB_KERNEL_TMA, "halo": B.LB_KERNEL_HALO, "node": B.LB_KERNEL_NODE}[args.kernel]
    sl = S.SlabBox(cfg.nx, cfg.ny, cfg.nz, rank, world, cfg.tau_r, cfg.tau_b, cfg.G, dtype=dtype, cuda_stream=stream.cuda_stream, device=dev, kernel=kernel)
    rr, rb = cfg.fields()
    sl.set_fields(rr, rb)
    del rr, rb
    steps, warmup = args.steps, max(args.warmup, 3)

    def advance(k):
        for _ in range(k):
            S.ring_exchange_dist(sl, dist)
            sl.step(1)
    advance(warmup)
    torch.cuda.synchronize(dev)
    dist.barrier()
    sampler = ClockSampler(local_rank)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = sl.box.launch_count()
    e0.record(stream)
    advance(steps)
    e1.record(stream)
    e1.synchronize()
    torch.cuda.synchronize(dev)
    dist.barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    launches = sl.box.launch_count() - l0
    ms_max, _ = aggregate_over_ranks(ms, 0.0, world, dev)
    N = cfg.n_nodes
    glups = N * steps / (ms_max * 1e-3) / 1e9
    kname = B.lb_kernel_name(sl.box.h)
    halo = 4 * sl.box.plane_buffer_bytes(S.GHOST)
    sl.close()
    if rank != 0:
        return
    es = 8 if cfg.dtype == "f64" else 4

    peak, peak_src = measured_peak()
    alg = ALG_BYTES[cfg.dtype]
    achieved = alg * N / world / (ms / steps * 1e-3) / 1e9
    print(json.dumps({
        "metric": METRIC, "value": glups, "unit": "GLUPS", "n_gpus": world, "steps": steps, "warmup": warmup, "ms_per_step": ms_max / steps,
        "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": cfg.dtype, "data": "synthetic",
        "config": {"workload": cfg.name, "box": [cfg.nx, cfg.ny, cfg.nz], "tau": [cfg.tau_r, cfg.tau_b], "G": cfg.G, "kernel": kname,
                   "parallelism": f"z slabs x{world}, {S.GHOST} ghost planes per side exchanged every step (torch.distributed P2P)",
                   "halo_bytes_per_rank_per_step": halo, "launches_per_step": launches / steps},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                     "peak_source": peak_src, "algorithmic_bytes_per_node": alg, "kernel_ms": ms / steps, "kernel": "whole step of one rank"},
        "e2e": {"value": None, "unit": "GLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0, "note": "not measured in slab mode"},
        "gpu_launches": launches, "clocks": clocks}), flush=True)


def run_one(args, cfg, B, torch, dev, rank, local_rank, world, cpu_baseline):
    if world > 1:
        import torch.distributed as dist
    note = None
    es = 8 if cfg.dtype == "f64" else 4
    need = (2 * 38 + 8) * cfg.n_nodes * es + 4 * cfg.n_nodes + (1 << 30)     # populations, carried density, links, staging
    free, _total = torch.cuda.mem_get_info(dev)
    if need > free and cfg.n_nodes > (1 << 24):
        note = f"{cfg.name} needs {need >> 30} GiB, {free >> 30} GiB free: fell back to config1"
        cfg = with_overrides(WORKLOADS["config1"], args)
    N = cfg.n_nodes
    steps, warmup = args.steps, max(args.warmup, 3)
    dtype = B.LB_F64 if cfg.dtype == "f64" else B.LB_F32

    # inputs: seeded, synthetic, in PINNED host memory (the e2e leg copies from / to these)
    rr_np, rb_np = cfg.fields()
    pin = [torch.empty(N, dtype=torch.float64).pin_memory() for _ in range(7)]
    rr, rb = pin[0].numpy(), pin[1].numpy()
    rr[:], rb[:] = rr_np, rb_np
    del rr_np, rb_np
    outs = [p.numpy() for p in pin[2:7]]
    mask = cfg.solid_mask()

    stream = torch.cuda.Stream(device=dev)
    box = B.Box(cfg.nx, cfg.ny, cfg.nz, cfg.tau_r, cfg.tau_b, cfg.G, dtype=dtype, cuda_stream=stream.cuda_stream)
    kernel = {"auto": B.LB_KERNEL_AUTO, "twopass": B.LB_KERNEL_TWOPASS, "onepass": B.LB_KERNEL_ONEPASS, "tma": B.LB_KERNEL_TMA, "halo": B.LB_KERNEL_HALO, "node": B.LB_KERNEL_NODE}[args.kernel]
    box.set_kernel(kernel)
    if args.diag:
        box.set_option(B.LB_OPT_DIAG, 1)
    if args.zc:
        box.set_option(B.LB_OPT_ZC, args.zc)
    if args.no_balance:
        box.set_option(B.LB_OPT_BALANCE, 0)
    if args.model == "cg":                       # the paper's own two-fluid operator, general two-pass path
        box.set_colour_gradient(args.sigma, args.beta)
    if mask is not None and args.moving_walls:   # prescribed sphere velocities + force / torque per sphere (N2), same path
        centres, _ = W.sphere_centres(cfg.nx, cfg.ny, cfg.nz, cfg.sphere_seed, cfg.n_spheres)
        vel = 0.01 * (2.0 * W.u01(cfg.sphere_seed + 1, np.arange(3 * cfg.n_spheres)) - 1.0)
        omg = 0.002 * (2.0 * W.u01(cfg.sphere_seed + 2, np.arange(3 * cfg.n_spheres)) - 1.0)
        box.set_spheres(centres, 5.5, vel, omg)
    elif mask is not None:
        box.set_solid_mask(mask)
    box.set_fields(rr, rb)
    kname = B.lb_kernel_name(box.h)

    # ---- device-resident timing: K steps between two events on the launching stream ----
    box.step(warmup)
    box.sync()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize(dev)
    sampler = ClockSampler(local_rank)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = box.launch_count()
    e0.record(stream)
    box.step(steps)
    e1.record(stream)
    e1.synchronize()
    torch.cuda.synchronize(dev)
    if world > 1:
        dist.barrier()
    launches = box.launch_count() - l0
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    ms_max, units = aggregate_over_ranks(ms, float(N) * steps, world, dev)
    glups = units / (ms_max * 1e-3) / 1e9
    diag = None
    if args.diag:
        m, p = box.get_diagnostics()            # the sums the last step left behind: no population pass
        diag = {"mass": [float(v) for v in m], "momentum": [float(v) for v in p]}
    fused = None
    if not args.diag and mask is None and args.model == "sc" and kname in ("tma", "halo", "node"):
        # the same K steps once more with the per-step diagnostics fused into the step kernel (LB_OPT_DIAG), for the record
        box.set_option(B.LB_OPT_DIAG, 1)
        box.step(3)
        box.sync()
        d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        d0.record(stream)
        box.step(steps)
        d1.record(stream)
        d1.synchronize()
        lq = box.launch_count()
        m, p = box.get_diagnostics()
        fused = {"ms_per_step": d0.elapsed_time(d1) / steps, "relative_to_plain": d0.elapsed_time(d1) / ms,
                 "launches_of_lb_get_diagnostics": box.launch_count() - lq,
                 "mass": [float(v) for v in m], "momentum": [float(v) for v in p]}
        box.set_option(B.LB_OPT_DIAG, 0)

    # ---- end to end through the C ABI with host buffers ----
    box.sync()
    if world > 1:
        dist.barrier()
    t0 = time.perf_counter()
    box.set_fields(rr, rb)                      # H2D: 2 fields of N doubles
    box.step(steps)
    B.lb_get_moments(box.h, N, outs)            # D2H: 5 fields of N doubles (synchronises)
    e2e_s = time.perf_counter() - t0
    e2e_ms_max, _ = aggregate_over_ranks(e2e_s * 1e3, 0.0, world, dev)
    e2e_glups = units / (e2e_ms_max * 1e-3) / 1e9
    mass_chk = float(outs[0].sum() + outs[1].sum())
    n_fluid = N if mask is None else int(N - int(mask.sum()))

    if rank != 0:
        box.close()
        return

    peak, peak_src = measured_peak()
    alg = ALG_BYTES[cfg.dtype]
    per_launch_ms = ms / max(launches, 1) * (launches / steps)      # = ms / steps: whole step (1 kernel on the one-pass path)
    achieved = alg * N / (per_launch_ms * 1e-3) / 1e9
    # captures are per workload, operator and kernel; a run with other options (moving walls, fused sums, an explicit chunk length)
    # has no capture of its own
    plain = not args.moving_walls and not args.diag and not args.zc
    traffic, traffic_src = committed_traffic(cfg.name + ("_cg" if args.model == "cg" else ""), kname) if plain else (None, None)
    line = {
        "metric": METRIC, "value": glups, "unit": "GLUPS", "n_gpus": world, "steps": steps, "warmup": warmup,
        "ms_per_step": ms_max / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": cfg.dtype, "data": "synthetic",
        "config": {"workload": cfg.name, "box": [cfg.nx, cfg.ny, cfg.nz], "tau": [cfg.tau_r, cfg.tau_b], "G": cfg.G,
                   "solid_spheres": cfg.n_spheres, "kernel": kname, "launches_per_step": launches / steps,
                   "planes_per_cta": box.get_option(B.LB_OPT_ZC),
                   "l2": f"state {2 * 38 * N * es / 2**30:.1f} GiB vs 126 MB L2" + (", no flush needed" if 2 * 38 * N * es > (1 << 30) else ": L2-resident, launch-bound, reported only"),
                   "parallelism": "replicas only" if world > 1 else "single GPU", "diagnostics_in_step": bool(args.diag),
                   "operator": "colour gradient (sigma %g, beta %g)" % (args.sigma, args.beta) if args.model == "cg" else "Shan-Chen",
                   "moving_walls": bool(mask is not None and args.moving_walls),
                   "whole_waves": bool(box.get_option(B.LB_OPT_BALANCE)) and not args.zc,
                   **({"note": note} if note else {})},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                     "algorithmic_bytes_per_node": alg, "kernel_ms": per_launch_ms,
                     "kernel": "whole step" if launches != steps else "fused one-pass step kernel"},
        "e2e": {"value": e2e_glups, "unit": "GLUPS", "h2d_bytes_per_step": 2 * N * 8 / steps,
                "d2h_bytes_per_step": 5 * N * 8 / steps, "seconds": e2e_s, "mass_check": mass_chk,
                "calls": "lb_set_fields(host) + lb_step(K) + lb_get_moments(host)"},
        "gpu_launches": launches, "clocks": clocks,
    }
    if mask is not None:
        line["config"]["fluid_nodes"] = n_fluid
        line["config"]["glups_fluid_nodes_only"] = glups * n_fluid / N      # no computation inside a particle
    if diag:
        line["diagnostics"] = diag
    if fused:
        line["diagnostics_fused_run"] = fused
    if cpu_baseline:
        sub = (min(cfg.nx, 128), min(cfg.ny, 128), min(cfg.nz, 64))
        cpu_steps = 12
        cg, cdt = time_oracle(cfg, sub, cpu_steps)
        c0 = WORKLOADS["config0"]
        cg0, cdt0 = time_oracle(c0, (c0.nx, c0.ny, c0.nz), 100)        # 32^3 x 100 steps
        line["cpu_baseline"] = {"value": cg, "unit": "GLUPS", "cores": 1, "kind": "oracle", "seconds": cdt, "cpu": cpu_model(),
                                "sample": f"periodic {sub[0]}x{sub[1]}x{sub[2]} corner of {cfg.name}'s seeded fields, {cpu_steps} steps",
                                "config0_32c_100_steps": {"value": cg0, "unit": "GLUPS", "seconds": cdt0}}
    box.close()
    del pin, outs, rr, rb
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config2", choices=sorted(WORKLOADS) + sorted(SINGLE) + ["all"])
    ap.add_argument("--tau-r", type=float, default=None, help="override the workload's tau_r (general-tau variant)")
    ap.add_argument("--tau-b", type=float, default=None)
    ap.add_argument("--G", type=float, default=None)
    ap.add_argument("--model", default="sc", choices=["sc", "cg"], help="collision operator: Shan-Chen (north_star) or colour gradient (PAPER.md:328-400)")
    ap.add_argument("--sigma", type=float, default=0.02)
    ap.add_argument("--beta", type=float, default=0.7)
    ap.add_argument("--moving-walls", action="store_true", help="config4: spheres with seeded velocities, force / torque per sphere each step")
    ap.add_argument("--f32", action="store_true", help="run the workload in fp32 (e.g. config1 --f32 --model cg: the paper's Table 2 setting)")
    ap.add_argument("--decomposition", default="replicas", choices=["replicas", "slab"],
                    help="--gpus N: N independent replicas (north_star: the path does not shard) or ONE box in N z slabs with halo exchange (N3)")
    ap.add_argument("--no-balance", action="store_true", help="LB_OPT_BALANCE = 0: no padding of the CTA count to whole waves (A/B)")
    ap.add_argument("--zc", type=int, default=0, help="planes per CTA of the one-pass kernels (LB_OPT_ZC); 0 = the library's heuristic")
    ap.add_argument("--diag", action="store_true", help="per-step mass / momentum sums fused into the step kernel (LB_OPT_DIAG)")
    ap.add_argument("--kernel", default="auto", choices=["auto", "twopass", "onepass", "tma", "halo", "node"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
