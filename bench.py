#!/usr/bin/env python
"""bench.py -- headline measurement of the APD hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-solve]

A step is ONE pass of the whole hot path -- one apd_assign evaluation through the C ABI (seed pack ->
voxel x seed kernel with label store, histograms and dual partials -> finalize) -- on BASELINE.json's
headline workload: config 4, 256^3 voxels x 10,000 rolled-steel-like grains (synthetic, seeded).
Metric: G voxel-seed pairs/s.  One JSON line is printed by rank 0.

N > 1 (torchrun): the path does not shard in this build ("replicas only"): every rank runs
an independent replica of the workload on its own GPU; no data-path collective.  value = pairs of all
ranks / max-over-ranks device time.

--impl reference: the fp64 CPU oracle (oracle/) as it stands, on the host cores, on a bounded sample
of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2403_03571_b200 import workloads  # noqa: E402

WORKLOAD_CFG = 4
METRIC = "G voxel-seed pairs/s"
UNIT = "Gpairs/s"
FLUSH_BYTES = 256 << 20            # > 126 MB L2


def workload_name(wl):
    return (f"cfg{WORKLOAD_CFG}: {'x'.join(map(str, wl.n))} voxels x {wl.M} grains, rolled-steel-like ellipsoids, "
            f"one apd_assign evaluation (labels + volumes + dual) at w=0")


# ------------------------------------------------------------------------------------------------
# clocks sampled DURING the timed region (B200_PROFILING.md recipe)
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc, self.thread = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for (_, r) in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def max_over_ranks(x: float, world: int, device) -> float:
    """Replicas-only multi-GPU rule: every rank times its own replica, the job's time is the
    MAX over ranks.  `device` is where the one-element tensor lives (cuda:<local> under NCCL, cpu under gloo)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(pairs_per_rank: int, world: int, ms_per_step: float) -> float:
    """Whole-job G pairs/s: all ranks' pairs over the max-over-ranks time of a step."""
    return world * pairs_per_rank / (ms_per_step * 1e-3) / 1e9


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p))
        except Exception:
            return {}
    return {}


# ------------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline of the default run; the whole run for --impl reference)
# ------------------------------------------------------------------------------------------------
def oracle_sample_rate(wl, target_s: float, seed: int = 0):
    """Times oracle_assign (fp64, as it stands) on a sample of voxels of `wl` sized for ~target_s.
    Returns (pairs_per_s, cores, n_voxels, seconds)."""
    from oracle.apd_oracle import Grid, oracle_assign, num_threads
    grid = Grid(wl.dim, wl.n, wl.lo, wl.hi)
    cal = workloads.voxel_sample(wl.N, 4096, 900 + seed)
    t = time.perf_counter()
    oracle_assign(grid, wl.X, wl.A, wl.w0, sel=cal, diagnostics=False)
    dt = max(time.perf_counter() - t, 1e-4)
    n = int(min(wl.N, max(4096, len(cal) * target_s / dt)))
    sel = workloads.voxel_sample(wl.N, n, 901 + seed)
    t = time.perf_counter()
    oracle_assign(grid, wl.X, wl.A, wl.w0, sel=sel, diagnostics=False)
    dt = time.perf_counter() - t
    return len(sel) * wl.M / dt, num_threads(), len(sel), dt


def cpu_baseline(wl, target_s: float):
    rate, cores, nvox, dt = oracle_sample_rate(wl, target_s)
    return {"value": rate / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"oracle_assign (fp64, gcc -O2, OpenMP) on {nvox} seeded random voxels of the {wl.N} x all "
                      f"{wl.M} grains: {nvox * wl.M:.3e} pairs in {dt:.1f} s"}


def run_reference(args):
    """--impl reference: the oracle as it stands, on this box's host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    wl = workloads.make_config(WORKLOAD_CFG)
    per_step_s = args.ref_seconds if args.ref_seconds > 0 else max(2.0, min(20.0, 150.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_sample_rate(wl, per_step_s)
    t_pairs, t_s, cores, nvox = 0.0, 0.0, 0, 0
    for i in range(args.steps):
        rate, cores, nvox, dt = oracle_sample_rate(wl, per_step_s, seed=10 + i)
        t_pairs += nvox * wl.M
        t_s += dt
    value = t_pairs / t_s / 1e9
    sample = (f"each step = oracle_assign (fp64, OpenMP) on ~{nvox} seeded random voxels of {wl.N} x all {wl.M} "
              f"grains (~{per_step_s:.0f} s of CPU work)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_s / max(1, args.steps),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(wl), "sampled": True},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------
# Algorithmic FP32 work per voxel-seed pair of each kernel form:
#   DIRECT  : 3 FADD + 3 FMUL + 6 FFMA               = 18 flop   (12 FP32 instructions, 3D)
#   ROWPOLY : 1.5 FMA (voxels at +-tau share the even part) + 7 FMA set-up per (row of 32 voxels, seed)
#             = 3 + 14/32 = 3.4375 flop (the once-per-(tile, seed) re-expansion, ~25 flop / 4096 voxels, not counted)
#   TENSOR  : the K = 32 bf16 contraction of the lifted form = 64 tensor-core flop per pair (30 of the 32 K slots carry
#             a product); reported against the MEASURED bf16 peak, bound "tensor" -- its real limit is the CUDA-core
#             argmin epilogue
FLOP_PER_PAIR = {1: 18.0, 2: 3.0 + 14.0 / 32.0, 3: 64.0}
KERNEL_NAME = {1: "assign_direct_kernel<3>", 2: "assign_rowpoly_kernel<3>", 3: "assign_tensor_kernel"}
FP32_LANES_PER_SM = 128
# dram__bytes_read.sum + dram__bytes_write.sum of one assign_rowpoly_kernel launch on this workload, from the
# `ncu --set full` capture summarised in profiles/ (None until a capture exists)
NCU_TRAFFIC_BYTES = 489472 + 15261696      # profiles/r01_assign_rowpoly_full.md (labels mostly still in L2 at kernel end)


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2403_03571_b200 import binding as apd

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU path; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    apd.load_library()

    wl = workloads.make_config(WORKLOAD_CFG)
    ctx = apd.ApdContext(wl.dim, wl.M, device=local)
    grid = apd.make_grid(wl.dim, wl.n, wl.lo, wl.hi)
    X = torch.from_numpy(wl.X).to(dev); A = torch.from_numpy(wl.A).to(dev)
    v = torch.from_numpy(wl.v).to(dev); w = torch.zeros(wl.M, dtype=torch.float32, device=dev)
    labels = torch.empty(wl.N, dtype=torch.int32, device=dev)
    vol = torch.zeros(wl.M, dtype=torch.float64, device=dev)
    dual = torch.zeros(1, dtype=torch.float64, device=dev)
    err = torch.zeros(1, dtype=torch.float64, device=dev)
    flush = torch.empty(FLUSH_BYTES, dtype=torch.uint8, device=dev)
    opts = apd.make_opts(kernel=args.kernel)
    kernel_id = args.kernel if args.kernel else apd.KERNEL_ROWPOLY

    def step():
        ctx.apd_assign(grid, X, A, w, target_vol=v, labels=labels, vol=vol, dual=dual, max_rel_err=err, opts=opts)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        flush.zero_(); step()
    barrier()

    # ---- timed region: K steps, each bracketed by CUDA events on the launching stream; the L2 flush between
    #      steps sits outside the event pairs ----
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    t0 = time.time()
    for i in range(args.steps):
        flush.zero_()
        ev[i][0].record()
        step()
        ev[i][1].record()
        if i % 8 == 7 or i == args.steps - 1:
            torch.cuda.synchronize()
    barrier()
    t1 = time.time()
    clocks = sampler.stop(t0, t1)
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = float(sum(step_ms))

    # the dominant kernel alone (library-side CUDA events around the launch, same stream), K more launches
    k_ms = []
    for i in range(args.steps):
        flush.zero_(); step(); torch.cuda.synchronize()
        k_ms.append(ctx.last_kernel_ms())
    kernel_ms = float(np.mean(k_ms))

    total_ms = max_over_ranks(total_ms, world, dev)
    ms_per_step = total_ms / args.steps
    value = aggregate_value(wl.pairs, world, ms_per_step)

    # ---- e2e: the same evaluation through the HOST-buffer C-ABI call (pinned host tensors; H2D of the inputs,
    #      D2H of labels + volumes + dual inside the timed region) ----
    hX = torch.from_numpy(wl.X).pin_memory(); hA = torch.from_numpy(wl.A).pin_memory()
    hw = torch.zeros(wl.M, dtype=torch.float32).pin_memory(); hv = torch.from_numpy(wl.v).pin_memory()
    hlab = torch.empty(wl.N, dtype=torch.int32).pin_memory()
    hvol = torch.empty(wl.M, dtype=torch.float64).pin_memory()
    e2e_steps = max(3, min(args.steps, 10))
    for _ in range(2):
        ctx.apd_assign_host(grid, hX, hA, hw, target_vol=hv, labels=hlab, vol=hvol, opts=opts)
    barrier()
    e2e_each = []
    for _ in range(e2e_steps):
        te = time.perf_counter()
        ctx.apd_assign_host(grid, hX, hA, hw, target_vol=hv, labels=hlab, vol=hvol, opts=opts)   # synchronous
        e2e_each.append(time.perf_counter() - te)
    e2e_s = float(np.median(e2e_each))       # per-call wall times; the median shrugs off a host hiccup (max reported)
    e2e_s = max_over_ranks(e2e_s, world, dev)
    h2d = 4 * (hX.numel() + hA.numel() + hw.numel() + hv.numel())
    d2h = 4 * hlab.numel() + 8 * hvol.numel() + 16 + 8

    line = None
    if rank == 0:
        peaks = measured_peaks()
        sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
        sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
        peak_tflops = sm_count * FP32_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
        ach = FLOP_PER_PAIR[kernel_id] * wl.pairs / (kernel_ms * 1e-3) / 1e12
        bf16_peak = float(peaks.get("bf16_tflops", 1662.1))
        roofline = {"bound": "tensor" if kernel_id == 3 else "alu", "kernel": KERNEL_NAME[kernel_id],
                    "achieved": ach, "peak": bf16_peak if kernel_id == 3 else peak_tflops, "unit": "TFLOP/s",
                    "frac": ach / (bf16_peak if kernel_id == 3 else peak_tflops),
                    "traffic": NCU_TRAFFIC_BYTES if kernel_id == 2 else None, "kernel_ms": kernel_ms,
                    "flop_per_pair": FLOP_PER_PAIR[kernel_id],
                    "peak_is": ("MEASURED_PEAKS.json bf16_tflops (burst, cuBLAS 8192^3)" if kernel_id == 3 else
                                f"{sm_count} SMs x {FP32_LANES_PER_SM} FP32 lanes x 2 flop x {sm_max_mhz:.0f} MHz "
                                "(guide unit counts and MEASURED_PEAKS.json sm_max_mhz; no FP32 figure is measured there)"),
                    "label_write_GBps": 4.0 * wl.N / (kernel_ms * 1e-3) / 1e9}
        extra = {}
        if not args.no_probe:
            try:
                from paper_2403_03571_b200 import probe
                p0, mhz0 = probe.apd_fp32_probe(0, local)
                p1, _ = probe.apd_fp32_probe(1, local)
                p3, _ = probe.apd_fp32_probe(3, local)
                extra["fp32_probe"] = {"ffma_tflops": 2 * p0 / 1e12, "ffma2_tflops": 2 * p1 / 1e12,
                                       "rowpoly_mix_gpairs": p3 / 1e9, "sm_mhz": mhz0}
                roofline["frac_of_rowpoly_mix_probe"] = (wl.pairs / (kernel_ms * 1e-3)) / p3
            except Exception as e:  # the probe is context, never the headline
                extra["fp32_probe"] = {"error": str(e)}
        if not args.no_direct and kernel_id != 1:
            # the un-hoisted 12-instruction reference kernel north_star's ">= 60% of FP32 peak" is read against
            o1 = apd.make_opts(kernel=apd.KERNEL_DIRECT)
            d_ms = []
            for _ in range(3):
                flush.zero_()
                ctx.apd_assign(grid, X, A, w, target_vol=v, labels=labels, vol=vol, dual=dual, max_rel_err=err, opts=o1)
                torch.cuda.synchronize()
                d_ms.append(ctx.last_kernel_ms())
            dm = float(np.mean(d_ms[1:]))
            dach = FLOP_PER_PAIR[1] * wl.pairs / (dm * 1e-3) / 1e12
            extra["roofline_direct"] = {"bound": "alu", "kernel": "assign_direct_kernel<3>", "achieved": dach,
                                        "peak": peak_tflops, "unit": "TFLOP/s", "frac": dach / peak_tflops,
                                        "kernel_ms": dm, "gpairs": wl.pairs / (dm * 1e-3) / 1e9, "flop_per_pair": 18.0}
        if not args.no_direct and kernel_id != 3:
            # row a8: the tensor-core lift of the cost matrix (opts.kernel = APD_KERNEL_TENSOR), same workload
            o3 = apd.make_opts(kernel=apd.KERNEL_TENSOR)
            t_ms = []
            for _ in range(4):
                flush.zero_()
                ctx.apd_assign(grid, X, A, w, target_vol=v, labels=labels, vol=vol, dual=dual, max_rel_err=err, opts=o3)
                torch.cuda.synchronize()
                t_ms.append(ctx.last_kernel_ms())
            tm = float(np.mean(t_ms[1:]))
            tach = FLOP_PER_PAIR[3] * wl.pairs / (tm * 1e-3) / 1e12
            extra["roofline_tensor"] = {"bound": "tensor", "kernel": "assign_tensor_kernel", "achieved": tach,
                                        "peak": bf16_peak, "unit": "TFLOP/s", "frac": tach / bf16_peak, "kernel_ms": tm,
                                        "gpairs": wl.pairs / (tm * 1e-3) / 1e9, "flop_per_pair": 64.0,
                                        "peak_is": "MEASURED_PEAKS.json bf16_tflops (burst, cuBLAS 8192^3)",
                                        "note": "K = 32 contraction per pair; paced by its CUDA-core argmin epilogue (one "
                                                "3-input min per 2 pairs on the half-rate ALU pipe) and by the per-M-tile "
                                                "accumulator ring, not by the tensor pipe (DESIGN.md 9)"}
        if not args.no_solve:
            pairs_t = torch.zeros(1, dtype=torch.int64, device=dev)
            oc = apd.make_opts(kernel=args.kernel, cull=1)
            c_ms = []
            for _ in range(5):
                flush.zero_()
                e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                e0.record()
                ctx.apd_assign(grid, X, A, w, target_vol=v, labels=labels, vol=vol, dual=dual, max_rel_err=err,
                               pairs_evaluated=pairs_t, opts=oc)
                e1.record(); torch.cuda.synchronize()
                c_ms.append(e0.elapsed_time(e1))
            cm = float(np.mean(c_ms[2:]))
            extra["culled_assign"] = {"workload": f"cfg{WORKLOAD_CFG}, opts.cull=1 (exact tile culling, labels identical)",
                                      "ms_per_step": cm, "pairs_evaluated": int(pairs_t.item()),
                                      "pruned_fraction": 1.0 - pairs_t.item() / wl.pairs,
                                      "effective_gpairs": wl.pairs / (cm * 1e-3) / 1e9}

            def solve_leg(ctx_, grid_, X_, A_, v_, wl_, labels_, vol_, cull):
                secs = []
                for _ in range(2 if cull else 1):    # culled: the first call also allocates the workspace (cold)
                    wS = torch.zeros(wl_.M, dtype=torch.float32, device=dev)
                    torch.cuda.synchronize()
                    ts = time.perf_counter()
                    info = ctx_.apd_solve(grid_, X_, A_, v_, wl_.eps, w=wS, labels=labels_, vol=vol_,
                                          opts=apd.make_opts(kernel=args.kernel, cull=cull, max_iters=args.solve_max_iters))
                    torch.cuda.synchronize()
                    secs.append(time.perf_counter() - ts)
                return {"seconds": secs[-1], "first_call_seconds": secs[0], "tol": wl_.eps, "cull": cull,
                        "status": info.status, "iters": info.iters, "evals": info.evals,
                        "max_rel_err": info.max_rel_err, "dual": info.dual}

            extra["solve"] = dict(workload=f"cfg{WORKLOAD_CFG} apd_solve", **solve_leg(ctx, grid, X, A, v, wl, labels, vol, 1))
            extra["solve_brute_force"] = dict(workload=f"cfg{WORKLOAD_CFG} apd_solve",
                                              **solve_leg(ctx, grid, X, A, v, wl, labels, vol, 0))
            if not args.no_cfg5:
                wl5 = workloads.make_config(5)
                ctx5 = apd.ApdContext(wl5.dim, wl5.M, device=local)
                grid5 = apd.make_grid(wl5.dim, wl5.n, wl5.lo, wl5.hi)
                X5 = torch.from_numpy(wl5.X).to(dev); A5 = torch.from_numpy(wl5.A).to(dev)
                v5 = torch.from_numpy(wl5.v).to(dev)
                lab5 = torch.empty(wl5.N, dtype=torch.int32, device=dev)
                vol5 = torch.zeros(wl5.M, dtype=torch.float64, device=dev)
                extra["solve_cfg5"] = dict(workload=f"cfg5 apd_solve: {'x'.join(map(str, wl5.n))} voxels x {wl5.M} grains",
                                           **solve_leg(ctx5, grid5, X5, A5, v5, wl5, lab5, vol5, 1))
                w5 = torch.zeros(wl5.M, dtype=torch.float32, device=dev)
                ctx5.apd_assign(grid5, X5, A5, w5, target_vol=v5, labels=lab5, vol=vol5, dual=dual, max_rel_err=err,
                                pairs_evaluated=pairs_t, opts=oc)
                torch.cuda.synchronize()
                extra["solve_cfg5"]["pruned_fraction_at_w0"] = 1.0 - pairs_t.item() / wl5.pairs
                del lab5
        cb = None
        if world == 1 and not args.no_cpu:
            cb = cpu_baseline(wl, args.cpu_seconds)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": workload_name(wl), "l2": f"flushed between steps ({FLUSH_BYTES >> 20} MiB write)",
                           "multi_gpu": "replicas only (no data-path collective)", "kernel": kernel_id},
                "clocks": clocks, "roofline": roofline, "cpu_baseline": cb,
                "e2e": {"value": world * wl.pairs / e2e_s / 1e9, "unit": UNIT, "h2d_bytes_per_step": h2d,
                        "d2h_bytes_per_step": d2h, "ms_per_step": e2e_s * 1e3, "ms_per_step_max": max(e2e_each) * 1e3,
                        "steps": e2e_steps,
                        "call": "apd_assign_host (pinned host buffers; H2D/D2H copies inside, device scratch kept by the context)"},
                "gpu_launches": (4 if kernel_id == 3 else 3) * args.steps,
                "launches_per_step": {1: ["pack_seeds_kernel", "assign_direct_kernel", "finalize_kernel"],
                                      2: ["pack_pairs_kernel", "assign_rowpoly_kernel", "finalize_kernel"],
                                      3: ["pack_seeds_kernel", "pack_qfix_kernel", "assign_tensor_kernel",
                                          "finalize_kernel"]}[kernel_id]}
        line.update(extra)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if line is not None:
        print(json.dumps(line), flush=True)


def run_solve_only(args):
    """--solve-only: one apd_solve of the headline workload with culling (the time-to-solve leg alone; this is the
    command the ncu launch list under profiles/ is taken from).  Prints one JSON line."""
    import torch
    from paper_2403_03571_b200 import binding as apd
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    wl = workloads.make_config(WORKLOAD_CFG)
    ctx = apd.ApdContext(wl.dim, wl.M, device=dev.index)
    grid = apd.make_grid(wl.dim, wl.n, wl.lo, wl.hi)
    X = torch.from_numpy(wl.X).to(dev); A = torch.from_numpy(wl.A).to(dev); v = torch.from_numpy(wl.v).to(dev)
    labels = torch.empty(wl.N, dtype=torch.int32, device=dev)
    vol = torch.zeros(wl.M, dtype=torch.float64, device=dev)
    out = None
    for _ in range(max(1, args.warmup) + 1):
        wS = torch.zeros(wl.M, dtype=torch.float32, device=dev)
        torch.cuda.synchronize()
        ts = time.perf_counter()
        info = ctx.apd_solve(grid, X, A, v, wl.eps, w=wS, labels=labels, vol=vol,
                             opts=apd.make_opts(cull=1, max_iters=args.solve_max_iters))
        torch.cuda.synchronize()
        out = {"metric": "APD time-to-solve at 1% vol tol", "value": time.perf_counter() - ts, "unit": "s",
               "higher_is_better": False, "workload": f"cfg{WORKLOAD_CFG} apd_solve, opts.cull=1", "status": info.status,
               "iters": info.iters, "evals": info.evals, "max_rel_err": info.max_rel_err,
               "cull_rebuilds": ctx.solve_stats()[1]}
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--kernel", type=int, default=0, help="0 auto, 1 DIRECT, 2 ROWPOLY, 3 TENSOR")
    ap.add_argument("--no-solve", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-probe", action="store_true")
    ap.add_argument("--no-direct", action="store_true")
    ap.add_argument("--no-cfg5", action="store_true")
    ap.add_argument("--solve-only", action="store_true", help="only the culled apd_solve of the headline workload")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--solve-max-iters", type=int, default=1000)
    ap.add_argument("--ref-seconds", type=float, default=0.0, help="--impl reference: CPU seconds per step (0 = auto)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.solve_only:
        run_solve_only(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
