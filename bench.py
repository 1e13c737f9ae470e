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
