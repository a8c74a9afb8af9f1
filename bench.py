#!/usr/bin/env python
"""bench.py -- throughput of the JANC per-step update (libjanc, sm_100a) in fp64 cell-updates/s.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--impl reference]

A "step" is one janc_step: cons->prim + reductions, ghost fill, 3 RK stages of LF-split WENO5 fluxes
with divergence, point-implicit chemistry (all SURVEY.md §8(a) rows) over the whole workload.
Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
"""
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

from paper_2504_13750_b200 import inputs as I  # noqa: E402

METRIC = "fp64 cell-updates/sec (RK3 step incl. point-implicit chemistry)"
UNIT = "cell-updates/s"

# algorithmic work / traffic per cell-update, derived in DESIGN.md "Roofline arithmetic"
WENO_OPS = 46            # DP instructions (FMA = 1, division = 1) of one WENO5-JS reconstruction


def flux_ops_per_cell_stage(ndim, nvar):
    # per component and direction: split (6) + 2 reconstructions + face sum/difference (4); RK update 3
    return nvar * (ndim * (6 + 2 * WENO_OPS + 4) + 3)


def flux_bytes_per_cell_stage(ndim, nvar):
    # read U^(k) (nvar) + p + u_d (ndim) + U^n (nvar, stages 2,3 -> counted always), write U^(k+1) (nvar)
    return (3 * nvar + 1 + ndim) * 8


def make_case(workload, rank=0):
    if workload == "cfg0":
        return I.config0(seed=1000 + 97 * rank)
    if workload == "cfg1":
        return I.config1(seed=1001 + 97 * rank)
    if workload == "cfg2":
        return I.config2(seed=1002 + 97 * rank)
    if workload == "cfg3":
        return I.config3(seed=1003 + 97 * rank)
    if workload == "cfg4":
        return I.config4(seed=1004 + 97 * rank)
    raise SystemExit(f"unknown workload {workload}")


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (profiling recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], False

    def run(self):
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                      "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
                self.rows.append([x.strip() for x in out.strip().split(",")])
            except Exception:
                pass
            time.sleep(0.1)

    def summary(self):
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i].lower() == "active"})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(self.rows)}


def oracle_throughput(case, budget_s=15.0):
    """The oracle as it stands, on a bounded sample of the workload (cropped IC), host cores."""
    from oracle import ref
    ref.build()
    g = case.grid
    if g.n_patches > 0 or g.ndim != 2:
        crop = case          # small / block cases: run as they are for a couple of steps
        desc = f"{case.name} (whole)"
    else:
        nx, ny = min(g.n[0], 512), min(g.n[1], 256)
        U = np.ascontiguousarray(case.U[:, :, :, :ny, :nx]); T = np.ascontiguousarray(case.T[:, :, :ny, :nx])
        crop = I.Case(case.name + "_crop", I.Grid(2, (nx, ny, 1), g.dx, g.bc_lo, g.bc_hi), case.mech, U, T, case.cfl, 1)
        desc = f"{case.name} cropped to {nx}x{ny} cells (columns 0..{nx - 1}, rows 0..{ny - 1})"
    s = ref.RefSolver(crop.grid, crop.mech, crop.blocks)
    s.set_state(crop.U, crop.T)
    cells = crop.cells
    t0 = time.perf_counter(); s.step(1, cfl=crop.cfl); t1 = time.perf_counter() - t0
    n = int(max(1, min(50, budget_s / max(t1, 1e-3))))
    t0 = time.perf_counter(); s.step(n, cfl=crop.cfl); tn = time.perf_counter() - t0
    s.close()
    return {"value": cells * n / tn, "unit": UNIT, "cores": ref.threads(), "kind": "oracle",
            "sample": f"{desc}, {n} steps after 1 warm-up, {tn:.1f} s"}, cells, tn / n
