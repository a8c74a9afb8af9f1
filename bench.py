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
WENO_OPS = 25            # DP instructions (FMA = 1) of one WENO5-JS reconstruction in difference form
                         # (flux.cuh: differences 4 amortised, betas 6, squares 3, candidates 3,
                         #  weights + numerator + denominator 9)


def flux_ops_per_cell_stage(ndim, nvar):
    # per component and direction: split flux 2f+- (3) + 2 reconstructions + face value from the two over one
    # reciprocal (10) + difference, scale (2); RK update 3.  Pencil-end faces and ghost-row split fluxes (the kernel's redundancy)
    # are NOT counted.
    return nvar * (ndim * (3 + 2 * WENO_OPS + 10 + 2) + 3)


def chem_ops_per_cell(mech):
    """Algorithmic DP instructions (FMA = 1) of the point-implicit update of one cell, counted from the mechanism
    (DESIGN.md section 6): 3 Newton iterations on e(T); per reaction 2 exponentials (23 each) + Arrhenius arguments,
    concentration products and the net rate (12); one multiply per non-zero dq_i/dX_j and one add per non-zero
    contribution to D_kj (third-body reactions touch every column); I - dt J (2 per entry); elimination n^3/3 and
    the two triangular solves n^2."""
    import numpy as np
    ns, nr, n1 = mech.ns, mech.nr, mech.ns - 1
    nu_f, nu_b = np.asarray(mech.nu_f), np.asarray(mech.nu_b)
    tb = np.asarray(mech.third_body).astype(bool) if mech.third_body is not None else np.zeros(nr, bool)
    deg = max([q for q in range(5) if np.any(np.asarray(mech.nasa)[:, q] != 0.0)] + [0])
    newton = 3 * ns * (2 * deg + 3)
    rates = nr * (2 * 23 + 12)
    entries = updates = 0
    for i in range(nr):
        rows = int(np.count_nonzero((nu_b[i] - nu_f[i])[:n1]))
        cols = ns if tb[i] else int(np.count_nonzero(nu_f[i] + nu_b[i]))
        entries += cols
        updates += rows * cols
    return newton + rates + entries + updates + 2 * n1 * n1 + n1 ** 3 // 3 + n1 * n1


# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch (flux: stages 2 and 3; the first stage reads U^n only
# once) from the committed `ncu --set full` captures named in profiles/*_summary.md; None where no capture exists.
NCU_TRAFFIC_BYTES = {                                   # profiles/r2_summary.md (captures prof_r2b_cfg4, prof_r2_cfg2 / cfg3)
    ("cfg4_3d_256cubed", "chem"): 5.98e9,
    ("cfg4_3d_256cubed", "flux"): 13.30e9,
    ("cfg2_2d_channel_4096x512", "flux"): 6.31e8,
    ("cfg2_2d_channel_4096x512", "chem"): 3.15e8,
    ("cfg3_amr_8192x16x16", "flux"): 9.65e8,
}
NCU_TRAFFIC_SOURCE = "ncu dram__bytes_read.sum + dram__bytes_write.sum per launch (profiles/*_summary.md)"


def flux_bytes_per_cell_stage(ndim, nvar):
    # read U^(k) (nvar) + p + u_d (ndim) + U^n (nvar, stages 2,3 -> counted always), write U^(k+1) (nvar)
    return (3 * nvar + 1 + ndim) * 8


def max_over_ranks(values, device, world):
    """Device times of one rank -> the maximum over all ranks (the contract's multi-GPU timing rule)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


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


def crop_case(case, nx2d, ny2d, n3d=32):
    """A bounded sample of a workload for the CPU oracle: 2-D uniform grids are cropped to their first nx2d x ny2d
    cells (the driver section and the ambient gas next to it), 3-D grids to the aligned n3d^3 sub-cube that holds the
    most hot cells; 1-D and block-list cases are small enough to run whole."""
    g = case.grid
    if g.n_patches == 0 and g.ndim == 2:
        nx, ny = min(g.n[0], nx2d), min(g.n[1], ny2d)
        U = np.ascontiguousarray(case.U[:, :, :, :ny, :nx]); T = np.ascontiguousarray(case.T[:, :, :ny, :nx])
        crop = I.Case(case.name + "_crop", I.Grid(2, (nx, ny, 1), g.dx, g.bc_lo, g.bc_hi), case.mech, U, T, case.cfl, 1)
        return crop, f"{case.name} cropped to {nx}x{ny} cells (columns 0..{nx - 1}, rows 0..{ny - 1})"
    if g.n_patches == 0 and g.ndim == 3 and g.n[0] > n3d:
        n = n3d
        nb = g.n[0] // n
        hot = (case.T[0] > 1000.0).reshape(nb, n, nb, n, nb, n).sum(axis=(1, 3, 5))
        kz, ky, kx = np.unravel_index(int(np.argmax(hot)), hot.shape)
        sl = (slice(kz * n, (kz + 1) * n), slice(ky * n, (ky + 1) * n), slice(kx * n, (kx + 1) * n))
        U = np.ascontiguousarray(case.U[(slice(None), slice(None)) + sl]); T = np.ascontiguousarray(case.T[(slice(None),) + sl])
        crop = I.Case(case.name + "_crop", I.Grid(3, (n, n, n), g.dx, g.bc_lo, g.bc_hi), case.mech, U, T, case.cfl, 1)
        return crop, (f"{case.name} cropped to the {n}^3 sub-cube at z,y,x = {kz * n},{ky * n},{kx * n} "
                      f"({int(hot[kz, ky, kx])} hot cells), periodic")
    return case, f"{case.name} (whole)"


def oracle_throughput(case, budget_s=15.0):
    """The oracle as it stands, on a bounded sample of the workload (cropped IC), host cores."""
    from oracle import ref
    ref.build()
    crop, desc = crop_case(case, 512, 256)
    s = ref.RefSolver(crop.grid, crop.mech, crop.blocks)
    s.set_state(crop.U, crop.T)
    cells = crop.cells
    t0 = time.perf_counter(); s.step(1, cfl=crop.cfl); t1 = time.perf_counter() - t0
    n = int(max(1, min(50, budget_s / max(t1, 1e-3))))
    t0 = time.perf_counter(); s.step(n, cfl=crop.cfl); tn = time.perf_counter() - t0
    s.close()
    return {"value": cells * n / tn, "unit": UNIT, "cores": ref.threads(), "kind": "oracle",
            "sample": f"{desc}, {n} steps after 1 warm-up, {tn:.1f} s"}, cells, tn / n


# ------------------------------------------------------------------------------------------------
def run_reference(args, rank, world):
    """--impl reference: the CPU oracle as it stands on a bounded sample per step (tier contract)."""
    if rank != 0:
        return
    case = make_case(args.workload)
    from oracle import ref
    ref.build()
    crop, desc = crop_case(case, 512, 128)
    desc += " per step"
    s = ref.RefSolver(crop.grid, crop.mech, crop.blocks)
    s.set_state(crop.U, crop.T)
    for _ in range(args.warmup):
        s.step(1, cfl=crop.cfl)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        s.step(1, cfl=crop.cfl)
    dt = time.perf_counter() - t0
    s.close()
    val = crop.cells * args.steps / dt
    cores = ref.threads()
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": case.name, "cells": case.cells, "ns": case.mech.ns, "nr": case.mech.nr,
                       "sample": desc},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def chem_bytes_per_cell(ndim, nvar, ns):
    # read U (nvar) + T guess, write rho Y_1..ns-1 + T
    return (nvar + 1 + ns) * 8


def measure(binding, case, K, W, local, world, barrier, do_e2e=True, crossover=False):
    """One workload on this rank's GPU: K timed steps with the state resident in HBM, K profiled steps (per-kernel
    device time, CUDA events on the library's stream), and (do_e2e) the end-to-end loop with pinned host buffers."""
    import torch
    dev = f"cuda:{local}"
    s = binding.Solver(case.grid, case.mech, case.blocks, device=local)
    out = {"chem_kernel": s.chem_kernel()}
    Ud = torch.from_numpy(case.U).to(dev); Td = torch.from_numpy(case.T).to(dev)
    s.set_state(Ud, Td)
    if crossover:      # timing of the sub-cycled level advance only (Fig 2a): no per-kernel phases, no e2e
        for _ in range(W):
            s.step(1, cfl=case.cfl, sync=False, crossover=True)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        for _ in range(K):
            s.step(1, cfl=case.cfl, sync=False, crossover=True)
        e1.record()
        barrier()
        assert s.status_sync() == 0
        out["ms"] = e0.elapsed_time(e1)
        s.close()
        return out
    for _ in range(W):
        s.step(1, cfl=case.cfl, sync=False)
    assert s.status_sync() == 0, "device flag raised during warm-up"
    l0 = s.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(K):
        s.step(1, cfl=case.cfl, sync=False)
    e1.record()
    barrier()
    out["ms"] = e0.elapsed_time(e1)
    out["launches"] = s.launch_count() - l0
    assert s.status_sync() == 0, "device flag raised during the timed region"
    phases = {}
    for _ in range(K):
        pr = s.profile_step(cfl=case.cfl)
        for k, (t, n) in pr.items():
            a = phases.setdefault(k, [0.0, 0]); a[0] += t; a[1] += n
    out["phases"] = phases
    if do_e2e:
        del Ud, Td
        Uh = torch.from_numpy(case.U).pin_memory(); Th = torch.from_numpy(case.T).pin_memory()
        Uo = torch.empty_like(Uh).pin_memory()
        Ke = max(1, min(K, 5))
        s.set_state(Uh.numpy(), Th.numpy()); s.step(1, cfl=case.cfl, sync=False); s.get_state_into(Uo.numpy())
        barrier()
        e0.record()
        for _ in range(Ke):
            s.set_state(Uh.numpy(), Th.numpy())
            s.step(1, cfl=case.cfl, sync=False)
            rc = s.get_state_into(Uo.numpy())
        e1.record()
        barrier()
        assert rc == 0
        out["ms_e2e"] = e0.elapsed_time(e1); out["Ke"] = Ke
        out["h2d"] = int(Uh.numel() * 8 + Th.numel() * 8); out["d2h"] = int(Uo.numel() * 8)
    s.close()
    return out


def measure_slab(binding, case, K, W, local, rank, world, barrier):
    """x-slab decomposition (slab.py): this rank's workload is one slab of a grid `world` times as long in x; per RK stage
    the 3 boundary columns go to the x neighbours (NCCL send / recv) and the reduction slots are max-all-reduced."""
    import torch
    from paper_2504_13750_b200 import slab
    g = case.grid
    assert g.n_patches == 0, "--parallel slab needs a uniform-grid workload"
    periodic = g.bc_lo[0] == I.BC_PERIODIC
    left, right = slab.neighbours(rank, world, periodic)
    lo, hi = list(g.bc_lo), list(g.bc_hi)
    if left is not None:
        lo[0] = binding.BC_EXCHANGE
    if right is not None:
        hi[0] = binding.BC_EXCHANGE
    lc = I.Case(case.name, I.Grid(g.ndim, g.n, g.dx, tuple(lo), tuple(hi)), case.mech, case.U, case.T, case.cfl, case.nsteps)
    run = slab.SlabRun(None, slab.DistComm(), device=local, local=[(lc, (rank * g.n[0], (rank + 1) * g.n[0]), (left, right))])
    s = run.solvers[0]
    out = {"chem_kernel": s.chem_kernel()}
    for _ in range(W):
        run.step(1, cfl=case.cfl)
    assert s.status_sync() == 0
    l0 = s.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    run.step(K, cfl=case.cfl)
    e1.record()
    barrier()
    out["ms"] = e0.elapsed_time(e1)
    out["launches"] = s.launch_count() - l0
    assert s.status_sync() == 0
    phases = {}
    for _ in range(K):      # per-kernel device times of this rank's slab advanced on its own (same kernels, stale halos)
        for k, (t, n) in s.profile_step(cfl=case.cfl).items():
            a = phases.setdefault(k, [0.0, 0]); a[0] += t; a[1] += n
    out["phases"] = phases
    # end to end: host -> device, K steps with exchange, device -> host
    Uh = torch.from_numpy(case.U).pin_memory(); Th = torch.from_numpy(case.T).pin_memory()
    Uo = torch.empty_like(Uh).pin_memory()
    Ke = max(1, min(K, 5))
    barrier()
    e0.record()
    for _ in range(Ke):
        s.set_state(Uh.numpy(), Th.numpy())
        run.step(1, cfl=case.cfl)
        rc = s.get_state_into(Uo.numpy())
    e1.record()
    barrier()
    assert rc == 0
    out["ms_e2e"] = e0.elapsed_time(e1); out["Ke"] = Ke
    out["h2d"] = int(Uh.numel() * 8 + Th.numel() * 8); out["d2h"] = int(Uo.numel() * 8)
    run.close()
    return out


def flux_kernel_name(case):
    """Which flux kernel janc.cu:do_flux launches for this workload with the default options."""
    g = case.grid
    even = (g.n[0] + 6) % 2 == 0                      # TMA needs 16-byte global strides: an even padded width
    if g.ndim == 1:
        return "k_flux_rk<1,128,1,1,4>"
    if g.ndim == 3:
        return "k_flux_rk3_tma<16,8,8,8>" if even else "k_flux_rk<3,16,8,8,8>"
    if g.n[0] <= 16 and g.n[1] <= 16 and g.n_patches > 0:
        return "k_flux_rk2<16,16,4,gather>"
    if case.cells < 600000:
        return "k_flux_rk2<32,16,4,gather>"
    return "k_flux_rk2_tma<64,16,8>" if even else "k_flux_rk2<64,16,8>"


def rooflines(case, m, K, dfma, hbm_peak, hbm_src):
    """Per-kernel roofline entries of one measured workload: algorithmic fp64 instructions and
    bytes per launch / the kernel's average launch duration (CUDA events, m["phases"]) against the DFMA rate measured
    in this run and the HBM copy bandwidth of MEASURED_PEAKS.json."""
    g, cells = case.grid, case.cells
    nd, nvar, ns = g.ndim, case.nvar, case.mech.ns
    ph = m["phases"]
    ent = {}
    fl_ms, fl_n = ph["flux_rk"]
    if fl_n:
        avg = fl_ms / fl_n * 1e-3
        ops = flux_ops_per_cell_stage(nd, nvar) * cells
        byt = flux_bytes_per_cell_stage(nd, nvar) * cells
        ent["flux"] = {"kernel": flux_kernel_name(case), "bound": "alu", "achieved": ops / avg / 1e12,
                       "peak": dfma / 1e12, "unit": "T fp64-instr/s (FMA=1)", "frac": ops / avg / dfma,
                       "traffic": NCU_TRAFFIC_BYTES.get((case.name, "flux")), "avg_launch_ms": avg * 1e3,
                       "launches_timed": fl_n, "ms_per_step": fl_ms / K,
                       "hbm": {"achieved": byt / avg / 1e9, "peak": hbm_peak, "unit": "GB/s", "frac": byt / avg / 1e9 / hbm_peak,
                               "peak_source": hbm_src}}
    ch_ms, ch_n = ph["chem"]
    if ch_n:
        avg = ch_ms / ch_n * 1e-3
        ops = chem_ops_per_cell(case.mech)
        byt = chem_bytes_per_cell(nd, nvar, ns) * cells
        ent["chem"] = {"kernel": "k_chem_jit (%s)" % m["chem_kernel"], "bound": "alu", "ops_per_cell": ops,
                       "achieved": ops * cells / avg / 1e12, "peak": dfma / 1e12, "unit": "T fp64-instr/s (FMA=1)",
                       "frac": ops * cells / avg / dfma, "traffic": NCU_TRAFFIC_BYTES.get((case.name, "chem")),
                       "avg_launch_ms": avg * 1e3, "launches_timed": ch_n, "ms_per_step": ch_ms / K,
                       "hbm": {"achieved": byt / avg / 1e9, "peak": hbm_peak, "unit": "GB/s", "frac": byt / avg / 1e9 / hbm_peak,
                               "peak_source": hbm_src}}
    return ent


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg4", choices=["cfg0", "cfg1", "cfg2", "cfg3", "cfg4"],
                    help="headline workload; default = the largest single-GPU config of BASELINE.json (configs[4])")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config block (N = 1 only)")
    ap.add_argument("--parallel", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: independent replicas (default; north_star keeps the path on one GPU) or the paper's x-slab "
                         "decomposition with halo exchange and max all-reduce over NCCL (PAPER.md:359-378), weak scaling: "
                         "every rank owns one workload-sized slab of a grid N times as long in x")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_2504_13750_b200 import binding, build
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libjanc has no CPU fallback")
    if rank == 0:
        build.build()
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
        dist.barrier()
    binding.lib()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    # replicas only: every rank advances its own independent problem
    case = make_case(args.workload, rank)
    K, W = args.steps, max(args.warmup, 3)
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
    if args.parallel == "slab" and world > 1:
        m = measure_slab(binding, case, K, W, local, rank, world, barrier)
    else:
        m = measure(binding, case, K, W, local, world, barrier)
    if sampler:           # clocks are sampled over the event-timed, the per-kernel and the end-to-end regions
        sampler.stop_flag = True
        sampler.join()
    dev = f"cuda:{local}"
    ms, ms_e2e = max_over_ranks([m["ms"], m["ms_e2e"]], dev, world)

    if rank == 0:
        cells, nvar = case.cells, case.nvar
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        hbm_peak = peaks.get("hbm_gbs", 6650.0)
        hbm_src = "measured (MEASURED_PEAKS.json)" if "hbm_gbs" in peaks else "fallback (B200_PROFILING.md)"
        dfma = binding.measure_dfma_peak(local)                      # DP instructions/s, measured now
        ent = rooflines(case, m, K, dfma, hbm_peak, hbm_src)
        # the dominant kernel of the step = the one with the most device time per step
        dom = max(ent, key=lambda k: ent[k]["ms_per_step"])
        roof = dict(ent[dom])
        roof["traffic_unit"] = NCU_TRAFFIC_SOURCE
        roof["peak_source"] = "measured: register-resident DFMA microbenchmark in this run"
        roof["kernels"] = {k: v for k, v in ent.items() if k != dom}
        line = {"metric": METRIC, "value": cells * world * K / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K,
                "warmup": W, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": case.name, "cells": cells, "ns": case.mech.ns, "nr": case.mech.nr,
                           "nvar": nvar, "cfl": case.cfl,
                           "parallelism": (f"x-slab decomposition x{world} (halo exchange + max all-reduce per RK stage, NCCL)"
                                           if args.parallel == "slab" and world > 1 else f"replicas x{world}"),
                           "l2": "state %.0f MB per register > 126 MB L2" % (cells * nvar * 8 / 1e6)
                                 if cells * nvar * 8 > 126e6 else "state fits L2 (no flush; noted)"},
                "clocks": sampler.summary(),
                "e2e": {"value": cells * world * m["Ke"] / (ms_e2e * 1e-3), "unit": UNIT,
                        "h2d_bytes_per_step": m["h2d"], "d2h_bytes_per_step": m["d2h"], "steps": m["Ke"]},
                "gpu_launches": int(m["launches"]),
                "roofline": roof,
                "phases_ms_per_step": {k: v[0] / K for k, v in m["phases"].items()},
                "context": {"paper_a100_cell_updates_per_s": 2.0e7, "note": "PAPER.md:448, other hardware and mechanism"}}
        if world == 1 and not args.no_per_config:
            # every BASELINE config at full size on this GPU (north_star: "throughput per config")
            per = {}
            for wl in ("cfg0", "cfg1", "cfg2", "cfg3", "cfg4"):
                if wl == args.workload:
                    c2, m2, K2 = case, m, K
                else:
                    c2 = make_case(wl, rank)
                    K2 = K
                    m2 = measure(binding, c2, K2, W, local, world, barrier, do_e2e=False)
                e2 = rooflines(c2, m2, K2, dfma, hbm_peak, hbm_src)
                step_ms = m2["ms"] / K2
                algo_bytes = (3 * ((c2.nvar + 3 + c2.grid.ndim) * 8 + flux_bytes_per_cell_stage(c2.grid.ndim, c2.nvar))
                              + chem_bytes_per_cell(c2.grid.ndim, c2.nvar, c2.mech.ns)) * c2.cells
                per[wl] = {"workload": c2.name, "cells": c2.cells, "value": c2.cells * K2 / (m2["ms"] * 1e-3),
                           "ms_per_step": step_ms, "gpu_launches_per_step": m2["launches"] / K2,
                           "phases_ms_per_step": {k: v[0] / K2 for k, v in m2["phases"].items()},
                           "flux": {k: e2["flux"][k] for k in ("kernel", "frac", "avg_launch_ms", "traffic")} if "flux" in e2 else None,
                           "flux_hbm_frac": e2["flux"]["hbm"]["frac"] if "flux" in e2 else None,
                           "chem": {k: e2["chem"][k] for k in ("kernel", "frac", "avg_launch_ms", "traffic")} if "chem" in e2 else None,
                           "hbm": {"achieved": algo_bytes / (step_ms * 1e-3) / 1e9, "frac": algo_bytes / (step_ms * 1e-3) / 1e9 / hbm_peak,
                                   "unit": "GB/s", "note": "algorithmic bytes of the whole step / step time"}}
                if c2.blocks is not None and c2.grid.n_levels == 2:
                    # the paper's recommended strategy (PAPER.md:186 Fig 2a, :476): one crossover step advances the
                    # solution as far as two synchronous steps
                    mx = measure(binding, c2, K2, W, local, world, barrier, do_e2e=False, crossover=True)
                    lev = c2.blocks.level
                    per[wl]["crossover"] = {"ms_per_level0_step": mx["ms"] / K2, "synchronous_ms_for_the_same_time": 2 * step_ms,
                                            "time_ratio": (mx["ms"] / K2) / (2 * step_ms),
                                            "cell_updates_per_s": (int((lev == 0).sum()) + 2 * int((lev == 1).sum())) * c2.cells // len(lev) * K2 / (mx["ms"] * 1e-3)}
                del c2
            line["per_config"] = per
        if not args.no_cpu_baseline and world >= 1:
            cb, _, _ = oracle_throughput(case)
            line["cpu_baseline"] = cb
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
