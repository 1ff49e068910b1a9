#!/usr/bin/env python
"""bench.py — the pressure projection on seeded synthetic grids, timed on the B200 (driver contract: see DESIGN.md §8).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]

One "step" = one pass of the whole hot path (SURVEY.md §8(a) H0–H9): ``wl_project(u, L, p=0)`` — coefficient hierarchy,
divergence, GMG V-cycles to ||r||inf <= 1e-4 ||b||inf (cap 32), pressure-gradient correction — on BASELINE.json
``configs[C]`` (default C = 4: 3-D 512^3 fp32, 32 seeded spheres, the largest single-GPU configuration).

The JSON line (rank 0):
  value      fine cells/s per V-cycle through the whole projection = n_gpus * M * cycles / seconds per step,
             inputs resident in HBM when the timed region starts (CUDA events on the ctx stream, summed over K steps);
  e2e        the same metric through ``wl_project_host`` with pinned HOST buffers: H2D of u, L, p and D2H of u, p inside
             the timed region;
  roofline   the dominant kernel — the fused level-0 DOWN kernel of the solve (mean shift on load, 2 pre-sweeps, residual of
             the input iterate, residual + restriction, bookkeeping ticket: the very template instance wl_solve's graph
             launches, selected through WL_OPT_SOLVE_KERNELS) — timed alone with CUDA events through ``wl_down``; achieved =
             algorithmic bytes (read p, b, n·L, write p, write b_c = (n+3+1/2^n)·s per cell) / duration,
             against MEASURED_PEAKS.json ``hbm_gbs`` (``frac``) and against the nominal 8 TB/s BASELINE.json names;
  cpu_baseline  the oracle as it stands on the box's host cores (1 thread), on a bounded sample (one V-cycle of the same
             workload);
  extra keys: ms per projection, ms per V-cycle (wl_solve with tol = 0 over --kernel-reps cycles: one graph launch per
             cycle, stop test on the device), effective GB/s per V-cycle (56 B/cell model) as a fraction of the measured and
             of the nominal peak; roofline.traffic = DRAM bytes of one DOWN launch from profiles/traffic.json (written from
             the last ``ncu --set full`` capture together with a hash of csrc/; null when the kernels have changed since).

N > 1 (torchrun): "replicas only" — every rank projects its own copy of the grid, no collective on the data path
(BASELINE.json north_star: one GPU, no sharding); value = units all ranks processed / max-over-ranks time.
``--impl reference`` times the CPU oracle (rank 0 only) on the same config and metric.
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

METRIC = "GMG V-cycle fine cells/s (whole projection)"
UNIT = "cells/s"


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
    except Exception:
        return 6650.0, "B200_PROFILING.md fallback 6.65 TB/s (of fallback)"


def max_over_ranks(values, device=None):
    """Element-wise MAX of a list of floats over all ranks of the default process group (identity at world size 1).
    The only collective of the N > 1 ("replicas only") path; works on NCCL (device tensor) and on gloo (CPU)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values]
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.tolist()]


def whole_job_value(world: int, cells: int, cycles: int, seconds_per_step: float) -> float:
    """Fine cells per second per V-cycle, summed over the `world` replicas (each rank projects its own grid)."""
    return world * cells * cycles / seconds_per_step if (cycles > 0 and seconds_per_step > 0) else 0.0


NOMINAL_HBM_GBS = 8000.0   # BASELINE.json north_star: "the B200's ~8 TB/s HBM peak"


def csrc_hash() -> str:
    """sha256 over the CUDA sources and the C header: identifies the kernels a recorded ncu number belongs to."""
    import glob
    import hashlib
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_2304_08159_b200", "csrc")
    files = sorted(glob.glob(os.path.join(csrc, "*.cu*")) + glob.glob(os.path.join(csrc, "*.h"))) + [os.path.join(ROOT, "include", "wl.h")]
    for f in files:
        with open(f, "rb") as fh:
            h.update(os.path.basename(f).encode() + b"\0" + fh.read())
    return h.hexdigest()[:16]


def recorded_traffic(workload: str, kernel_key: str):
    """DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) of one launch of `kernel_key` on `workload` from
    profiles/traffic.json, or None if there is no record for the kernels as they are now (ncu never runs inside bench.py)."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            rec = json.load(f)
        if rec.get("csrc_hash") != csrc_hash():
            return None
        e = rec["kernels"][workload][kernel_key]
        return float(e["dram_bytes_read"]) + float(e["dram_bytes_write"])
    except Exception:
        return None


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        self.paused = False   # set while the benchmark idles on purpose: idle clocks are not 'clocks under load'
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nv = None

    def _loop(self):
        nv = self._nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4),
        }
        while not self._stop.is_set():
            if self.paused:
                self._stop.wait(0.05)
                continue
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(0.05)

    def __enter__(self):
        if self._nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        med = int(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def _algorithmic_bytes_down(n: int, esz: int) -> float:
    """Level-0 DOWN kernel, per cell: read p, b, n·L; write p; write b_c (1/2^n of a cell)."""
    return (n + 3 + 1.0 / 2 ** n) * esz


# convdiff (NEXT-4), per face flux as the oracle's formula states it: U (2), third-order value (5 incl. the division), limiter
# bound (3), two medians (8 compare/select), flux (4) = 22 operations; 9 fluxes per 3-D cell (each face flux serves two control
# volumes) + 2 per flux difference accumulated x 9 = 216 operations per cell (2-D: 4 fluxes, 96).  None can fuse into an FMA
# (every operation rounds separately, reading 12), so the ALU ceiling is one operation per FP32 lane and clock:
# SMs x 128 lanes x SM clock (B200_PROFILING.md: 148 SMs; the clock is the one sampled during the run).  The packed f32x2
# instructions the kernel uses do not raise that ceiling: wl_selftest_fp32_rates measures 128 lane-operations per clock and SM
# for scalar and packed adds and fmas alike (profiles/r3_packed_rate.md); the measured figure rides along as `alu_rates`.
def convdiff_report(cd, n, M, esz, hbm_peak, clocks, rates=None):
    if cd is None:
        return None
    sec = cd["ms"] * 1e-3
    nb = 2 * n * esz * M                       # read u, write r: n components each
    ops = (22 * n * n + 2 * n * n) * M
    mhz = clocks.get("sm_mhz") or clocks.get("sm_max_mhz") or 1965
    lanes = 128 if esz == 4 else 64            # FP64 units per SM: half the FP32 lanes
    alu_peak = 148 * lanes * mhz * 1e6 / 1e12
    return {"kernel": "k_convdiff3d (TMA-staged tiles, every flux once)" if n == 3 else "k_convdiff (one thread per cell)",
            "ms": cd["ms"], "cells_per_s": M / sec,
            "roofline": {"bound": "alu", "achieved": ops / sec / 1e12, "peak": alu_peak, "unit": "TFLOP/s", "frac": ops / sec / 1e12 / alu_peak,
                         "ops_per_cell": ops // M, "peak_source": f"148 SMs x {lanes} lanes x sampled SM clock ({mhz} MHz), one non-fused operation per lane and clock",
                         "alu_rates": None if rates is None else {k: {"warp_instr_per_clk_sm": v[0], "lane_ops_per_clk_sm": v[1]} for k, v in rates.items()}},
            "hbm": {"algorithmic_bytes": nb, "achieved_GBps": nb / sec / 1e9, "frac_of_measured": nb / sec / 1e9 / hbm_peak}}


def run_reference(args, rank: int):
    """The oracle timed on host cores: each step = one V-cycle (+ mean removal + residual norm) of the same workload."""
    if rank != 0:
        return
    from paper_2304_08159_b200 import synth
    import oracle
    oracle.build()
    cfg = synth.make_donut(args.donut) if args.donut else synth.make_config(args.config, scale=args.scale)
    dims, dt = cfg["dims"], cfg["dtype"]
    M = int(np.prod(dims))
    o = oracle.Oracle(dims, dt)
    o.set_coeff(cfg["L"])
    b = o.divergence(cfg["u"])
    p = np.zeros(tuple(reversed(dims)), dt)
    times = []
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        p, _ = o.vcycle(p, b)
        t1 = time.perf_counter()
        if it >= args.warmup:
            times.append(t1 - t0)
    sec = float(np.sum(times)) / max(1, len(times))
    val = M / sec
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if dt == np.float32 else "f64", "data": "synthetic",
        "config": {"workload": cfg["name"], "dims": list(dims), "sample": "each step = one oracle V-cycle"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": f"{args.steps} V-cycles of {cfg['name']} after {args.warmup} warm-up cycles"},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--scale", type=int, default=1, help="divide every extent (debug only; the default 1 is the workload)")
    ap.add_argument("--donut", type=int, default=0, help="P in 4..7: the paper-shaped (2^(P+1), 2^P, 2^P) torus grid instead of --config")
    ap.add_argument("--dtype", default=None, choices=[None, "float32", "float64"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-upload-L", action="store_true", help="e2e leg: upload the n·M coefficient array instead of the body records")
    ap.add_argument("--no-pcg", action="store_true", help="skip the conjugate-gradient leg (reported beside the V-cycle solver)")
    ap.add_argument("--no-convdiff", action="store_true", help="skip the convdiff leg (NEXT-4, timed alone on the same velocity)")
    ap.add_argument("--no-vcycle-256", action="store_true", help="skip the 256^3 V-cycle leg that rides on the default config-4 run")
    ap.add_argument("--fused", type=int, default=1)
    ap.add_argument("--graph", type=int, default=1)
    ap.add_argument("--pdl", type=int, default=1, help="WL_OPT_PDL: programmatic dependent launch between the kernels of a cycle")
    ap.add_argument("--kernel-reps", type=int, default=20)
    ap.add_argument("--roofline-idle", type=float, default=1.5, help="seconds of idle before the dominant kernels are timed alone")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.warmup < 3:
        args.warmup = 3  # timing rule: W >= 3

    import torch
    import torch.distributed as dist
    from paper_2304_08159_b200 import binding as wl, synth, build
    build.build_cuda()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (there is no CPU path)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    dt_np = None if args.dtype is None else np.dtype(args.dtype)
    cfg = synth.make_donut(args.donut, dtype=dt_np) if args.donut else synth.make_config(args.config, dtype=dt_np, scale=args.scale)
    dims, dt = cfg["dims"], cfg["dtype"]
    n, M, esz = len(dims), int(np.prod(dims)), cfg["dtype"].itemsize
    tol, maxc = cfg["tol"], cfg["maxcycles"]
    if tol == 0.0:  # config 0 is a fixed-cycle case
        tol = 0.0

    pr = wl.Projector(dims, dt, dev)
    wl.wl_set_option(pr.ctx, wl.WL_OPT_FUSED, args.fused)
    wl.wl_set_option(pr.ctx, wl.WL_OPT_GRAPH, args.graph)
    wl.wl_set_option(pr.ctx, wl.WL_OPT_PDL, args.pdl)
    u_host = torch.from_numpy(cfg["u"]).pin_memory()
    L_host = torch.from_numpy(cfg["L"]).pin_memory()
    u0 = u_host.to(dev, non_blocking=True)
    Ld = L_host.to(dev, non_blocking=True)
    u = torch.empty_like(u0)
    p = pr.zeros_cells()
    stream = torch.cuda.current_stream()

    def one_step():
        u.copy_(u0)
        p.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        hist, nc, rc = wl.wl_project(pr.ctx, u, Ld, p, tol, maxc)
        e1.record(stream)
        e1.synchronize()
        return e0.elapsed_time(e1), hist, nc, rc

    for _ in range(args.warmup):
        one_step()
    barrier()
    launches0 = wl.wl_launch_count(pr.ctx)
    ms = []
    with ClockSampler(local_rank) as clk:
        for _ in range(args.steps):
            t, hist, nc, rc = one_step()
            ms.append(t)
        launches = wl.wl_launch_count(pr.ctx) - launches0
        barrier()
        total_ms = float(np.sum(ms))

        # the dominant kernels alone (roofline leg): first straight after the timed steps, with the board in the power / clock
        # state a long step leaves it in ("in_step"), then again after a short idle ("burst": MEASURED_PEAKS.json's copy rate
        # is a burst figure — a copy kernel timed alone on an idle GPU — so that is the like-for-like fraction).
        kern, kern_in_step = {}, {}
        reps = max(5, args.kernel_reps)
        if pr.num_levels > 1:
            wl.wl_set_option(pr.ctx, wl.WL_OPT_SOLVE_KERNELS, 1)   # time the instances the solve's graph launches
            bd = pr.empty_cells()
            wl.wl_divergence(pr.ctx, u0, bd)
            xo = pr.empty_cells()

            def time_level0(out):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                for name, fn in (("down", lambda: wl.wl_down(pr.ctx, 0, p, bd, xo)),
                                 ("up", lambda: wl.wl_up(pr.ctx, 0, xo, None, bd, p))):
                    for _ in range(3):
                        fn()
                    l0 = wl.wl_launch_count(pr.ctx)
                    torch.cuda.synchronize()
                    e0.record(stream)
                    for _ in range(reps):
                        fn()
                    e1.record(stream)
                    e1.synchronize()
                    out[name] = {"ms": e0.elapsed_time(e1) / reps, "launches_per_call": (wl.wl_launch_count(pr.ctx) - l0) // reps}

            for _ in range(2):                      # two more projections so the kernels below start from the step's own state
                one_step()
            time_level0(kern_in_step)
            torch.cuda.synchronize()
            clk.paused = True
            time.sleep(args.roofline_idle)
            clk.paused = False
            time_level0(kern)
            wl.wl_set_option(pr.ctx, wl.WL_OPT_SOLVE_KERNELS, 0)
            del xo

        # where the part of ms_per_step that is not V-cycles goes: the pieces of one projection timed one by one through their
        # own entry points (same kernels; wl_solve = cycles + the final mean shift)
        breakdown = None
        if pr.num_levels > 1:
            def timed(fn, nrep=3):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                fn()
                torch.cuda.synchronize()
                e0.record(stream)
                for _ in range(nrep):
                    fn()
                e1.record(stream)
                e1.synchronize()
                return e0.elapsed_time(e1) / nrep
            bq = pr.empty_cells()
            u.copy_(u0)
            breakdown = {"set_coeff": timed(lambda: wl.wl_set_coeff(pr.ctx, Ld)),
                         "divergence": timed(lambda: wl.wl_divergence(pr.ctx, u, bq))}
            def solve_once():
                p.zero_()
                return wl.wl_solve(pr.ctx, p, bq, tol, maxc)
            breakdown["solve"] = timed(solve_once, 2)
            breakdown["solve_cycles"] = int(solve_once()[1])
            breakdown["gradient"] = timed(lambda: wl.wl_gradient(pr.ctx, u, p))
            breakdown["sum"] = breakdown["set_coeff"] + breakdown["divergence"] + breakdown["solve"] + breakdown["gradient"]
            breakdown["note"] = "ms; solve includes p.zero_() and the final mean shift; pieces timed alone, so their sum need not equal ms_per_step"
            del bq

        # e2e: the same projection through the host-buffer entry point with pinned HOST buffers.  Inputs of a step: the
        # face velocity u (n·M values) and the bodies' analytic description (8 doubles each) from which wl_set_bodies builds
        # the coefficient hierarchy on the device (no coefficient array crosses the bus); p starts from 0
        # (WL_OPT_HOST_P_ZERO).  Results read back every step: u and p.  --e2e-upload-L uploads the n·M coefficients instead.
        if not args.no_e2e:
            uh = torch.empty_like(u_host).pin_memory()
            ph = torch.zeros(pr.cell_shape(), dtype=pr.torch_dtype).pin_memory()
            wl.wl_set_option(pr.ctx, wl.WL_OPT_HOST_P_ZERO, 1)
            e2e_ms = []
            for it in range(2 + args.steps):
                uh.copy_(u_host)
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                if args.e2e_upload_L:
                    h2, nc2, rc2 = wl.wl_project_host(pr.ctx, uh, L_host, ph, tol, maxc)
                else:
                    wl.wl_set_bodies(pr.ctx, cfg["bodies"])
                    h2, nc2, rc2 = wl.wl_project_host(pr.ctx, uh, None, ph, tol, maxc)
                e1.record(stream)
                e1.synchronize()
                if it >= 2:
                    e2e_ms.append(e0.elapsed_time(e1))
            e2e_total = float(np.sum(e2e_ms))
            wl.wl_set_option(pr.ctx, wl.WL_OPT_HOST_P_ZERO, 0)
            wl.wl_set_coeff(pr.ctx, Ld)   # back to the uploaded field for the legs below

        # NEXT-1 beside the specified solver: the same projection with V-cycle-preconditioned conjugate gradients
        pcg = None
        if not args.no_pcg:
            wl.wl_set_option(pr.ctx, wl.WL_OPT_SOLVER, 1)
            pms = []
            for it in range(1 + max(2, args.steps)):
                tms, hp, ncp, rcp = one_step()
                if it >= 1:
                    pms.append(tms)
            wl.wl_set_option(pr.ctx, wl.WL_OPT_SOLVER, 0)
            pcg = {"solver": "wl_solve_pcg (one V-cycle per CG iteration)", "iterations": int(ncp), "converged": bool(rcp == 0),
                   "ms_per_projection": float(np.mean(pms)), "final_rel_residual": float(hp[-1] / hp[0]) if hp[0] > 0 else 0.0}

        # NEXT-4: the other dominant routine of the paper's step (`convdiff!`) on the same velocity field, timed alone
        cd, fp32_rates = None, None
        if not args.no_convdiff:
            rcd = torch.empty_like(u0)
            for _ in range(3):
                wl.wl_convdiff(pr.ctx, u0, 1e-3, rcd)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record(stream)
            for _ in range(reps):
                wl.wl_convdiff(pr.ctx, u0, 1e-3, rcd)
            e1.record(stream)
            e1.synchronize()
            cd = {"ms": e0.elapsed_time(e1) / reps}
            del rcd
            fp32_rates = wl.wl_selftest_fp32_rates(pr.ctx)   # measured lane-operations per clock and SM, scalar and packed

        # V-cycles alone: wl_solve with tol = 0 runs exactly `reps` cycles (one graph launch + one 8-byte readback each,
        # mean shift deferred into the next cycle); the dominant kernels alone follow
        if pr.num_levels <= 1:
            bd = pr.empty_cells()
            wl.wl_divergence(pr.ctx, u0, bd)
        p.zero_()
        wl.wl_solve(pr.ctx, p, bd, 0.0, 3)
        p.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        wl.wl_solve(pr.ctx, p, bd, 0.0, reps)
        e1.record(stream)
        e1.synchronize()
        vcycle_ms = e0.elapsed_time(e1) / reps

        # the other grid BASELINE.json's target names (256^3 fp32, config 3): V-cycles alone on a context of its own (0.3 GB)
        vc256 = None
        if world == 1 and not args.donut and args.config == 4 and args.scale == 1 and not args.no_vcycle_256:
            c3 = synth.make_config(3)
            d3, M3, n3, es3 = c3["dims"], int(np.prod(c3["dims"])), len(c3["dims"]), c3["dtype"].itemsize
            pr3 = wl.Projector(d3, c3["dtype"], dev)
            wl.wl_set_option(pr3.ctx, wl.WL_OPT_PDL, args.pdl)
            wl.wl_set_coeff(pr3.ctx, torch.from_numpy(c3["L"]).to(dev))
            b3, p3 = pr3.empty_cells(), pr3.zeros_cells()
            wl.wl_divergence(pr3.ctx, torch.from_numpy(c3["u"]).to(dev), b3)
            wl.wl_solve(pr3.ctx, p3, b3, 0.0, 3)
            best = None
            for _ in range(3):
                p3.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                e0.record(stream)
                wl.wl_solve(pr3.ctx, p3, b3, 0.0, reps)
                e1.record(stream)
                e1.synchronize()
                t3 = e0.elapsed_time(e1) / reps
                best = t3 if best is None else min(best, t3)
            eff3 = (2 * (n3 + 3) + 2.0 / 2 ** n3) * es3 * (2 ** n3 / (2 ** n3 - 1.0)) * M3 / (best * 1e-3) / 1e9
            vc256 = {"workload": c3["name"], "ms": best, "effective_GBps_56B_model": eff3, "frac_of_measured": eff3 / _peaks()[0],
                     "frac_of_nominal_8TBs": eff3 / NOMINAL_HBM_GBS, "timed": f"best of 3 x {reps} cycles (wl_solve, tol = 0); working set fits L2"}
            pr3.close()
            del b3, p3

    clocks = clk.summary()

    # max over ranks
    if world > 1:
        red = max_over_ranks([total_ms, 0.0 if args.no_e2e else e2e_total], dev)
        total_ms = red[0]
        if not args.no_e2e:
            e2e_total = red[1]

    sec_per_step = total_ms / 1e3 / args.steps
    value = whole_job_value(world, M, int(nc), sec_per_step)
    peak, peak_src = _peaks()
    roof = None
    if kern:
        bytes_down = _algorithmic_bytes_down(n, esz) * M
        ach = bytes_down / (kern["down"]["ms"] * 1e-3) / 1e9
        fused3 = (n == 3 and args.fused != 0)
        roof = {"bound": "hbm",
                "kernel": ("level-0 DOWN of the solve: k_fused3d<SHIFT, STAGE3, RESTRICT, RIN, TICKET> (mean shift on load, 2 pre-sweeps, "
                           "input-residual norm, residual + restriction, bookkeeping), via wl_down with WL_OPT_SOLVE_KERNELS") if fused3
                          else "level-0 DOWN half (2 pre-sweeps + residual + restriction), via wl_down",
                "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "frac_of_nominal_8TBs": ach / NOMINAL_HBM_GBS,
                "traffic": recorded_traffic(cfg["name"], "down"),
                "peak_source": peak_src, "algorithmic_bytes_per_launch": bytes_down,
                "launches_per_call": kern["down"]["launches_per_call"], "ms": kern["down"]["ms"],
                "timed": f"{reps} launches alone after 3 warm-ups and {args.roofline_idle} s of idle (burst, as the peak was measured); "
                         "in_step = the same launches straight after the timed projections, no idle",
                "in_step": {"ms": kern_in_step["down"]["ms"],
                            "achieved": bytes_down / (kern_in_step["down"]["ms"] * 1e-3) / 1e9,
                            "frac": bytes_down / (kern_in_step["down"]["ms"] * 1e-3) / 1e9 / peak,
                            "up_ms": kern_in_step["up"]["ms"],
                            "up_frac": bytes_down / (kern_in_step["up"]["ms"] * 1e-3) / 1e9 / peak},
                "up_kernel": {"ms": kern["up"]["ms"], "achieved": bytes_down / (kern["up"]["ms"] * 1e-3) / 1e9,
                              "frac": bytes_down / (kern["up"]["ms"] * 1e-3) / 1e9 / peak,
                              "traffic": recorded_traffic(cfg["name"], "up"),
                              "launches_per_call": kern["up"]["launches_per_call"]}}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": sec_per_step * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if dt == np.float32 else "f64", "data": "synthetic",
        "config": {"workload": cfg["name"], "dims": list(dims), "cells": M, "tol": tol, "maxcycles": maxc,
                   "cycles_run": int(nc), "converged": bool(rc == 0), "fused": args.fused, "graph": args.graph, "pdl": args.pdl,
                   "l2": "inputs larger than L2 (no flush needed)" if (n + 3) * M * esz > 200e6 else "working set fits L2",
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "ms_per_projection": sec_per_step * 1e3,
        "vcycle": (lambda eff: {"ms": vcycle_ms, "cells_per_s": M / (vcycle_ms * 1e-3), "effective_GBps_56B_model": eff,
                                "frac_of_measured": eff / peak, "frac_of_nominal_8TBs": eff / NOMINAL_HBM_GBS})(
            (2 * (n + 3) + 2.0 / 2 ** n) * esz * (2 ** n / (2 ** n - 1.0)) * M / (vcycle_ms * 1e-3) / 1e9),
        "vcycle_256": vc256,
        "breakdown_ms": breakdown,
        "pcg": pcg,
        "convdiff": convdiff_report(cd, n, M, esz, peak, clocks, fp32_rates),
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": roof,
    }
    if not args.no_e2e:
        e2e_sec = e2e_total / 1e3 / args.steps
        h2d = u_host.numel() * esz + (L_host.numel() * esz if args.e2e_upload_L else int(cfg["bodies"].size) * 8)
        d2h = u_host.numel() * esz + M * esz
        line["e2e"] = {"value": whole_job_value(world, M, int(nc2), e2e_sec), "unit": UNIT, "ms_per_step": e2e_sec * 1e3,
                       "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "cycles_run": int(nc2),
                       "inputs": "u + coefficient array L (wl_set_coeff inside wl_project_host)" if args.e2e_upload_L
                                 else "u + body records (wl_set_bodies builds L on the device); p0 = 0 not uploaded"}

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        # the oracle as it stands, one thread, bounded sample: one V-cycle of the same workload
        import oracle
        oracle.build()
        o = oracle.Oracle(dims, dt)
        o.set_coeff(cfg["L"])
        bo = o.divergence(cfg["u"])
        po = np.zeros(tuple(reversed(dims)), dt)
        ncyc = 1 if M >= (1 << 26) else max(1, min(10, int(2e8 // M)))
        t0 = time.perf_counter()
        for _ in range(ncyc):
            po, _ = o.vcycle(po, bo)
        tc = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": M * ncyc / tc, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"{ncyc} oracle V-cycle(s) of {cfg['name']} ({tc:.1f} s), host nproc={os.cpu_count()}"}
        if line.get("convdiff"):
            # the oracle's convdiff on a bounded sample: the first planes of the same velocity field as a closed box of its own
            # (same work per cell; about 10 s)
            us = np.ascontiguousarray(cfg["u"][:, : max(4, min(cfg["u"].shape[1], int(1.6e7 // max(1, M // cfg["u"].shape[1]))))])
            t0 = time.perf_counter()
            oracle.convdiff(us, 1e-3)
            tcd = time.perf_counter() - t0
            line["convdiff"]["cpu_baseline"] = {"value": us[0].size / tcd, "unit": "cells/s", "cores": 1, "kind": "oracle",
                                                "sample": f"oracle convdiff on the first {us.shape[1]} planes of {cfg['name']} ({tcd:.1f} s)"}
    if rank == 0:
        print(json.dumps(line), flush=True)
    pr.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
