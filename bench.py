#!/usr/bin/env python
"""bench.py — FP64 cell-updates/s of the explicit cardiac time step on B200(s).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

One "step" = one pass of the whole hot path over the config's workload: ALL time steps of the
chosen BASELINE.json config (default configs[1]: FHN 512x512, 4th-order cross stencil, RK4,
10,000 time steps), every time step being stencil + no-flux boundary + reaction + RK stages.
Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for the accounting.
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

from paper_1309_1720_b200 import workloads as W  # noqa: E402
from paper_1309_1720_b200 import dist as D       # noqa: E402

METRIC = "fp64_cell_updates_per_second"
UNIT = "Gcell-step/s"

# algorithmic bytes per cell-step with one global dependency per RK stage, every field stored
# (SURVEY.md §8(d) / DESIGN.md "Roofline"): doubles read+written per field x 8 B
ALGO_DOUBLES = {W.EULER: 2, W.HEUN: 5, W.RK4: 13, W.RUSH_LARSEN: 2, W.IMPLICIT_EULER: 2}


def algo_bytes_per_cell_step(cfg) -> int:
    return 8 * ALGO_DOUBLES[cfg.integrator] * cfg.n_v


# Algorithmic FP64 work per cell-step of the five configs: FP64 instructions (DFMA + DMUL + DADD) and
# flops (DFMA = 2) of the non-redundant update of ONE cell through all substeps, counted in the SASS of
# the stage kernels (cuobjdump, body of ring_stage_kernel<model, stencil, kind>, per pair / 2; DESIGN.md
# "Roofline").  Peak: 148 SM x 64 FP64 lanes/clk x 1.965 GHz = 18.6 T instr/s = 37.2 TFLOP/s.
FP64_PER_CELL_STEP = {   # (model, stencil, integrator): (instructions, flops)
    (W.FHN, W.LAP5, W.EULER): (18, 26),
    (W.FHN, W.LAP9X4, W.RK4): (120, 170),
    (W.KARMA, W.LAP5, W.RK4): (220, 342),
    (W.BOCF, W.LAP9X4, W.RK4): (633, 1045),
}
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12


def floor_bytes_per_cell_step(cfg) -> int:
    return 16 * cfg.n_v   # read + write every field once, if all stages were fused on chip


def fp64_view(cfg, gcell_steps_per_s):
    """The other candidate bound of north_star: algorithmic FP64 flops per cell-step at the FP64 peak."""
    k = (cfg.model, cfg.stencil, cfg.integrator)
    if k not in FP64_PER_CELL_STEP:
        return None
    instr, flops = FP64_PER_CELL_STEP[k]
    ach = gcell_steps_per_s * flops / 1e3
    return {"achieved": ach, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": ach / FP64_PEAK_TFLOPS,
            "flops_per_cell_step": flops, "fp64_instructions_per_cell_step": instr,
            "peak_source": "derived: 148 SM x 64 FP64 lanes/clk x 2 x 1.965 GHz (DESIGN.md)"}


def measured_peaks() -> tuple[float, str]:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def recorded_traffic(cfg, plan_name):
    """ncu dram bytes per launch of the dominant kernel, if a capture was committed for this config
    (profiles/traffic.csv, written by hand from the .ncu-rep named there)."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(p):
        import csv
        for row in csv.DictReader(open(p)):
            if row.get("config:plan") == f"{cfg.name}:{plan_name}":
                try:
                    return int(row["dram_bytes_per_launch"])
                except (KeyError, ValueError):
                    return None
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None
        self.path = f"/tmp/bench_clocks_{os.getpid()}.csv"

    def start(self):
        try:
            self.fh = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=self.fh, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.fh.close()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in open(self.path):
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 9:
                continue
            try:
                sm.append(float(parts[1])); mx.append(float(parts[2]))
            except ValueError:
                continue
            for name, val in zip(names, parts[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        try:
            os.remove(self.path)
        except OSError:
            pass
        if sm:
            # "under load": the upper half of the samples (idle gaps between steps drop the clock)
            out.update(sm_mhz=statistics.median(sorted(sm)[len(sm) // 2:]), sm_max_mhz=max(mx),
                       reasons=sorted(reasons), samples=len(sm))
        return out


def oracle_rate(cfg, Z0, budget_s: float):
    """Time the oracle as it stands on a bounded sample of the same workload (same grid, same
    scheme, first steps of the run).  Returns (Gcell-step/s, threads, steps timed, seconds)."""
    import oracle as O
    one = Z0[:1] if cfg.batch > 1 else Z0
    cells = cfg.nx * cfg.ny * one.shape[0]
    best = None
    for omp in (False, True):
        t = time.perf_counter()
        O.step(cfg.model, one, cfg.dx, cfg.dt, cfg.scheme, 1, omp=omp)
        dt1 = time.perf_counter() - t
        if best is None or dt1 < best[1]:
            best = (omp, dt1)
    omp, dt1 = best
    if dt1 * 10 < budget_s:                 # the first call pays the thread start-up: calibrate on 10 more
        t = time.perf_counter()
        O.step(cfg.model, one, cfg.dx, cfg.dt, cfg.scheme, 10, omp=omp)
        dt1 = (time.perf_counter() - t) / 10
    n = max(1, int(budget_s / max(dt1, 1e-6)))
    t = time.perf_counter()
    O.step(cfg.model, one, cfg.dx, cfg.dt, cfg.scheme, n, omp=omp)
    dt = time.perf_counter() - t
    return cells * n / dt / 1e9, O.threads(omp), n, dt


def run_reference(args, cfg, rank):
    """--impl reference: the oracle on the host cores, same metric/config; each step is a bounded
    sample (a few time steps of the config's grid)."""
    if rank != 0:
        return
    import oracle as O
    Z0 = W.initial_state(cfg)
    rate, threads, n, secs = oracle_rate(cfg, Z0, 1.0)
    per_step = max(1, int(n * 3.0 / max(secs, 1e-6)))          # ~3 s of CPU work per bench step
    omp = threads > 1
    one = Z0[:1] if cfg.batch > 1 else Z0
    cells = cfg.nx * cfg.ny * one.shape[0]
    for _ in range(args.warmup):
        O.step(cfg.model, one, cfg.dx, cfg.dt, cfg.scheme, 1, omp=omp)
    t = time.perf_counter()
    z = one
    for _ in range(args.steps):
        z = O.step(cfg.model, z, cfg.dx, cfg.dt, cfg.scheme, per_step, omp=omp)
    total = time.perf_counter() - t
    value = cells * per_step * args.steps / total / 1e9
    sample = f"{per_step} of {cfg.nsteps} time steps of {cfg.describe()} per bench step (1 batch member)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 0,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": cfg.describe(), "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


PLAN_NAMES = {1: "stage", 2: "fused", 3: "persistent", 4: "pair"}


def time_config(C, torch, cfg, Z0, steps, warmup, flush, plan=0, plan_param=0):
    """Device-timed throughput of `steps` whole runs of cfg (state resident), L2 flushed between."""
    with C.Context.from_config(cfg, plan=plan, plan_param=plan_param) as ctx:
        ctx.set_state(Z0)
        for _ in range(warmup):
            ctx.step(cfg.nsteps)
        torch.cuda.synchronize()
        l0 = ctx.launches
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        D.barrier()
        torch.cuda.synchronize()
        for a, b in ev:
            flush.zero_()                      # > L2 (126 MB): evict the state between timed steps
            a.record()
            ctx.step(cfg.nsteps)
            b.record()
        torch.cuda.synchronize()
        D.barrier()
        ms = sum(a.elapsed_time(b) for a, b in ev)
        launches = ctx.launches - l0
        plan_used = ctx.plan
        final = ctx.get_state()
    if not np.all(np.isfinite(final)):
        raise RuntimeError("non-finite state after the timed run")
    return ms, launches, plan_used


def run_sweep(args):
    """Size sweep 'S' (the shape of the paper's Fig. 5): each model, RK4,
    N = 64 .. 8192, AUTO plan and the STAGE plan; one JSON line.  Not the bench line."""
    import torch
    torch.cuda.set_device(0)
    from paper_1309_1720_b200 import cardiac as C
    peak, _ = measured_peaks()
    rows = []
    for model in (W.FHN, W.KARMA, W.BOCF):
        for n in W.sweep_sizes():
            cfg = W.sweep_config(model, n)
            Z = W.sweep_state(cfg)
            for plan in (0, 1):
                with C.Context.from_config(cfg, plan=plan) as ctx:
                    used = ctx.plan
                    if plan == 1 and rows and rows[-1]["n"] == n and rows[-1]["plan"] == "stage":
                        continue                              # AUTO already was STAGE
                    ctx.set_state(Z)
                    ctx.step(cfg.nsteps)
                    torch.cuda.synchronize()
                    best = min(C.cardiac_time_steps(ctx.ctx, cfg.nsteps, 1) for _ in range(3))
                v = cfg.cells * cfg.nsteps / (best * 1e-3) / 1e9
                rows.append({"model": W.MODEL_NAMES[model], "n": n, "stencil": W.STENCIL_NAMES[cfg.stencil],
                             "plan": PLAN_NAMES.get(used, str(used)), "nsteps": cfg.nsteps,
                             "us_per_step": best * 1e3 / cfg.nsteps, "value": v, "unit": UNIT,
                             "hbm_frac_stage_sync": v * algo_bytes_per_cell_step(cfg) / peak})
            del Z
    print(json.dumps({"sweep": rows, "integrator": "rk4", "peak_gbs": peak}))


def run_slabs(args, cfg):
    """`--decompose slabs`: ONE grid of the config cut into row slabs over the ranks (strong scaling;
    DESIGN.md "Multi-GPU", paper_1309_1720_b200/dist.py): every rank advances its slab plus ghost rows
    with the single-GPU kernels and swaps r x substeps x k ghost rows with its neighbours every k time
    steps (NCCL send/recv).  Not the default bench line: the BASELINE configs fit one GPU."""
    import torch
    rank, local_rank, world = D.env_world()
    D.init("nccl")
    torch.cuda.set_device(local_rank)
    from paper_1309_1720_b200 import cardiac as C
    stages = {W.EULER: 1, W.HEUN: 2, W.RK4: 4}.get(cfg.integrator, 1)
    every = max(1, args.exchange_every)
    g = D.ghost_depth(2 if cfg.stencil == W.LAP9X4 else 1, stages, every)
    slab = D.slab_of(cfg.ny, rank, world, g, bool(cfg.boundary))
    Z0 = np.ascontiguousarray(W.initial_state(cfg)[:, :, slab.global_rows(), :])
    alloc = lambda n: torch.empty((cfg.batch, cfg.n_v, n, cfg.nx), dtype=torch.float64, device="cuda")
    with C.Context(cfg.model, cfg.nx, slab.ext_rows, cfg.dx, cfg.dt, cfg.scheme, cfg.batch,
                   plan=args.plan, plan_param=args.plan_param) as ctx:
        ctx.set_state(Z0)
        exchange = lambda: D.exchange_dist(ctx, slab, alloc)
        for _ in range(args.warmup):
            D.advance_slab(ctx, slab, cfg.nsteps, every, exchange)
            exchange()
        torch.cuda.synchronize(); D.barrier()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = ctx.launches
        a.record()
        for _ in range(args.steps):
            D.advance_slab(ctx, slab, cfg.nsteps, every, exchange)
            exchange()                          # the next run starts from fresh ghosts
        b.record()
        torch.cuda.synchronize(); D.barrier()
        ms = D.max_over_ranks(a.elapsed_time(b))
        launches = ctx.launches - l0
        own = ctx.get_rows(slab.g_lo, slab.own)
    if not np.all(np.isfinite(own)):
        raise RuntimeError("non-finite state after the timed run")
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": cfg.cells * cfg.nsteps * args.steps / (ms * 1e-3) / 1e9, "unit": UNIT,
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
            "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.describe(), "parallelism": f"row slabs x{world}, {g} ghost rows per cut, "
                       f"one exchange per {every} time step(s)", "rows_per_rank": slab.own},
            "gpu_launches": int(launches)}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config, 1-based (default 2 = configs[1])")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--plan", type=int, default=0, help="CARDIAC_PLAN_* (0 = auto)")
    ap.add_argument("--plan-param", type=int, default=0)
    ap.add_argument("--nsteps", type=int, default=0, help="override the config's time steps per run (profiling only)")
    ap.add_argument("--no-extras", action="store_true", help="skip cpu_baseline, e2e and the other configs")
    ap.add_argument("--sweep", action="store_true", help="size sweep S of SURVEY.md 8(d) instead of the bench line")
    ap.add_argument("--decompose", default="replicas", choices=["replicas", "slabs"],
                    help="N > 1: independent replicas (default, weak scaling) or ONE grid in row slabs (strong)")
    ap.add_argument("--exchange-every", type=int, default=1, help="slabs: time steps between ghost exchanges")
    args = ap.parse_args()
    if args.warmup < 3 and not args.no_extras:
        args.warmup = 3                         # timing rule: W >= 3

    cfg = W.baseline_config(args.config)
    if args.nsteps:
        import dataclasses
        cfg = dataclasses.replace(cfg, nsteps=args.nsteps)
    rank, local_rank, world = D.env_world()

    if args.impl == "reference":
        run_reference(args, cfg, rank)
        return
    if args.sweep:
        if rank == 0:
            run_sweep(args)
        return

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the product has no CPU fallback)")
    if args.decompose == "slabs":
        run_slabs(args, cfg)
        return
    D.init("nccl")
    torch.cuda.set_device(local_rank)
    from paper_1309_1720_b200 import cardiac as C

    Z0 = W.initial_state(cfg)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    sampler = ClockSampler(local_rank)

    # ---- device-resident throughput (the headline `value`)
    sampler.start()
    ms, launches, plan_used = time_config(C, torch, cfg, Z0, args.steps, args.warmup, flush,
                                          args.plan, args.plan_param)
    clocks = sampler.stop()
    ms = D.max_over_ranks(ms)
    cell_steps_per_rank = cfg.cells * cfg.nsteps * args.steps
    value = world * cell_steps_per_rank / (ms * 1e-3) / 1e9

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_extras:
        zin = torch.from_numpy(Z0).pin_memory()
        zout = torch.empty_like(zin).pin_memory()
        with C.Context.from_config(cfg, plan=args.plan, plan_param=args.plan_param) as ctx:
            for _ in range(2):
                ctx.set_state(zin); ctx.step(cfg.nsteps); ctx.get_state(zout)
            D.barrier(); torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(args.steps):
                ctx.set_state(zin)              # H2D of this step's input
                ctx.step(cfg.nsteps)
                ctx.get_state(zout)             # D2H of this step's result
            b.record()
            torch.cuda.synchronize(); D.barrier()
            ms_e2e = D.max_over_ranks(a.elapsed_time(b))
        e2e = {"value": world * cell_steps_per_rank / (ms_e2e * 1e-3) / 1e9, "unit": UNIT,
               "h2d_bytes_per_step": int(zin.numel() * 8), "d2h_bytes_per_step": int(zout.numel() * 8)}

    if rank != 0:
        return

    # ---- roofline of the dominant kernel (live CUDA-event time / launches in the timed region)
    peak, peak_src = measured_peaks()
    algo_b = algo_bytes_per_cell_step(cfg)
    per_launch_bytes = algo_b * cfg.cells * cfg.nsteps * args.steps / max(launches, 1)
    per_launch_s = ms * 1e-3 / max(launches, 1)
    achieved = per_launch_bytes / per_launch_s / 1e9
    plan_name = PLAN_NAMES.get(plan_used, str(plan_used))
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": recorded_traffic(cfg, plan_name),
                "peak_source": peak_src, "algorithmic_bytes_per_cell_step": algo_b,
                "bytes_per_launch": per_launch_bytes, "us_per_launch": per_launch_s * 1e6,
                "floor_bytes_per_cell_step": floor_bytes_per_cell_step(cfg),
                "frac_of_fused_floor": (floor_bytes_per_cell_step(cfg) * cfg.cells * cfg.nsteps * args.steps
                                        / (ms * 1e-3) / 1e9) / peak,
                "fp64": fp64_view(cfg, value),
                "note": ("state is L2-resident within a step for this config (working set "
                         f"{cfg.cells * cfg.n_v * 8 / 2**20:.0f} MiB per buffer set): frac > 1 is possible and "
                         "means less DRAM traffic than the stage-synchronous count")
                if cfg.cells * cfg.n_v * 8 * 4 < 100 << 20 else "streaming working set"}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.describe(), "plan": plan_name,
                   "l2": "flushed between timed steps (256 MiB write); within a step the workload itself is "
                         "10^3-10^4 dependent time steps over the same state",
                   "parallelism": f"replicas x{world} (no data-path collective)" if world > 1 else "single GPU",
                   "dt": cfg.dt, "dx": cfg.dx},
        "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline,
    }
    if e2e:
        out["e2e"] = e2e

    if not args.no_extras and world == 1:
        rate, threads, n, secs = oracle_rate(cfg, Z0, 12.0)
        out["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": threads, "kind": "oracle",
                               "sample": f"first {n} of {cfg.nsteps} time steps of {cfg.describe()} "
                                         f"({secs:.1f} s of CPU time)"}
        # the other BASELINE configs, one run each (context for the roofline table; not bench lines)
        others = []
        for i in (1, 3, 4, 5):
            if i == args.config:
                continue
            c = W.baseline_config(i)
            try:
                z = W.initial_state(c)
                m, l, p = time_config(C, torch, c, z, 1, 1, flush)
                v = c.cells * c.nsteps / (m * 1e-3) / 1e9
                others.append({"workload": c.describe(), "plan": PLAN_NAMES.get(p, str(p)), "value": v,
                               "unit": UNIT, "ms": m, "launches": int(l),
                               "hbm_frac_stage_sync": v * algo_bytes_per_cell_step(c) / peak})
            except Exception as ex:  # keep the headline line even if an extra config fails
                others.append({"workload": c.describe(), "error": str(ex)})
        out["other_configs"] = others
    print(json.dumps(out))


if __name__ == "__main__":
    main()
