#!/usr/bin/env python
"""bench.py — FP64 cell-updates/s of the explicit cardiac time step on B200(s).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

One "step" = one pass of the whole hot path over the config's workload: ALL time steps of the chosen
BASELINE.json config, every time step being stencil + no-flux boundary + reaction + RK stages, plus
what the config itself does around them (config 4: the cross-field stimulus at step 500 through
get_state / edit / set_state; config 5: the 16 finite-difference Jacobian-vector products at the end).
Default = config 4, the largest single-GPU config: BOCF (the exp-heavy 4-field model),
2048 x 2048, 4th-order cross stencil, RK4, 2,000 time steps — the streaming regime the >= 70 % bar of
north_star applies to.  Prints ONE JSON line (rank 0); its `configs` list carries a full record
(own warm-up, repetitions, clocks, roofline with three denominators, CPU baseline) for each of the
other four BASELINE configs.  See DESIGN.md "Roofline accounting".
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
# "Roofline"); written by `python -m paper_1309_1720_b200.sass_count`, re-run whenever models.cuh /
# fastmath.cuh change (round 1, degree-13 exp and two-step reciprocal: Karma 220 / 342, BOCF 633 / 1045).
FP64_PER_CELL_STEP = {   # (model, stencil, integrator): (instructions, flops)
    (W.FHN, W.LAP5, W.EULER): (18, 26),
    (W.FHN, W.LAP9X4, W.RK4): (120, 170),
    (W.KARMA, W.LAP5, W.RK4): (188, 274),
    (W.BOCF, W.LAP9X4, W.RK4): (529.5, 825.5),
}
# nominal FP64 peak, for context only: 148 SM x 64 FP64 lanes/clk x 2 x 1.965 GHz (the measured one is
# taken live by cardiac_measure_fp64_peak, include/cardiac_diag.h)
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12


def floor_bytes_per_cell_step(cfg) -> int:
    return 16 * cfg.n_v   # read + write every field once, if all stages were fused on chip


def measured_peaks() -> tuple[float, str]:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json:hbm_gbs)"
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
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in open(self.path):
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 9:
                continue
            try:
                sm.append(float(parts[1])); mx.append(float(parts[2]))
            except ValueError:
                continue
            try:
                pw.append(float(parts[3]))
            except ValueError:
                pass
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
            if pw:
                out["power_w_max"] = max(pw)
        return out


# ----------------------------------------------------------------------------- the CPU baseline (oracle)
def oracle_rate(cfg, Z0, budget_s: float, omp: bool):
    """Time the oracle as it stands — its source compiled -O3 -march=native on this host (oracle.build_timing;
    SURVEY.md 8(d) "Oracle timing") — on a bounded sample of the same workload: the first time steps of ONE
    batch member on the config's grid.  Returns (Gcell-step/s, threads, time steps timed, seconds)."""
    import oracle as O
    one = Z0[:1]
    cells = cfg.nx * cfg.ny
    t = time.perf_counter()
    O.step(cfg.model, one, cfg.dx, cfg.dt, cfg.scheme, 1, omp=omp, timing=True)   # also pays the thread start-up
    dt1 = time.perf_counter() - t
    if dt1 * 10 < budget_s:
        t = time.perf_counter()
        O.step(cfg.model, one, cfg.dx, cfg.dt, cfg.scheme, 10, omp=omp, timing=True)
        dt1 = (time.perf_counter() - t) / 10
    n = max(1, int(budget_s / max(dt1, 1e-6)))
    t = time.perf_counter()
    O.step(cfg.model, one, cfg.dx, cfg.dt, cfg.scheme, n, omp=omp, timing=True)
    dt = time.perf_counter() - t
    return cells * n / dt / 1e9, O.threads(omp), n, dt


def cpu_baseline(cfg, Z0, budget_s: float) -> dict:
    """All host cores (the contract's `value`) and one thread, same build, same sample recipe."""
    import oracle as O
    r1, _, n1, s1 = oracle_rate(cfg, Z0, budget_s / 2, omp=False)
    ra, threads, na, sa = oracle_rate(cfg, Z0, budget_s / 2, omp=True)
    return {"value": ra, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": f"first {na} of {cfg.nsteps} time steps of {cfg.describe()}, one batch member "
                      f"({sa:.1f} s on {threads} threads)",
            "one_thread": {"value": r1, "unit": UNIT, "cores": 1,
                           "sample": f"first {n1} time steps ({s1:.1f} s)"},
            "build": "oracle/cardiac_oracle.c, gcc -O3 -march=native (-fopenmp for all cores)",
            "cpu": O.cpu_model()}


def oracle_initial_state(cfg):
    """--impl reference only: the config's initial state with the oracle itself integrating config 5's base."""
    if cfg.name != "cfg5":
        return W.initial_state(cfg)
    import oracle as O
    one, z2, n = W.base_recipe_cfg5(cfg)
    base = O.step(one.model, z2, one.dx, one.dt, one.scheme, n, omp=True, timing=True)[0]
    return W.initial_state(cfg, base=base)


def run_reference(args, cfg, rank):
    """--impl reference: the oracle (timing build, all host cores) on the same metric/config; each bench
    step is a bounded sample: a few time steps of the config's grid, about 3 s of CPU work."""
    if rank != 0:
        return
    import oracle as O
    Z0 = oracle_initial_state(cfg)
    rate, threads, n, secs = oracle_rate(cfg, Z0, 1.0, omp=True)
    per_step = max(1, int(n * 3.0 / max(secs, 1e-6)))
    one = Z0[:1]
    cells = cfg.nx * cfg.ny
    for _ in range(args.warmup):
        O.step(cfg.model, one, cfg.dx, cfg.dt, cfg.scheme, 1, omp=True, timing=True)
    t = time.perf_counter()
    z = one
    for _ in range(args.steps):
        z = O.step(cfg.model, z, cfg.dx, cfg.dt, cfg.scheme, per_step, omp=True, timing=True)
    total = time.perf_counter() - t
    value = cells * per_step * args.steps / total / 1e9
    sample = f"{per_step} of {cfg.nsteps} time steps of {cfg.describe()} per bench step (1 batch member)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 0,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(cfg, 1),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample,
                         "build": "oracle/cardiac_oracle.c, gcc -O3 -march=native -fopenmp", "cpu": O.cpu_model()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


PLAN_NAMES = {1: "stage", 2: "fused", 3: "persistent", 4: "pair"}


def workload_config(cfg, world):
    """The `config` object: the same keys and values for both arms."""
    return {"workload": cfg.describe(),
            "l2": "flushed between timed steps (256 MiB write); within a step the workload itself is "
                  "10^2-10^4 dependent time steps over the same state",
            "parallelism": f"replicas x{world} (no data-path collective)" if world > 1 else "single GPU",
            "dt": cfg.dt, "dx": cfg.dx}


# ----------------------------------------------------------------------------- one pass of a config's workload
def gpu_initial_state(C, cfg):
    """The config's initial state; config 5's base (the config-2 state after 5,000 RK4 steps,
    BASELINE.json:configs[4]) is integrated by the library itself, outside every timed region."""
    if cfg.name != "cfg5":
        return W.initial_state(cfg)
    one, z2, n = W.base_recipe_cfg5(cfg)
    with C.Context.from_config(one) as ctx:
        ctx.set_state(z2)
        ctx.step(n)
        base = ctx.get_state()[0]
    return W.initial_state(cfg, base=base)


class Workload:
    """One pass = everything the config does between its input and its output, state resident."""

    def __init__(self, C, torch, cfg, ctx, host: bool):
        self.C, self.torch, self.cfg, self.ctx, self.host = C, torch, cfg, ctx, host
        self.mid = None
        self.jvp = None
        shape = (cfg.batch, cfg.n_v, cfg.ny, cfg.nx)
        if cfg.name == "cfg4" and cfg.nsteps > 500:
            self.mid = torch.empty(shape, dtype=torch.float64, device="cpu" if host else "cuda")
            if host:
                self.mid = self.mid.pin_memory()
        if cfg.name == "cfg5":
            self.jvp = torch.empty((cfg.batch - 1,) + shape[1:], dtype=torch.float64,
                                   device="cpu" if host else "cuda")
            if host:
                self.jvp = self.jvp.pin_memory()

    def run(self):
        cfg, ctx = self.cfg, self.ctx
        if self.mid is not None:       # config 4: cross-field stimulus at step 500 via get / edit / set
            ctx.step(500)
            ctx.get_state(self.mid)
            W.stimulus_cfg4_inplace(self.mid)
            ctx.set_state(self.mid)
            ctx.step(cfg.nsteps - 500)
        else:
            ctx.step(cfg.nsteps)
        if self.jvp is not None:       # config 5: the output IS the 16 JVPs
            ctx.get_jvp(1e-7, self.jvp)


def time_config(C, torch, cfg, Z0, steps, warmup, flush, plan=0, plan_param=0):
    """Device-timed throughput of `steps` whole passes of cfg (state resident), L2 flushed between."""
    with C.Context.from_config(cfg, plan=plan, plan_param=plan_param) as ctx:
        zd = torch.from_numpy(Z0).cuda()
        wl = Workload(C, torch, cfg, ctx, host=False)
        for _ in range(warmup):
            ctx.set_state(zd)
            wl.run()
        torch.cuda.synchronize()
        l0 = ctx.launches
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        D.barrier()
        torch.cuda.synchronize()
        for a, b in ev:
            ctx.set_state(zd)                  # device-to-device, outside the event pair: every pass runs the same input
            flush.zero_()                      # > L2 (126 MB): evict the state between timed steps
            a.record()
            wl.run()
            b.record()
        torch.cuda.synchronize()
        D.barrier()
        times = [a.elapsed_time(b) for a, b in ev]
        launches = ctx.launches - l0
        plan_used = ctx.plan
        final = ctx.get_state()
    if not np.all(np.isfinite(final)):
        raise RuntimeError("non-finite state after the timed run")
    return sum(times), launches, plan_used, times


def time_e2e(C, torch, cfg, Z0, steps, plan=0, plan_param=0):
    """The same pass through the C ABI with HOST buffers: every step copies its input from pinned host
    memory (set_state), runs the workload (config 4's stimulus goes through the host too) and reads its
    result back (get_state; config 5: the JVPs).  Returns (ms, h2d bytes per step, d2h bytes per step)."""
    zin = torch.from_numpy(Z0).pin_memory()
    with C.Context.from_config(cfg, plan=plan, plan_param=plan_param) as ctx:
        wl = Workload(C, torch, cfg, ctx, host=True)
        zout = None if wl.jvp is not None else torch.empty_like(zin).pin_memory()

        def one():
            ctx.set_state(zin)              # H2D of this step's input
            wl.run()
            if zout is not None:
                ctx.get_state(zout)         # D2H of this step's result
        for _ in range(2):
            one()
        D.barrier(); torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(steps):
            one()
        b.record()
        torch.cuda.synchronize(); D.barrier()
        ms = D.max_over_ranks(a.elapsed_time(b))
    h2d = zin.numel() * 8 + (wl.mid.numel() * 8 if wl.mid is not None else 0)
    d2h = (wl.jvp.numel() * 8 if wl.jvp is not None else zout.numel() * 8) + (wl.mid.numel() * 8 if wl.mid is not None else 0)
    return ms, int(h2d), int(d2h)


def measure_fp64(C, cfg_small, gpu_index=0):
    """FP64-pipe peak of this GPU, measured now: a burst (best of 5 launches of ~15 ms) and a sustained
    figure (one ~0.5 s launch, the regime of a kernel timed inside a long step), clocks sampled."""
    with C.Context.from_config(cfg_small) as ctx:
        burst = C.cardiac_measure_fp64_peak(ctx.ctx, 4000, 5)
        sampler = ClockSampler(gpu_index)
        sampler.start()
        sustained = C.cardiac_measure_fp64_peak(ctx.ctx, 120000, 2)
        clocks = sampler.stop()
        # what an FP64 instruction costs a scheduler's issue port: DFMA rate with 0 / 2 / 4 independent integer
        # instructions between the DFMAs (cycles = 2 x FP64 + others)
        mhz = clocks.get("sm_mhz") or 1965.0
        issue = {}
        for m in (0, 2, 4):
            r = C.cardiac_measure_fp64_issue(ctx.ctx, m, 4000, 3)
            issue[str(m)] = {"dfma_per_s": r, "cycles_per_dfma_per_scheduler": 148 * 4 * 32 * mhz * 1e6 / r}
    return {"dfma_per_s_burst": burst, "dfma_per_s_sustained": sustained, "issue_port_probe": issue,
            "tflops_burst": 2 * burst / 1e12, "tflops_sustained": 2 * sustained / 1e12,
            "nominal_tflops": FP64_NOMINAL_TFLOPS, "clocks_sustained": clocks,
            "how": "cardiac_measure_fp64_peak (include/cardiac_diag.h): 148 x 4 CTAs x 256 threads x 8 independent "
                   "DFMA chains, registers only, CUDA events"}


def roofline_record(cfg, value, ms, launches, steps, plan_name, hbm_peak, hbm_src, fp64):
    """`roofline` of one config.  Unit = cell-step.  Three denominators (north_star: "the slower of
    bytes-per-cell-step over HBM bandwidth and FP64 flops-per-cell-step at peak"):
      stage-synchronous HBM bytes (one global dependency per RK stage) — the headline
      `achieved` / `frac`, per launch; the 16 n_v floor of a fully fused step; the measured FP64 pipe."""
    algo_b = algo_bytes_per_cell_step(cfg)
    cellsteps = cfg.cells * cfg.nsteps * steps
    per_launch_bytes = algo_b * cellsteps / max(launches, 1)
    per_launch_s = ms * 1e-3 / max(launches, 1)
    achieved = per_launch_bytes / per_launch_s / 1e9
    working_set = cfg.cells * cfg.n_v * 8 * (4 if cfg.integrator == W.RK4 else 2)
    resident = working_set < 100 << 20
    rec = {"bound": "hbm", "achieved": achieved, "peak": hbm_peak, "unit": "GB/s",
           "frac": achieved / hbm_peak, "traffic": recorded_traffic(cfg, plan_name),
           "peak_source": hbm_src, "algorithmic_bytes_per_cell_step": algo_b,
           "bytes_per_launch": per_launch_bytes, "us_per_launch": per_launch_s * 1e6,
           "launches_per_time_step": launches / max(cfg.nsteps * steps, 1),
           "floor_bytes_per_cell_step": floor_bytes_per_cell_step(cfg),
           "frac_of_fused_floor": floor_bytes_per_cell_step(cfg) * value / hbm_peak,
           "regime": ("L2-resident (working set %.0f MiB < 126 MB L2): frac is NOT an HBM statement here — no such "
                      "DRAM traffic exists; see traffic and fp64" % (working_set / 2**20)) if resident
                     else "streaming (working set %.0f MiB)" % (working_set / 2**20)}
    k = (cfg.model, cfg.stencil, cfg.integrator)
    if k in FP64_PER_CELL_STEP and fp64:
        instr, flops = FP64_PER_CELL_STEP[k]
        peak_i = fp64["dfma_per_s_sustained"]
        rec["fp64"] = {"achieved": value * flops / 1e3, "peak": 2 * peak_i / 1e12, "unit": "TFLOP/s",
                       "frac": value * 1e9 * instr / peak_i, "flops_per_cell_step": flops,
                       "fp64_instructions_per_cell_step": instr,
                       "frac_is": "algorithmic FP64 instructions per second / measured sustained DFMA rate",
                       "peak_source": "measured (cardiac_measure_fp64_peak, sustained)",
                       "peak_burst": 2 * fp64["dfma_per_s_burst"] / 1e12, "peak_nominal": FP64_NOMINAL_TFLOPS}
        # the slower of the two candidate bounds decides which roofline binds the stage-synchronous path
        t_hbm = algo_b / (hbm_peak * 1e9)
        t_fp = instr / peak_i
        rec["binding"] = "hbm" if t_hbm >= t_fp else "fp64"
        rec["frac_of_binding"] = max(t_hbm, t_fp) * value * 1e9
    return rec


def config_record(C, torch, cfg, steps, warmup, flush, hbm_peak, hbm_src, fp64, gpu_index, cpu_budget,
                  plan=0, plan_param=0):
    """A full record of one config: device-resident value with its own warm-up, repetitions and clock
    samples, roofline, end-to-end number and CPU baseline."""
    Z0 = gpu_initial_state(C, cfg)
    sampler = ClockSampler(gpu_index)
    sampler.start()
    ms, launches, plan_used, times = time_config(C, torch, cfg, Z0, steps, warmup, flush, plan, plan_param)
    clocks = sampler.stop()
    value = cfg.cells * cfg.nsteps * steps / (ms * 1e-3) / 1e9
    plan_name = PLAN_NAMES.get(plan_used, str(plan_used))
    ms_e, h2d, d2h = time_e2e(C, torch, cfg, Z0, max(1, min(steps, 3)), plan, plan_param)
    rec = {"workload": cfg.describe(), "plan": plan_name, "value": value, "unit": UNIT, "steps": steps,
           "warmup": warmup, "ms_per_step": ms / steps, "ms_min": min(times), "ms_max": max(times),
           "gpu_launches": int(launches), "clocks": clocks,
           "roofline": roofline_record(cfg, value, ms, launches, steps, plan_name, hbm_peak, hbm_src, fp64),
           "e2e": {"value": cfg.cells * cfg.nsteps * max(1, min(steps, 3)) / (ms_e * 1e-3) / 1e9, "unit": UNIT,
                   "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h}}
    if cpu_budget > 0:
        rec["cpu_baseline"] = cpu_baseline(cfg, Z0, cpu_budget)
    return rec


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
    Z0 = np.ascontiguousarray(gpu_initial_state(C, cfg)[:, :, slab.global_rows(), :])
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
    ap.add_argument("--config", type=int, default=4,
                    help="BASELINE.json config, 1-based (default 4 = configs[3], the largest single-GPU config)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--plan", type=int, default=0, help="CARDIAC_PLAN_* (0 = auto)")
    ap.add_argument("--plan-param", type=int, default=0)
    ap.add_argument("--nsteps", type=int, default=0, help="override the config's time steps per run (profiling only)")
    ap.add_argument("--no-extras", action="store_true", help="skip cpu_baseline, e2e, fp64 peak and the other configs")
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

    Z0 = gpu_initial_state(C, cfg)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    sampler = ClockSampler(local_rank)

    # ---- device-resident throughput (the headline `value`)
    sampler.start()
    ms, launches, plan_used, times = time_config(C, torch, cfg, Z0, args.steps, args.warmup, flush,
                                                 args.plan, args.plan_param)
    clocks = sampler.stop()
    ms = D.max_over_ranks(ms)
    cell_steps_per_rank = cfg.cells * cfg.nsteps * args.steps
    value = world * cell_steps_per_rank / (ms * 1e-3) / 1e9

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_extras:
        ms_e2e, h2d, d2h = time_e2e(C, torch, cfg, Z0, args.steps, args.plan, args.plan_param)
        e2e = {"value": world * cell_steps_per_rank / (ms_e2e * 1e-3) / 1e9, "unit": UNIT,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h}

    if rank != 0:
        return

    # ---- roofline of the dominant kernel (live CUDA-event time / launches in the timed region)
    hbm_peak, hbm_src = measured_peaks()
    fp64 = None if args.no_extras else measure_fp64(C, W.baseline_config(1), local_rank)
    plan_name = PLAN_NAMES.get(plan_used, str(plan_used))
    roofline = roofline_record(cfg, value / world, ms, launches, args.steps, plan_name, hbm_peak, hbm_src, fp64)

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg, world), "plan": plan_name,
        "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline,
        "ms_min": min(times), "ms_max": max(times),
    }
    if e2e:
        out["e2e"] = e2e
    if fp64:
        out["fp64_peak"] = fp64

    if not args.no_extras and world == 1:
        out["cpu_baseline"] = cpu_baseline(cfg, Z0, 8.0)
        # the other BASELINE configs: a full record each (own warm-up, repetitions, clocks, roofline, CPU baseline)
        others = []
        reps = max(3, min(args.steps, 5))
        for i in (1, 2, 3, 4, 5):
            if i == args.config:
                continue
            c = W.baseline_config(i)
            try:
                others.append(config_record(C, torch, c, reps, 3, flush, hbm_peak, hbm_src, fp64, local_rank, 5.0))
            except Exception as ex:  # keep the headline line even if an extra config fails
                others.append({"workload": c.describe(), "error": f"{type(ex).__name__}: {ex}"})
        out["configs"] = others
    print(json.dumps(out))


if __name__ == "__main__":
    main()
