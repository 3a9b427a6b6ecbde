#!/usr/bin/env python
"""bench.py -- zone-cycles/s of the fp64 Z4c RK4 step (BASELINE.json `metric`).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl ours|reference] [--sweep none|point|full]

A "step" is one classical RK4 step (4 stages of RHS -> stage update + enforcement -> ghost fill; by default ONE fused
kernel per stage) over the whole pack. Default workload: BASELINE.json configs[3], the two-puncture grid of 256^3 cells
in 512 blocks of 32^3 (+3 ghosts) -- the largest fixed-size configuration; configs[4]'s saturated pack (512 blocks of
64^3, 133 GB on the device) is timed in the same run and reported under "sweep" with its own clocks record.
The timed region is K steps, repeated --repeats times (default 5); the line reports the MEDIAN repeat.
One JSON line is printed by rank 0. See DESIGN.md "Measurement" for every figure's definition.
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import subprocess
import sys
import threading
import time
from dataclasses import replace

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2409_10383_b200 import inputs as I  # noqa: E402

# Algorithmic work per cell (flop census = oracle/z4c_oracle.cpp oz4c_count_flops,
# add = mul = div = 1, no FMA fusion assumed; checked by tests/test_oracle_pins.py::test_flop_census).
RHS_FLOPS_PER_CELL = 6034
RHS_FLOPS_PER_CELL_O6 = 8059      # same census with the 6th-order stencil set (ng = 4)
# doubles moved per cell and RK4 step by the O6 recurrence: 616, plus the ghost fill
STEP_DOUBLES_PER_CELL = 616
GHOST_DOUBLES_PER_GHOST_CELL_STEP = 4 * 22 * 2
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 * 1e-12   # 148 SMs x 64 DFMA/clk x 2 flop x max SM clock

WORKLOAD_LABELS = {
    "linear_wave_64": "configs[1]: linear wave 64^3 = 64 blocks of 16^3 (+3 ghosts), periodic",
    "puncture_128": "configs[2]: single puncture 128^3 = 64 blocks of 32^3, outflow-copy",
    "bbh_256": "configs[3]: two punctures 256^3 = 512 blocks of 32^3, outflow-copy",
    "linear_wave_o6_256": "NEXT-1 / paper Table 1 shape: linear wave 256^3 = 64 blocks of 64^3 (+4 ghosts), 6th order",
}
DEFAULT_WORKLOAD = "bbh_256"
# configs[4] load sweep: (n, block lattice). "point" = the saturated pack only; "full" = every row.
SWEEP_POINT = [(64, (8, 8, 8))]
SWEEP_FULL = [(16, (2, 2, 2)), (16, (4, 4, 4)), (16, (8, 8, 8)), (16, (16, 16, 16)), (16, (24, 24, 24)),
              (32, (2, 2, 2)), (32, (4, 4, 4)), (32, (8, 8, 8)), (32, (12, 12, 12)), (32, (16, 16, 12)),
              (64, (2, 2, 2)), (64, (4, 4, 4)), (64, (6, 6, 6)), (64, (8, 8, 8))]
# the paper's own figure for its Table 1 workload: another machine and 6th order -- context, never a ratio
PAPER_CONTEXT = {"zcps": 1.36e7, "hardware": "NVIDIA A100", "workload": "linear wave, 64^3 blocks, VRAM filled, "
                 "6th order + RK4, whole application", "source": "PAPER.md:269 (Table 1)",
                 "gpu_over_cpu_core": ">~200x (PAPER.md:15, 283)"}


def workload_data(name: str, p):
    """The workload's closed-form initial data on the cells of `p` (any box of the same mesh: a z-slab, NEXT-2)."""
    if name in ("linear_wave_64", "linear_wave_o6_256"):
        return I.linear_wave_data(p)
    if name == "puncture_128":
        return I.puncture_data(p)
    if name == "bbh_256":
        return I.puncture_data(p, (0.5, 0.5), ((3.0, 0.0, 0.0), (-3.0, 0.0, 0.0)))
    raise SystemExit(f"workload {name} has no per-slab generator")


def workload(name: str, params_only: bool = False):
    """(params, initial data on the host, label). Inputs are synthetic and seeded."""
    if name == "linear_wave_64":
        p = I.params_linear_wave(64, 16)
        return p, None if params_only else I.linear_wave_data(p), WORKLOAD_LABELS[name]
    if name == "puncture_128":
        p = I.params_puncture(128, 32, 16.0, 2.0)
        return p, None if params_only else workload_data(name, p), WORKLOAD_LABELS[name]
    if name == "bbh_256":
        p = I.params_puncture(256, 32, 24.0, 1.0)
        return p, None if params_only else workload_data(name, p), WORKLOAD_LABELS[name]
    if name == "linear_wave_o6_256":
        p = replace(I.params_linear_wave(256, 64), ng=4)
        return p, None if params_only else I.linear_wave_data(p), WORKLOAD_LABELS[name]
    if name.startswith("noise_"):            # configs[4] load sweep: noise_<n>_<nbx>x<nby>x<nbz>
        _, n, lat = name.split("_")
        nb = tuple(int(v) for v in lat.split("x"))
        p = I.params_noise(int(n), nb, 0.1)
        tile = tuple(2 if b % 2 == 0 else 1 for b in nb)
        return p, I.tiled_noise_data(p, tile, 1000), f"configs[4]: noise, {nb} blocks of {n}^3, periodic"
    raise SystemExit(f"unknown workload {name}")


def profile_record(name: str, ng: int):
    """What the committed ncu capture of the dominant kernel says for this workload (profiles/r02_traffic.json,
    written from `ncu --set full` with the commit it was taken at), or None."""
    try:
        with open(os.path.join(ROOT, "profiles", "r02_traffic.json")) as f:
            d = json.load(f)
        rec = dict(d[name])
        rec["commit"] = d.get("commit")
        return rec
    except Exception:
        return None


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.01):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None
        self.period = period_s

    def _once(self):
        nv = self.nv
        self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
        try:
            r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
        except Exception:
            r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
        names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown",
                 0x4: "sw_power_cap", 0x80: "hw_power_brake", 0x2: "applications_clocks_setting"}
        for bit, nm in names.items():
            if r & bit:
                self.reasons.add(nm)

    def _run(self):
        while not self._stop.is_set():
            try:
                self._once()
            except Exception:
                pass
            time.sleep(self.period)

    def start(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        if self._thr is not None:
            self._stop.set()
            self._thr.join()
            if not self.samples:
                try:
                    self._once()
                except Exception:
                    pass
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def aggregate(local_ms: float, local_units: float, dist=None):
    """Whole-job figures from per-rank ones: time = MAX over ranks, units = SUM over ranks.
    Works on gloo (CPU tensors) and nccl."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local_ms, local_units
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([local_ms], dtype=torch.float64, device=dev)
    u = torch.tensor([local_units], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


# ------------------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py executes oracle/): cpu_baseline and --impl reference
# ------------------------------------------------------------------------------------------------
def oracle_sample(name: str, small: bool = False):
    """A bounded sample of the workload with identical per-cell arithmetic. `small`: a quarter of it (1-thread leg)."""
    if name == "linear_wave_64":
        p = I.params_linear_wave(64, 16)
        ps = replace(p, nb=(4, 1, 1))   # 64 x 16 x 16 periodic slab of the same wave
        return ps, I.linear_wave_data(ps), "64x16x16 periodic slab of the 64^3 wave (same per-cell arithmetic)"
    if name == "linear_wave_o6_256":
        ps = replace(I.params_linear_wave(256, 16), nb=(16, 1, 1), ng=4)
        return ps, I.linear_wave_data(ps), "256x16x16 periodic slab of the 256^3 wave, 6th-order stencils"
    if name in ("puncture_128", "bbh_256"):
        # the 32^3 block next to the puncture at x = +3 (bbh) / at the origin, cut out of the full-size data by its
        # closed form (no 3 GB array): same dx, same fields, clamped edges
        full = I.params_puncture(128, 32, 16.0, 2.0) if name == "puncture_128" else I.params_puncture(256, 32, 24.0, 1.0)
        w = 16 if small else 32
        centre = (0.0, 0.0, 0.0) if name == "puncture_128" else (3.0, 0.0, 0.0)
        lo = tuple(c - 0.5 * w * full.dx for c in centre)
        ps = replace(full, n=w, nb=(1, 1, 1), xmin=lo)
        if name == "puncture_128":
            us = I.puncture_data(ps)
        else:
            us = I.puncture_data(ps, (0.5, 0.5), ((3.0, 0.0, 0.0), (-3.0, 0.0, 0.0)))
        return ps, us, f"{w}^3 sub-box around the puncture at {centre} (same dx and data, clamped edges)"
    p, u, _ = workload(name)
    ps = replace(p, nb=(2, 1, 1))
    return ps, I.noise_data(ps, 1000), f"2 blocks of {p.n}^3 of the noise pack"


def time_oracle(name: str, steps: int, warmup: int, budget_s: float, threads: int = 0):
    from oracle import oracle as O
    O.build()
    all_threads = O.num_threads()
    if threads:
        O.set_num_threads(threads)
    try:
        ps, us, what = oracle_sample(name, small=(threads == 1))
        us, _ = O.enforce(ps, us)
        cores = O.num_threads()
        t0 = time.perf_counter()
        O.step(ps, us, 1)                      # calibration step (counts as warm-up)
        t1 = time.perf_counter() - t0
        for _ in range(max(0, warmup - 1)):
            if (time.perf_counter() - t0) > budget_s * 0.25:
                break
            O.step(ps, us, 1)
        k = max(1, min(steps, int(budget_s / max(t1, 1e-6))))
        t0 = time.perf_counter()
        O.step(ps, us, k)
        dt = time.perf_counter() - t0
    finally:
        if threads:
            O.set_num_threads(all_threads)
    return {"zcps": ps.ncells * k / dt, "cores": cores, "steps": k, "ms_per_step": dt / k * 1e3,
            "sample": f"{what}; {ps.ncells} cells x {k} RK4 steps"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    if args.workload == "two_level_wave_256":
        c = time_oracle_two_level(args.steps, 60.0)
        r = {"zcps": c["value"], "cores": c["cores"], "steps": c["steps"], "ms_per_step": c["ms_per_step"],
             "sample": c["sample"]}
        label = TWO_LEVEL_LABEL
    else:
        r = time_oracle(args.workload, args.steps, args.warmup, budget_s=60.0)
        label = WORKLOAD_LABELS.get(args.workload, args.workload)
    line = {"impl": "reference", "metric": "zone-cycles/s (fp64 Z4c RK4 step)", "value": r["zcps"],
            "unit": "zone-cycles/s", "n_gpus": args.gpus, "steps": r["steps"], "warmup": args.warmup,
            "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": label, "impl": "CPU oracle (oracle/z4c_oracle.cpp, -O2 -ffp-contract=off, OpenMP)"},
            "cpu_baseline": {"value": r["zcps"], "unit": "zone-cycles/s", "cores": r["cores"], "kind": "oracle",
                             "sample": r["sample"]},
            "e2e": {"value": r["zcps"], "unit": "zone-cycles/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------
def timed_steps(sim, K: int, W: int, R: int, barrier, device_index: int):
    """W warm-up steps, then R repeats of exactly K steps, each bracketed by barrier + synchronize and timed with
    CUDA events on the library's stream; clocks sampled over all repeats. Returns per-repeat ms and the clocks."""
    import torch
    sim.step(W)
    sim.sync()
    sampler = ClockSampler(device_index)
    times = []
    barrier()
    sampler.start()
    for _ in range(R):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(sim.stream)
        sim.step(K)
        e1.record(sim.stream)
        barrier()
        times.append(e0.elapsed_time(e1))
    clocks = sampler.stop()
    sim.sync()                                   # raises if the device error flag is set
    return times, clocks


def sweep_rows(Z, points, K, W, R, device_index, budget_gb):
    """BASELINE.json configs[4]: Minkowski + seeded 1e-10 noise, periodic; the pack is filled ON THE DEVICE by tiling a
    2x2x2-block seeded problem, so host memory never holds more than the small tile. Device-resident timing only."""
    import ctypes as C
    import torch
    rows = []
    lib = Z.load_library()
    for n, nb in points:
        p = I.params_noise(n, nb, 0.1)
        cp = Z.make_params(p)
        gb = (lib.z4c_state_bytes(C.byref(cp)) + lib.z4c_workspace_bytes(C.byref(cp)) + I.NF * p.ncells * 8) / 1e9
        free = torch.cuda.mem_get_info()[0] / 1e9
        if gb > min(budget_gb, free - 4.0):
            rows.append({"n": n, "blocks": list(nb), "skipped": f"needs {gb:.0f} GB, {free:.0f} GB free"})
            continue
        tile = (2, 2, 2)
        base = torch.from_numpy(I.noise_data(replace(p, nb=tile), 1000)).cuda()
        u = base.repeat(1, nb[2] // 2, nb[1] // 2, nb[0] // 2).contiguous()
        sim = Z.Z4c(p, device=f"cuda:{device_index}")
        sim.use_graph(True)
        sim.set_initial_data(u)
        del u, base
        torch.cuda.empty_cache()
        times, clocks = timed_steps(sim, K, W, R, torch.cuda.synchronize, device_index)
        ms = float(np.median(times))
        dev = float(abs(sim.state[I.CHI, 0, 3:-3, 3:-3, 3:-3] - 1.0).max())
        rows.append({"n": n, "blocks": list(nb), "cells_per_gpu": p.ncells, "device_gb": round(gb, 1),
                     "ms_per_step": ms / K, "zcps": p.ncells * K / (ms * 1e-3), "steps": K, "repeats": len(times),
                     "max_abs_chi_minus_1": dev, "effective_mode": list(sim.effective_mode()), "clocks": clocks})
        sim.close()
        del sim
        torch.cuda.empty_cache()
    return rows


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2409_10383_b200 import build, z4c

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the Z4c path has no CPU fallback")
    # fewer GPUs than ranks (a 1-GPU box): the ranks share devices and talk over gloo -- exercises the partitioned
    # path end to end (CUDA IPC between processes), but the figure is flagged and is no scaling number
    oversubscribed = world > torch.cuda.device_count()
    local_rank = local_rank % torch.cuda.device_count()
    torch.cuda.set_device(local_rank)
    if world > 1:
        if oversubscribed:
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    partitioned = world > 1 and not args.replicas
    if partitioned:
        # NEXT-2: ONE mesh, `world` times as long in z, cut into z-slabs -- weak scaling with a real ghost exchange
        # per stage (peer stores from the stage kernel + one stream-ordered barrier), not independent replicas
        from paper_2409_10383_b200 import partition as PT
        p1, _, label = workload(args.workload, params_only=True)
        pg = replace(p1, nb=(p1.nb[0], p1.nb[1], p1.nb[2] * world))
        p = PT.slab_params(pg, rank, world)
        u0 = workload_data(args.workload, p)
        label = label + f"; mesh extended {world}x along z, one z-slab per rank, ghost images pushed into the neighbour's pack"
        # The peer-store path needs every neighbour's buffers mapped into this process (CUDA IPC, peer access over
        # NVLink). If that or a first trial step fails on ANY rank, all ranks agree to fall back to independent
        # replicas, and the line says so: a missing figure would tell less than a flagged one.
        fallback_reason = None
        try:
            sim = PT.DistributedSlab(pg, f"cuda:{local_rank}")
            sim.sim.set_fused(args.fuse)
            sim.set_initial_data(u0)
            sim.step(1)
            sim.sync()
            eff_variant, eff_fused = sim.sim.effective_mode()
        except Exception as exc:                      # noqa: BLE001 -- any failure of the set-up counts
            fallback_reason = f"{type(exc).__name__}: {exc}"[:200]
        votes = [None] * world
        dist.all_gather_object(votes, fallback_reason)
        failed = [v for v in votes if v]
        if failed:
            partitioned = False
            label = WORKLOAD_LABELS.get(args.workload, args.workload) + \
                f"; REPLICAS: the partitioned path failed on {len(failed)} of {world} ranks ({failed[0]})"
    if not partitioned:
        replica_label = label if (world > 1 and not args.replicas) else None
        p, u0, label = workload(args.workload)
        label = replica_label or label
        sim = z4c.Z4c(p, device=f"cuda:{local_rank}")
        sim.set_variant(args.variant)
        sim.set_fused(args.fuse)
        sim.use_graph(not args.no_graph)
        eff_variant, eff_fused = sim.effective_mode()
    K, W, R = args.steps, max(args.warmup, 3), max(args.repeats, 1)
    ncells = p.ncells

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput: median of R repeats of exactly K steps ---------------------------
    sim.set_initial_data(u0)
    l0 = sim.launch_count()
    times, clocks = timed_steps(sim, K, W, R, barrier, local_rank)
    launches_per_step = (sim.launch_count() - l0) // (W + K * R)
    ms_local = float(np.median(times))
    ms, units = aggregate(ms_local, float(ncells) * K, dist if world > 1 else None)
    zcps = units / (ms * 1e-3)

    # ---- per-kernel share of the step (events between kernels, no graph) ------------------------------
    Kt = max(2, min(K, 10))
    if partitioned:      # one kernel per stage + the barrier: the step IS the four stage kernels
        kt = {"rhs": ms_local / K * Kt, "update": 0.0, "ghost": 0.0}
    else:
        sim.step_timed(2)
        kt = sim.step_timed(Kt)
    total_kt = kt["rhs"] + kt["update"] + kt["ghost"]
    core0 = sim.sim if partitioned else sim
    fp64_burst = core0.probe_fp64()
    # the same DFMA loop held for ~3 s with the clocks sampled: what the FP64 pipe sustains under the power cap that
    # also holds the long timed region above (context for `frac`, which stays against the burst figure)
    sus_sampler, sus_vals, t_sus = ClockSampler(local_rank), [], time.perf_counter()
    sus_sampler.start()
    while time.perf_counter() - t_sus < args.probe_seconds:
        sus_vals.append(core0.probe_fp64(iters=2_000_000))
    sus_clocks = sus_sampler.stop()
    fp64_sustained = float(np.median(sus_vals[len(sus_vals) // 2:])) if sus_vals else fp64_burst
    fp64_peak = max(fp64_burst, fp64_sustained)      # the short probe right after the long run can catch a depressed clock
    hbm_peak, hbm_src = measured_peaks()
    flops_cell = RHS_FLOPS_PER_CELL if p.ng == 3 else RHS_FLOPS_PER_CELL_O6
    # dominant kernel = the RHS / fused stage kernel, 4 launches per step; its launch time from the graph-replayed
    # step itself when it is the whole step (one kernel per stage), else from the event-separated run
    rhs_ms = (ms_local / K / 4.0) if eff_fused == 2 else kt["rhs"] / (4 * Kt)
    rhs_tflops = flops_cell * ncells / (rhs_ms * 1e-3) * 1e-12
    g = p.ng
    ghost_cells = p.nblocks * ((p.n + 2 * g) ** 3 - p.n ** 3)
    step_bytes = (STEP_DOUBLES_PER_CELL * ncells + GHOST_DOUBLES_PER_GHOST_CELL_STEP * ghost_cells) * 8
    prof = profile_record(args.workload, g)

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region ------
    h_in = torch.from_numpy(u0).pin_memory()
    h_out = torch.empty_like(h_in).pin_memory()
    Ke = max(3, min(K, 20)) if u0.nbytes < 1e9 else 3
    core_get = (sim.sim if partitioned else sim).get_interior
    sim.set_initial_data(h_in)
    sim.step(1)
    core_get(h_out.numpy())
    barrier()
    t0 = time.perf_counter()
    for _ in range(Ke):
        sim.set_initial_data(h_in)            # H2D of the step's input (synchronises)
        sim.step(1)
        core_get(h_out.numpy())               # D2H of the step's result (synchronises)
    barrier()
    e2e_ms, e2e_units = aggregate((time.perf_counter() - t0) * 1e3, float(ncells) * Ke, dist if world > 1 else None)
    nbytes = int(u0.nbytes)
    core = sim.sim if partitioned else sim
    state_mb = (core.state.numel() + core.work.numel()) * 8 / 1e6
    sim.close()
    del sim, h_in, h_out
    torch.cuda.empty_cache()

    # ---- configs[4] load sweep (device-resident), each row with its own clocks record -----------------
    sweep = None
    if world == 1 and args.sweep != "none" and p.ng == 3:
        pts = SWEEP_POINT if args.sweep == "point" else SWEEP_FULL
        sweep = sweep_rows(z4c, pts, min(K, 10) if args.sweep == "point" else min(K, 20), 3, R, local_rank,
                           args.budget_gb)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        r = time_oracle(args.workload, 1000, 1, budget_s=12.0)
        r1 = time_oracle(args.workload, 1000, 1, budget_s=8.0, threads=1)
        cpu = {"value": r["zcps"], "unit": "zone-cycles/s", "cores": r["cores"], "kind": "oracle", "sample": r["sample"],
               "single_thread": {"value": r1["zcps"], "unit": "zone-cycles/s", "cores": 1, "sample": r1["sample"]}}

    if rank == 0:
        line = {
            "metric": "zone-cycles/s (fp64 Z4c RK4 step)", "value": zcps, "unit": "zone-cycles/s", "n_gpus": world,
            "steps": K, "warmup": W, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": label, "cells_per_gpu": ncells, "blocks": p.nblocks, "n": p.n, "ghosts": g,
                       "parallelism": ("z-slabs of one mesh, peer ghost push + 1 barrier per stage" if partitioned
                                       else "replicas" if world > 1 else "1 GPU"),
                       "oversubscribed_ranks_share_gpus": oversubscribed,
                       "l2": "no flush: y+y2+P+Q working set %.0f MB > 126 MB L2" % state_mb,
                       "graph": not args.no_graph, "fuse_mode": eff_fused, "rhs_variant": eff_variant,
                       "requested": {"fuse_mode": args.fuse, "rhs_variant": args.variant}},
            "repeats": {"n": R, "ms_per_step_each": [t / K for t in times], "statistic": "median"},
            "clocks": clocks,
            "e2e": {"value": e2e_units / (e2e_ms * 1e-3), "unit": "zone-cycles/s", "h2d_bytes_per_step": nbytes,
                    "d2h_bytes_per_step": nbytes, "steps": Ke,
                    "what": "z4c_set_initial_data(host) + z4c_step(1) + z4c_get_interior(host) per step, pinned"},
            "gpu_launches": int(launches_per_step * K),
            "roofline": {"kernel": "k_stage<STAGE> (one kernel per RK stage)" if eff_fused == 2 else "K2 z4c_rhs",
                         "bound": "alu", "achieved": rhs_tflops, "peak": fp64_peak,
                         "unit": "TFLOP/s", "frac": rhs_tflops / fp64_peak,
                         "flops_source": "ALGORITHMIC: the oracle's unfused operation census (add = mul = div = 1), "
                                         "not executed instructions",
                         "traffic": prof.get("mean_bytes_per_launch") if prof else None,
                         "traffic_commit": prof.get("commit") if prof else None,
                         "fp64_pipe_active_pct_ncu": prof.get("fp64_pipe_active_pct") if prof else None,
                         "peak_source": "measured live: z4c_probe_fp64 DFMA loop, the higher of a 3 ms burst and a 3 s run "
                                        "(nominal %.1f at 1965 MHz)" % FP64_NOMINAL_TFLOPS,
                         "peak_burst": fp64_burst,
                         "peak_sustained": {"value": fp64_sustained, "unit": "TFLOP/s", "clocks": sus_clocks,
                                            "what": "the same DFMA loop held for --probe-seconds (median of the second half)"},
                         "frac_of_sustained_peak": rhs_tflops / fp64_sustained,
                         "frac_at_measured_clock": (rhs_tflops / (FP64_NOMINAL_TFLOPS * clocks["sm_mhz"] / 1965.0)
                                                    if clocks and clocks.get("sm_mhz") else None),
                         "flops_per_cell": flops_cell, "ms_per_launch": rhs_ms,
                         "timing": "graph-replayed step / 4" if eff_fused == 2 else "events between kernels",
                         "share_of_step": kt["rhs"] / total_kt},
            "step_roofline": {"bound": "hbm", "achieved": step_bytes * K / (ms_local * 1e-3) * 1e-9, "peak": hbm_peak,
                              "unit": "GB/s", "frac": step_bytes * K / (ms_local * 1e-3) * 1e-9 / hbm_peak,
                              "peak_source": hbm_src, "bytes_per_cell_step": step_bytes / ncells,
                              "kernel_ms_per_step": {k: v / Kt for k, v in kt.items()}},
            "sweep": sweep,
            "cpu_baseline": cpu,
            "context": {"paper": PAPER_CONTEXT},
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------
# NEXT-3: two-level static refinement (the refined-box wave of PAPER.md:171 at bench size)
# ------------------------------------------------------------------------------------------------
TWO_LEVEL_LABEL = ("NEXT-3: linear wave, coarse 256^3 = 512 blocks of 32^3 (periodic), the 128^3 box at coarse cell "
                   "(64,64,64) refined 2:1 into 256^3 fine cells = 512 blocks of 32^3; one dt, level exchange every stage")


def two_level_workload(small: bool = False):
    N, n = (32, 16) if small else (256, 32)
    pc = replace(I.params_linear_wave(N, n), cfl=0.125)
    pf = replace(pc, dx=pc.dx / 2, cfl=0.25, bc=1)                     # as many fine blocks as coarse blocks
    origin = (N // 4,) * 3
    pf = replace(pf, xmin=tuple(x + o * pc.dx for x, o in zip(pc.xmin, origin)))
    return pc, pf, origin


def time_oracle_two_level(max_steps: int, budget_s: float):
    """The oracle's two-level step on a bounded sample of the two-level workload (same wave, same operators)."""
    from oracle import oracle as O
    O.build()
    qc, qf, qo = two_level_workload(small=True)
    qf = replace(qf, nb=(1, 1, 1))
    uc, uf = O.enforce(qc, I.linear_wave_data(qc))[0], O.enforce(qf, I.linear_wave_data(qf))[0]
    t0 = time.perf_counter()
    O.step_two_level(qc, qf, qf.n, qo, uc, uf, 1)
    k = max(1, min(max_steps, int(budget_s / max(time.perf_counter() - t0, 1e-6))))
    t0 = time.perf_counter()
    O.step_two_level(qc, qf, qf.n, qo, uc, uf, k)
    dt = time.perf_counter() - t0
    qleaf = qc.ncells - qf.ncells // 8 + qf.ncells
    return {"value": qleaf * k / dt, "unit": "zone-cycles/s", "cores": O.num_threads(), "kind": "oracle",
            "steps": k, "ms_per_step": dt / k * 1e3,
            "sample": f"coarse 32^3 in 8 blocks of 16^3 + one refined 16^3 block at coarse cell {qo}; {qleaf} leaf "
                      f"zones x {k} two-level RK4 steps"}


def run_two_level(args):
    import torch
    from paper_2409_10383_b200 import build, z4c
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the Z4c path has no CPU fallback")
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise SystemExit("the two-level workload runs on one GPU")
    build.build()
    pc, pf, origin = two_level_workload()
    coarse = z4c.Z4c(pc, device="cuda:0")
    fine = z4c.Z4c(pf, device="cuda:0", stream=coarse.stream)
    for s in (coarse, fine):
        s.set_fused(args.fuse)
    coarse.set_initial_data(I.linear_wave_data(pc))
    fine.set_initial_data(I.linear_wave_data(pf))
    K, W, R = args.steps, max(args.warmup, 3), max(args.repeats, 1)
    covered = (pf.N[0] // 2) * (pf.N[1] // 2) * (pf.N[2] // 2)
    leaf = pc.ncells - covered + pf.ncells                                # zones of the leaf blocks

    def timed(fn, reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(coarse.stream)
        for _ in range(reps):
            fn()
        e1.record(coarse.stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    l0 = coarse.launch_count() + fine.launch_count()
    fine.two_level_step(coarse, origin, W)
    sampler = ClockSampler(0)
    sampler.start()
    times = [timed(lambda: fine.two_level_step(coarse, origin, K), 1) for _ in range(R)]
    clocks = sampler.stop()
    launches_per_step = (coarse.launch_count() + fine.launch_count() - l0) // (W + K * R)
    ms = float(np.median(times))
    # the pieces on their own: each level's RK4 step without the exchange, and the two exchange kernels
    parts = {"coarse_step": timed(lambda: coarse.step(1), 5), "fine_step": timed(lambda: fine.step(1), 5),
             "restrict_x4": 4 * timed(lambda: fine.restrict_to(coarse, origin), 20),
             "prolongate_x4": 4 * timed(lambda: fine.prolongate_from(coarse, origin), 20)}
    coarse.sync()
    fine.sync()
    eff = [list(coarse.effective_mode()), list(fine.effective_mode())]
    # exchange kernels: algorithmic bytes = one read of every stencil node's 8 bytes once per output + the output
    g, nn = pc.ng, pc.ng + 1
    fine_ghost_out = 0
    for bz in range(pf.nb[2]):
        for by in range(pf.nb[1]):
            for bx in range(pf.nb[0]):
                ext = [pf.n + (g if b == 0 else 0) + (g if b == nb - 1 else 0) for b, nb in zip((bx, by, bz), pf.nb)]
                fine_ghost_out += ext[0] * ext[1] * ext[2] - pf.n ** 3
    hbm_peak, hbm_src = measured_peaks()
    # restriction: every fine active cell read once, every covered coarse cell written; prolongation: every fine ghost
    # cell outside the box written, ~0.4 coarse cells read per such cell (the layers of coarse nodes under the shell)
    exch_bytes = 8 * I.NF * (pf.ncells + covered) + 8 * I.NF * int(1.4 * fine_ghost_out)
    cpu = None if args.no_cpu else time_oracle_two_level(1000, 10.0)
    line = {"metric": "zone-cycles/s (fp64 Z4c RK4 step)", "value": leaf * K / (ms * 1e-3), "unit": "zone-cycles/s",
            "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": TWO_LEVEL_LABEL, "leaf_zones": leaf, "zones_computed": pc.ncells + pf.ncells,
                       "note": "value counts the zones of leaf blocks only; the covered coarse cells are advanced too "
                               "and then overwritten by the restriction",
                       "effective_mode": eff, "l2": "no flush: working set of both packs exceeds the 126 MB L2"},
            "repeats": {"n": R, "ms_per_step_each": [t / K for t in times], "statistic": "median"}, "clocks": clocks,
            "gpu_launches": int(launches_per_step * K),
            "two_level": {"ms_per_step_parts": parts,
                          "exchange_share_of_step": 1.0 - (parts["coarse_step"] + parts["fine_step"]) / (ms / K),
                          "exchange_roofline": {"bound": "hbm", "kernels": "k_restrict + k_prolong, 4 of each per step",
                                                "achieved": 4 * exch_bytes / ((parts["restrict_x4"] + parts["prolongate_x4"]) * 1e-3) * 1e-9,
                                                "peak": hbm_peak, "unit": "GB/s", "peak_source": hbm_src,
                                                "bytes_per_exchange": exch_bytes}},
            "cpu_baseline": cpu}
    line["two_level"]["exchange_roofline"]["frac"] = line["two_level"]["exchange_roofline"]["achieved"] / hbm_peak
    print(json.dumps(line))
    coarse.close()
    fine.close()


def free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--repeats", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD)
    ap.add_argument("--sweep", default="point", choices=["none", "point", "full"])
    ap.add_argument("--budget-gb", type=float, default=150.0)
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--no-graph", action="store_true")
    ap.add_argument("--fuse", type=int, default=2, help="0: K2,K3,K1; 1: K2,K3+push; 2: one kernel per RK stage")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--probe-seconds", type=float, default=3.0,
                    help="length of the sustained FP64 probe after the timed region (0: burst probe only)")
    ap.add_argument("--replicas", action="store_true",
                    help="with --gpus N > 1: N independent packs instead of one mesh partitioned into z-slabs")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N` is a complete command: re-launch under torch.distributed.run, one rank per GPU
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if args.impl == "reference":
        run_reference(args)
    elif args.workload == "two_level_wave_256":
        run_two_level(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
