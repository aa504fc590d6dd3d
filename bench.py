#!/usr/bin/env python
"""bench.py -- the headline measurement: fp64 cell-updates/s per RK stage of the convective RHS on one B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl b200|reference] [--workload config4|config2|config3|config5]

A "step" is one pass of the whole hot path over the workload, xf_step_cfl: the CFL max-wave-speed reduction (fused
into the first stage's primitives kernel) and three times (ghost fill, primitives, x/y/z sweeps with the flux
divergence and the fused SSP-RK3 stage combination).  One step is therefore 3 convective-RHS evaluations of every interior cell, and

    value = interior cells x 3 x K x N / time          [cell-updates/s per RK stage, whole job]

Default workload: BASELINE.json configs[3] (3-D 10-species shock-bubble, 512x256x256), the configuration the
north-star target is quoted on.  The state advances from step to step (a real simulation), inputs are synthetic
and seeded, each U copy is 4 GB >> the 126 MB L2, so no L2 flush is needed.

N > 1 (torchrun): the path has no exchange step on one GPU (replicas only), so every rank
runs an independent replica of the same problem, no data-path collective; timing is max over ranks; "weak".

--workload config5 is BASELINE.json configs[4] as it is stated there: 640x384x384 random states generated on the device,
a "step" = one convective-RHS evaluation with the temperature guess restored before it (outside the timed span), 50 of
them by default; not the bench line (config 4 is), for the record in DESIGN.md.

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample of the same
workload; it is a deliberately plain program -- parity and the roofline fraction are the headline, not that ratio.
"""
from __future__ import annotations

import argparse
import csv
import hashlib
import json
import os
import subprocess
import sys
import tempfile
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "fp64 cell-updates/s per RK stage (convective RHS)"
UNIT = "cell-updates/s"

WORKLOADS = {
    # name: (generator, full grid, grid of the bounded oracle sample for cpu_baseline, grid of a --impl reference step)
    "config4": ("config4_shock_bubble_3d_10sp", (512, 256, 256), (320, 160, 160), (128, 64, 64)),
    "config3": ("config3_shock_bubble_3d", (256, 256, 256), (128, 128, 128), (96, 96, 96)),
    "config2": ("config2_shock_bubble_2d", (2048, 1024, 1), (1024, 512, 1), (1024, 512, 1)),
    "config5": ("config5_random_states", (640, 384, 384), (128, 128, 128), (96, 96, 96)),
    "react": ("reacting_box", (256, 128, 128), (64, 32, 32), (64, 32, 32)),
}


def make_workload(name: str, grid):
    from paper_2403_05910_b200 import workloads as wl

    gen = getattr(wl, WORKLOADS[name][0])
    if name == "config3":
        return gen(grid[0])
    if name == "config2":
        return gen(grid[0], grid[1])
    return gen(*grid)


FP64_NOMINAL_TFLOPS = 37.2   # 148 SMs x 64 fp64 FMA lanes x 2 flop x 1.965 GHz


def flops_per_face(N: int) -> int:
    """Algorithmic fp64 flops of one face flux + its share of the divergence."""
    return 222 * N + 954


def flops_per_cell_rhs(N: int, D: int, newton_its: float) -> float:
    return D * flops_per_face(N) + 24 * N * newton_its + 3 * N + 40


def bytes_per_cell_rhs(N: int) -> int:
    """Compulsory HBM bytes of one RHS evaluation: read U, write rhs/U', read the T guess, write T."""
    return (2 * (N + 4) + 2) * 8


# ---------------------------------------------------------------------------------------------------------------
# clocks: nvidia-smi sampled DURING the timed region (B200_PROFILING.md "clocks line")
# ---------------------------------------------------------------------------------------------------------------
_CLK_FIELDS = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
               "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
               "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")


class ClockSampler:
    def __init__(self, gpu_index: int):
        self.path = Path(tempfile.gettempdir()) / f"xf_clocks_{os.getpid()}.csv"
        self.gpu = gpu_index
        self.proc = None

    def start(self):
        try:
            self.fh = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={_CLK_FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=self.fh,
                                         stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.fh.close()
        sm, smax, power, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.path.read_text().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1]))
                smax.append(float(f[2]))
                power.append(float(f[3]))
            except ValueError:
                continue
            for nm, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        try:
            self.path.unlink()
        except OSError:
            pass
        if sm:
            sm.sort()
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(smax), power_w_max=max(power), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


# ---------------------------------------------------------------------------------------------------------------
# the CPU oracle legs (cpu_baseline of the main arm; the whole --impl reference arm)
# ---------------------------------------------------------------------------------------------------------------
def oracle_threads() -> int:
    env = os.environ.get("OMP_NUM_THREADS")
    return int(env) if env and env.isdigit() else (os.cpu_count() or 1)


def oracle_step_seconds(w, steps: int, warmup: int = 0):
    """Times `steps` hot-path steps (max wave speed + one RK3 step = 3 RHS) of the oracle on workload w."""
    import oracle

    O = oracle.Oracle.from_workload(w)
    U, T = w.U.copy(), w.T_guess.copy()
    for _ in range(warmup):
        S = O.max_wavespeed(U, T)
        O.rk3_step(U, T, w.cfl / S)
    t0 = time.perf_counter()
    for _ in range(steps):
        S = O.max_wavespeed(U, T)
        O.rk3_step(U, T, w.cfl / S)
    return time.perf_counter() - t0


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def cpu_baseline(name: str) -> dict:
    grid = WORKLOADS[name][2]
    w = make_workload(name, grid)
    sec = oracle_step_seconds(w, 1)
    out = {"value": w.interior_cells * 3 / sec, "unit": UNIT, "cores": oracle_threads(), "kind": "oracle",
           "cpu": cpu_model(),
           "sample": f"1 step (max wave speed + RK3 = 3 RHS) of {name} generated at {grid[0]}x{grid[1]}x{grid[2]} "
                     f"(same set-up, reduced grid), {sec:.1f} s, oracle/xf_oracle.c with OpenMP"}
    # the one-thread figure on a smaller sample of the same set-up
    try:
        import ctypes

        gomp = ctypes.CDLL("libgomp.so.1")
        small = tuple(max(8, g // 4) for g in grid)
        w1 = make_workload(name, small)
        gomp.omp_set_num_threads(1)
        sec1 = oracle_step_seconds(w1, 1)
        gomp.omp_set_num_threads(oracle_threads())
        out["one_thread_value"] = w1.interior_cells * 3 / sec1
        out["one_thread_sample"] = f"{small[0]}x{small[1]}x{small[2]}, {sec1:.1f} s"
    except OSError:
        pass
    return out


def run_reference(args, rank: int, world: int) -> None:
    if rank != 0:
        return
    name = args.workload
    grid = tuple(args.grid) if args.grid else WORKLOADS[name][3]
    w = make_workload(name, grid)
    sec = oracle_step_seconds(w, args.steps, args.warmup)
    value = w.interior_cells * 3 * args.steps / sec
    sample = (f"each step = max wave speed + RK3 (3 RHS) of {name} generated at {grid[0]}x{grid[1]}x{grid[2]} "
              f"(bounded sample of the {'x'.join(map(str, WORKLOADS[name][1]))} workload)")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": name, "grid": list(WORKLOADS[name][1]), "nspecies": w.nspecies, "sample_grid": list(grid)},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------------------
# the B200 arm
# ---------------------------------------------------------------------------------------------------------------
class Ranks:
    """The N > 1 plumbing of the bench: one process per GPU, independent replicas (the path has
    no exchange step on one GPU), a barrier on both sides of the timed region and the MAX over ranks of the device
    time.  backend "nccl" on the GPU box; the CPU test drives the same class over "gloo" with world_size 2."""

    def __init__(self, world: int, backend: str = "nccl", device=None):
        self.world, self.device, self.dist = world, device, None
        if world > 1:
            import torch.distributed as dist

            if not dist.is_initialized():
                kw = {"device_id": device} if backend == "nccl" and device is not None else {}
                dist.init_process_group(backend, **kw)
            self.dist = dist

    def barrier(self) -> None:
        import torch

        if self.dist is not None:
            self.dist.barrier()
        if self.device is not None and self.device.type == "cuda":
            torch.cuda.synchronize()

    def max(self, x: float) -> float:
        if self.dist is None:
            return x
        import torch

        t = torch.tensor([x], dtype=torch.float64, device=self.device if self.device is not None else "cpu")
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def whole_job_value(self, cells_per_rank: int, rhs_per_step: int, ms_per_step_local: float) -> float:
        """cell-updates/s of ALL ranks: every rank does the same work, the slowest rank sets the time."""
        return cells_per_rank * rhs_per_step * self.world / (self.max(ms_per_step_local) * 1e-3)

    def close(self) -> None:
        if self.dist is not None and self.dist.is_initialized():
            self.dist.destroy_process_group()


def measured_peaks() -> dict:
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return {"hbm_gbs": float(d["hbm_gbs"]), "hbm_source": "MEASURED_PEAKS.json (of measured)"}
    return {"hbm_gbs": 6650.0, "hbm_source": "B200_PROFILING.md fallback (of fallback)"}


def lib_source_hash() -> str:
    """Hash of the CUDA sources of the benchmark path (sweeps, face flux, primitives, ghost fill, shared declarations): ties
    an ncu capture under profiles/ to the code it describes."""
    h = hashlib.sha256()
    src = ROOT / "paper_2403_05910_b200" / "csrc"
    for name in ("xf_common.cuh", "xf_flux.cuh", "xf_sweeps.cuh", "xf_sweep_x.cu", "xf_sweep_y.cu", "xf_sweep_z.cu",
                 "xf_prim.cu", "xf_ghost.cu"):
        h.update(name.encode())
        h.update((src / name).read_bytes())
    return h.hexdigest()[:16]


def ncu_capture(workload: str, kernel: str):
    """Per-launch figures of one kernel from the committed ncu --set full capture (profiles/r2_ncu_kernels.csv: dram bytes
    read + written, thread-level DFMA / DMUL / DADD counts) -- or None if there is no capture of that kernel, or the
    sources have changed since it was taken (the capture then describes other code)."""
    path = ROOT / "profiles" / "r2_ncu_kernels.csv"
    if not path.exists():
        return None
    here = lib_source_hash()
    for row in csv.DictReader(line for line in path.read_text().splitlines() if not line.startswith("#")):
        if row["workload"] == workload and row["kernel"] == kernel and row["source_hash"] == here:
            return {"dram_bytes": float(row["dram_bytes"]), "dfma": float(row["dfma"]), "dmul": float(row["dmul"]),
                    "dadd": float(row["dadd"]), "capture": f"profiles/r2_ncu_kernels.csv ({row['capture']})"}
    return None


def run_b200(args, rank: int, local_rank: int, world: int) -> None:
    import numpy as np
    import torch

    from paper_2403_05910_b200 import xf

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU path")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    ranks = Ranks(world, "nccl", dev)
    barrier, max_over_ranks = ranks.barrier, ranks.max

    name = args.workload
    grid = tuple(args.grid) if args.grid else WORKLOADS[name][1]
    if name == "config5":
        return run_config5(args, rank, local_rank, world, ranks)
    if name == "react":
        return run_react(args, rank, local_rank, world, ranks)
    if args.blocks:
        return run_blocks(args, rank, local_rank, world, ranks)
    w = make_workload(name, grid)
    if args.reconstruction == 2:
        from paper_2403_05910_b200 import workloads as wl

        w = wl.with_ghost_width(w, 4)
    N, Nv, cells = w.nspecies, w.nvars, w.interior_cells
    D = sum(1 for n in (w.nx, w.ny, w.nz) if n > 1)
    transport = None
    if args.viscous:
        from paper_2403_05910_b200 import workloads as wl

        transport = wl.synthetic_transport(w.table, seed=4, mu0=2e-4)
    ctx = xf.Context.from_workload(w, device=local_rank, viscosity=args.viscosity, reconstruction=args.reconstruction,
                                   positivity=args.positivity, transport=transport)
    U = torch.from_numpy(w.U).to(dev)
    T = torch.from_numpy(w.T_guess).to(dev)
    work = ctx.workspace()
    S = torch.zeros(1, dtype=torch.float64, device=dev)
    cfl = float(w.cfl)

    # fp64-pipe peak measured on this GPU, now (the denominator of the "alu" roofline): the burst
    # figure (best of five 136 ms launches) and the sustained one (back to back for 1.5 s, at the clocks a long fp64 load
    # holds); a kernel timed inside a long step is set against the sustained figure
    peak_burst_tf, probe_ms = xf.xf_probe_fp64_peak(local_rank, 60000)
    peak_tf, sustained_ms = xf.xf_probe_fp64_sustained(local_rank, 1.5)

    def step():
        ctx.xf_step_cfl(U, T, cfl, S, work)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    if ctx.xf_status() != 0:
        raise RuntimeError("non-physical state or Newton failure during warm-up")

    ctx.xf_timing_enable(32 * args.steps + 32)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    launches0 = ctx.xf_launch_count()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    clocks = sampler.stop()
    ms_total = max_over_ranks(float(e0.elapsed_time(e1)))
    launches = ctx.xf_launch_count() - launches0
    ktimes = ctx.xf_timing_read()
    ctx.xf_timing_enable(0)
    status = ctx.xf_status()
    if status != 0:
        raise RuntimeError(f"xf_status = {status} after the timed region")
    # mean Newton iteration count of the state the timed region ended on (debug counter; outside the timed region)
    ctx.xf_fill_ghosts(U)
    Tn = T.clone()
    ctx.xf_primitives(U, Tn)
    newton_its = ctx.xf_newton_mean_iterations()
    del Tn

    ms_per_step = ms_total / args.steps                      # ms_total is already the max over ranks
    value = cells * 3 * world / (ms_per_step * 1e-3)

    # ---- the same metric for xf_convective_rhs alone: ghosts + primitives + sweeps, no RK combine
    rhs_out = torch.empty_like(U)
    for _ in range(2):
        ctx.xf_convective_rhs(U, T, rhs_out, work)
    barrier()
    r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n_rhs = 3 * max(1, min(args.steps, 5))
    r0.record()
    for _ in range(n_rhs):
        ctx.xf_convective_rhs(U, T, rhs_out, work)
    r1.record()
    barrier()
    ms_rhs = max_over_ranks(float(r0.elapsed_time(r1))) / n_rhs
    del rhs_out
    rhs_only = {"value": cells * world / (ms_rhs * 1e-3), "unit": UNIT, "ms_per_rhs": ms_rhs, "evaluations": n_rhs,
                "api": "xf_convective_rhs (ghost fill, primitives, x/y/z sweeps; the residual written to its own array)"}

    # ---- roofline of the dominant kernel (per launch, CUDA events on the launching stream inside the timed region)
    peaks = measured_peaks()
    sweeps = {k: v for k, v in ktimes.items() if k.startswith("sweep") and v[1] > 0}
    dom = max(sweeps, key=lambda k: sweeps[k][0])
    dom_ms = sweeps[dom][0] / sweeps[dom][1]
    alg_flops = flops_per_face(N) * cells                      # one sweep launch = every face of one direction
    # bytes one sweep launch must move in THIS design: U (Nv) + p, c, Gamma, chi_s (N + 3) read, the partial residual
    # read (all but the first sweep) and one write of Nv fields
    first = dom == "sweep_x"
    alg_bytes = ((Nv + N + 3) + (0 if first else Nv) + Nv) * 8 * cells
    achieved_tf = alg_flops / (dom_ms * 1e-3) * 1e-12
    kernel_sum_ms = sum(v[0] for v in ktimes.values())
    cap = ncu_capture(name, dom)
    executed = None
    if cap is not None:   # what the fp64 pipe really did: the algorithmic count above is a model, not a minimum
        ex_flops = 2.0 * cap["dfma"] + cap["dmul"] + cap["dadd"]
        ex_inst = (cap["dfma"] + cap["dmul"] + cap["dadd"]) / 32.0          # warp instructions, 2 pipe cycles each
        sm_clock_hz = (clocks["sm_mhz"] or 0.0) * 1e6
        executed = {"flops_per_launch": ex_flops, "tflops": ex_flops / (dom_ms * 1e-3) * 1e-12,
                    "frac_of_sustained": ex_flops / (dom_ms * 1e-3) * 1e-12 / peak_tf,
                    "frac_of_nominal": ex_flops / (dom_ms * 1e-3) * 1e-12 / FP64_NOMINAL_TFLOPS,
                    "fp64_instructions_per_face": (cap["dfma"] + cap["dmul"] + cap["dadd"]) / cells,
                    "fp64_issue_slot_frac": (ex_inst * 2.0 / (148 * 4) / (sm_clock_hz * dom_ms * 1e-3)) if sm_clock_hz else None,
                    "source": cap["capture"]}
    roofline = {
        "bound": "alu", "achieved": achieved_tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": achieved_tf / peak_tf,
        "traffic": cap["dram_bytes"] if cap is not None else None,
        "traffic_source": cap["capture"] if cap is not None else "no ncu capture of this kernel at these sources",
        "peak_burst": peak_burst_tf, "frac_of_burst": achieved_tf / peak_burst_tf,
        "peak_nominal": FP64_NOMINAL_TFLOPS, "frac_of_nominal": achieved_tf / FP64_NOMINAL_TFLOPS,
        "executed": executed,
        "kernel": dom, "launch_ms": dom_ms, "launches_timed": sweeps[dom][1],
        "algorithmic_flops_per_launch": alg_flops, "algorithmic_bytes_per_launch": alg_bytes,
        "hbm_gbs_achieved": alg_bytes / (dom_ms * 1e-3) * 1e-9, "hbm_gbs_peak": peaks["hbm_gbs"],
        "hbm_frac": alg_bytes / (dom_ms * 1e-3) * 1e-9 / peaks["hbm_gbs"],
        "peak_source": f"of builder-measured: xf_probe_fp64_sustained on this GPU in this run ({sustained_ms:.0f} ms of "
                       f"back-to-back register-resident DFMA launches; burst = best of five {probe_ms:.0f} ms launches; "
                       f"MEASURED_PEAKS.json has no fp64 entry); HBM: {peaks['hbm_source']}",
        "kernel_share_of_step": {k: v[0] / kernel_sum_ms for k, v in ktimes.items() if v[1] > 0},
        "kernel_ms_per_launch": {k: v[0] / v[1] for k, v in ktimes.items() if v[1] > 0},
    }
    # whole step against the north-star roofline: the slower of bytes / HBM BW and fp64 flops / fp64 peak
    step_flops = flops_per_cell_rhs(N, D, newton_its) * cells * 3
    step_bytes = bytes_per_cell_rhs(N) * cells * 3
    t_alu, t_hbm = step_flops / (peak_tf * 1e12), step_bytes / (peaks["hbm_gbs"] * 1e9)
    step_roofline = {"t_roof_ms": max(t_alu, t_hbm) * 1e3, "t_alu_ms": t_alu * 1e3, "t_hbm_ms": t_hbm * 1e3,
                     "frac": max(t_alu, t_hbm) * 1e3 / ms_per_step,
                     "frac_of_nominal": max(step_flops / (FP64_NOMINAL_TFLOPS * 1e12), t_hbm) * 1e3 / ms_per_step,
                     "newton_mean_iterations": newton_its,
                     "flops_per_cell_rhs": flops_per_cell_rhs(N, D, newton_its),
                     "bytes_per_cell_rhs": bytes_per_cell_rhs(N)}

    # ---- end to end through the host-buffer C-ABI call: pinned host U, T -> device -> one step -> host, every step
    del U, T, work
    torch.cuda.empty_cache()
    Uh = torch.empty(w.U.shape, dtype=torch.float64, pin_memory=True)
    Th = torch.empty(w.T_guess.shape, dtype=torch.float64, pin_memory=True)
    Uh.copy_(torch.from_numpy(w.U))
    Th.copy_(torch.from_numpy(w.T_guess))
    Uh_np, Th_np = Uh.numpy(), Th.numpy()
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    ctx.xf_rk3_steps_host(Uh_np, Th_np, cfl, 1)                # warm-up: allocates the device mirrors
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        ctx.xf_rk3_steps_host(Uh_np, Th_np, cfl, 1)
    torch.cuda.synchronize()
    e2e_s = max_over_ranks(time.perf_counter() - t0)
    barrier()
    io_bytes = (Nv + 1) * ctx.cells * 8
    e2e = {"value": cells * 3 * world * e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": io_bytes,
           "d2h_bytes_per_step": io_bytes, "steps": e2e_steps, "ms_per_step": e2e_s / e2e_steps * 1e3,
           "api": "xf_rk3_steps_host (pinned host U, T in and out every step)"}
    if ctx.xf_status() != 0:
        raise RuntimeError("non-physical state during the end-to-end run")
    ctx.close()

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": name, "grid": list(grid), "nspecies": N, "nvars": Nv, "interior_cells": cells,
                       "step": "xf_step_cfl = max wave speed (in the first primitives kernel) + 3 x (ghost fill, "
                               "primitives, x/y/z sweeps, RK combine)", "rhs_per_step": 3, "l2": "inputs larger than L2 (one U copy = "
                               f"{Nv * ctx.cells * 8 / 1e9:.2f} GB), no flush", "parallelism": "replicas", "viscosity": ["LLF", "ROE", "GLF"][args.viscosity],
                       "reconstruction": ["WENO5-JS", "WENO-CU6", "WENO7"][args.reconstruction],
                       "positivity_limiter": bool(args.positivity), "viscous_terms": bool(args.viscous)},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline,
            "step_roofline": step_roofline, "rhs_only": rhs_only, "source_hash": lib_source_hash(),
        }
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(name)
        print(json.dumps(line), flush=True)
    ranks.close()


def run_config5(args, rank: int, local_rank: int, world: int, ranks) -> None:
    """BASELINE.json configs[4]: 640x384x384 random states generated on the device; K back-to-back xf_convective_rhs, each
    with the T guess restored to T (1 +- 2 %) OUTSIDE its timed span (events around every evaluation, summed)."""
    import torch

    from paper_2403_05910_b200 import workloads as wl
    from paper_2403_05910_b200 import xf

    grid = tuple(args.grid) if args.grid else WORKLOADS["config5"][1]
    w = wl.config5_random_states_device(*grid, device=f"cuda:{local_rank}")
    ctx = xf.Context.from_workload(w, device=local_rank)
    U, Tg = w.U, w.T_guess
    T = Tg.clone()
    work = ctx.workspace(rhs_only=True)
    out = torch.empty_like(U)
    peak_tf, sustained_ms = xf.xf_probe_fp64_sustained(local_rank, 1.5)
    steps = args.steps if args.steps != 5 else 50            # BASELINE.json: 50 evaluations
    for _ in range(args.warmup):
        T.copy_(Tg)
        ctx.xf_convective_rhs(U, T, out, work)
    ctx.xf_fill_ghosts(U)
    T.copy_(Tg)
    ctx.xf_primitives(U, T)
    newton_its = ctx.xf_newton_mean_iterations()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    ctx.xf_timing_enable(8 * steps + 8)
    sampler = ClockSampler(local_rank)
    ranks.barrier()
    sampler.start()
    l0 = ctx.xf_launch_count()
    for a, b in ev:
        T.copy_(Tg)
        a.record()
        ctx.xf_convective_rhs(U, T, out, work)
        b.record()
    ranks.barrier()
    clocks = sampler.stop()
    launches = ctx.xf_launch_count() - l0
    ms = ranks.max(sum(float(a.elapsed_time(b)) for a, b in ev)) / steps
    kt = ctx.xf_timing_read()
    if ctx.xf_status() != 0:
        raise RuntimeError("non-physical state in config 5")
    frac_out = float(((T < 200.0) | (T > 3000.0)).double().mean())
    cells, N = w.interior_cells, w.nspecies
    flops = flops_per_cell_rhs(N, 3, newton_its) * cells
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": cells * world / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": "config5", "grid": list(grid), "nspecies": N, "interior_cells": cells,
                       "step": "one xf_convective_rhs, T guess restored to T (1 +- 2 %) before it, outside the timed span",
                       "rhs_per_step": 1, "l2": "inputs larger than L2 (one U copy = 11 GB), no flush",
                       "cells_outside_fit_range": frac_out},
            "clocks": clocks, "gpu_launches": launches,
            "kernel_ms_per_launch": {k: v[0] / v[1] for k, v in kt.items() if v[1] > 0},
            "step_roofline": {"frac": flops / (peak_tf * 1e12) * 1e3 / ms, "newton_mean_iterations": newton_its,
                              "peak": peak_tf, "peak_source": f"xf_probe_fp64_sustained, {sustained_ms:.0f} ms"},
        }), flush=True)
    ctx.close()
    ranks.close()


def run_blocks(args, rank: int, local_rank: int, world: int, ranks) -> None:
    """The workload cut into px x py x pz blocks that live in this one process (halo.LocalTransport): every step goes through
    xf_fill_ghosts_dir / xf_pack_halo / device copy / xf_unpack_halo per direction and xf_rk3_stage per block -- the calls a
    multi-GPU run makes, minus the wire.  Reports the step time beside which the single-block figure can be set."""
    import torch

    from paper_2403_05910_b200 import halo

    name = args.workload
    grid = tuple(args.grid) if args.grid else WORKLOADS[name][1]
    w = make_workload(name, grid)
    dec, blocks = halo.make_blocks(w, args.blocks, device=local_rank)
    sol = halo.Solver(halo.LocalTransport(blocks))
    for _ in range(args.warmup):
        sol.step_cfl(float(w.cfl))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = sum(b.ctx.xf_launch_count() for b in blocks.values())
    ranks.barrier()
    e0.record()
    for _ in range(args.steps):
        sol.step_cfl(float(w.cfl))
    e1.record()
    ranks.barrier()
    ms = ranks.max(float(e0.elapsed_time(e1))) / args.steps
    launches = sum(b.ctx.xf_launch_count() for b in blocks.values()) - l0
    for b in blocks.values():
        if b.ctx.xf_status() != 0:
            raise RuntimeError("non-physical state in a block")
    halo_bytes = sum(8 * buf.numel() for b in blocks.values() for buf in b.send.values()) * 3
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": w.interior_cells * 3 * world / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": name, "grid": list(grid), "blocks": list(args.blocks), "transport": "in-process device copies",
                       "halo_bytes_per_step": halo_bytes, "step": "max wave speed over the blocks (host reduction) + 3 x (per "
                       "direction: ghost fill, pack, copy, unpack; xf_rk3_stage per block)"},
            "gpu_launches": launches}), flush=True)
    for b in blocks.values():
        b.ctx.close()
    ranks.close()


def run_react(args, rank: int, local_rank: int, world: int, ranks) -> None:
    """The reaction step alone (not the bench line): xf_react over dt with 4 sub-steps of one
    predictor and one corrector on 256x128x128 cells of the nine-species reacting box, 19-reaction seeded mechanism; the
    state is restored before every timed call (outside the timed span), so every call does the same work."""
    import torch

    from paper_2403_05910_b200 import workloads as wl
    from paper_2403_05910_b200 import xf

    grid = tuple(args.grid) if args.grid else WORKLOADS["react"][1]
    w = wl.reacting_box(*grid, seed=11)
    mech = wl.synthetic_mechanism(w.table, wl.reacting_table()[1], 19, seed=19, rate=5.0)
    ctx = xf.Context.from_workload(w, device=local_rank)
    ctx.xf_set_mechanism(mech)
    dev = torch.device("cuda", local_rank)
    U0, T0 = torch.from_numpy(w.U).to(dev), torch.from_numpy(w.T_guess).to(dev)
    U, T = U0.clone(), T0.clone()
    n_sub, dt = 4, 5e-4
    for _ in range(args.warmup):
        U.copy_(U0); T.copy_(T0)
        ctx.xf_react(U, T, dt, n_sub, 1)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sampler = ClockSampler(local_rank)
    ranks.barrier()
    sampler.start()
    for a, b in ev:
        U.copy_(U0); T.copy_(T0)
        a.record()
        ctx.xf_react(U, T, dt, n_sub, 1)
        b.record()
    ranks.barrier()
    clocks = sampler.stop()
    ms = ranks.max(sum(float(a.elapsed_time(b)) for a, b in ev)) / args.steps
    if ctx.xf_status() != 0:
        raise RuntimeError("reaction step failed")
    cells = w.interior_cells
    if rank == 0:
        print(json.dumps({
            "metric": "cell reaction steps/s (alpha-QSS, 4 sub-steps x (predictor + corrector) = 8 rate evaluations)",
            "value": cells * world / (ms * 1e-3), "unit": "cell-steps/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": "react", "grid": list(grid), "nspecies": w.nspecies, "reactions": 19, "n_sub": n_sub,
                       "n_corr": 1, "rate_evaluations_per_cell_per_s": cells * world * 2 * n_sub / (ms * 1e-3)},
            "clocks": clocks, "gpu_launches": args.steps}), flush=True)
    ctx.close()
    ranks.close()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=("b200", "reference"))
    ap.add_argument("--workload", default="config4", choices=sorted(WORKLOADS))
    ap.add_argument("--grid", type=int, nargs=3, default=None, help="override the grid (debugging only)")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--viscosity", type=int, default=0, help="0 LLF (the benchmark), 1 ROE, 2 GLF")
    ap.add_argument("--reconstruction", type=int, default=0, help="0 WENO5-JS (the benchmark), 1 WENO-CU6, 2 WENO7")
    ap.add_argument("--positivity", action="store_true", help="positivity-preserving flux blending on (not the benchmark)")
    ap.add_argument("--blocks", type=int, nargs=3, default=None,
                    help="run the workload as px py pz blocks IN THIS PROCESS through the halo-exchange path (halo.py, "
                         "LocalTransport): what the decomposition costs on one GPU; not the benchmark")
    ap.add_argument("--viscous", action="store_true",
                    help="viscous / diffusive terms on, seeded synthetic transport fits (not the benchmark)")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.warmup < 3:
        args.warmup = 3 if args.impl == "b200" else args.warmup
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_b200(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
