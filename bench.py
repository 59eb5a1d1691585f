#!/usr/bin/env python
"""bench.py — MLUPS and DRAM roofline fraction of the fused D3Q19 LES + forest LBM step on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg5] [--impl b200|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is one time step of the whole hot path: one fused step-kernel
launch plus, on the configs that accumulate statistics every step, the stage-2 reduction launch.
The default workload is BASELINE.json:configs[4] ("cfg5", 1536x384x1024, single-array AA storage,
45.9 GB of populations), the largest configuration, on which north_star states its target.

One JSON line is printed by rank 0:
  value        MLUPS (1e6 lattice-cell updates per second), whole job, state resident in HBM
  e2e          the same metric through the C ABI with HOST buffers: lbm_set_macros_host (pinned
               host rho,u -> device) + K x [lbm_step(1) + lbm_stats_read (device -> host)]
  roofline     step kernel only: 152 B/cell x cells / mean device time of the step-kernel launches
               (CUDA events recorded by the library on its launch stream, lbm_set_kernel_timing)
               against MEASURED_PEAKS.json's hbm_gbs
  cpu_baseline the fp64 oracle, as it stands, on the host cores on a bounded slab of the workload
--gpus N > 1: north_star asks for one GPU; by default every rank runs an independent replica of
the workload and `value` is the sum over replicas.  --sharded instead cuts ONE lattice of
nx x ny x (N nz) cells into N z slabs with a halo exchange per step.
--impl reference times the oracle alone (the reference arm of this tier).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402

BYTES_PER_CELL = 152.0  # 2 x 19 x 4 B (BASELINE.json:north_star)
# dram__bytes_read.sum + dram__bytes_write.sum per step-kernel launch / cells, from ncu captures
# of the current kernels on the named config (profiles/): the line quotes the figure of its own
# config when one exists, else null.
NCU_TRAFFIC_BYTES_PER_CELL = {
    ("cfg5", "aax"): (152.11, "profiles/r02_dram_cfg5.csv, ncu dram__bytes_read+write on cfg5 itself, both parities"),
    ("cfg4", "aax"): (151.7, "profiles/r02_step_kernel_cfg4_details.txt, ncu --set full on cfg4, both parities"),
    ("cfg3", "two_lattice"): (149.1, "profiles/r02_step_kernel_cfg3_stats_details.txt, ncu --set full on cfg3"),
    ("cfg2", "aax"): (138.8, "profiles/r02_step_kernel_cfg2_details.txt, ncu --set full on cfg2 (part of the writes "
                             "is still dirty in the L2 when the launch ends)"),
}
METRIC = "MLUPS"
UNIT = "MLUPS (1e6 lattice-cell updates/s)"


def measured_peak():
    """HBM copy peak from MEASURED_PEAKS.json (driver-written), else the guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML every 100 ms while the timed region runs."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index = index
        self.stop_flag = threading.Event()
        self.sm, self.reasons, self.sm_max, self.power = [], set(), None, []
        self.err = None
        self.ready = threading.Event()

    def begin(self):
        """Start sampling and wait until NVML is up, so that short timed regions get samples."""
        self.start()
        self.ready.wait(5.0)

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.sm_max = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {
                getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
                getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
                getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
                getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4): "sw_power_cap",
            }
            self.ready.set()
            while not self.stop_flag.is_set():
                self.sm.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                try:
                    self.power.append(nv.nvmlDeviceGetPowerUsage(h) / 1000.0)
                except Exception:
                    pass
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
                self.stop_flag.wait(0.1)
        except Exception as e:  # NVML missing: report it, do not fail the bench
            self.err = repr(e)
            self.ready.set()

    def result(self):
        self.stop_flag.set()
        self.join(timeout=2.0)
        sm = sorted(self.sm)
        out = {"sm_mhz": (sm[len(sm) // 2] if sm else None), "sm_max_mhz": self.sm_max,
               "reasons": sorted(self.reasons), "samples": len(sm)}
        if self.power:
            out["power_w_max"] = round(max(self.power), 1)
        if self.err:
            out["error"] = self.err
        return out


# ---------------------------------------------------------------------------------------------
# the oracle leg (cpu_baseline of the default arm; the whole of --impl reference)
# ---------------------------------------------------------------------------------------------
def oracle_sample_config(cfg: dict, max_nx: int = 256, max_nz: int = 64) -> dict:
    """Bounded sample of the workload for the CPU oracle: the same physics, boundary set, canopy
    table and full wall-normal extent ny, on an x-z sub-slab (periodic) of at most 256 x 64
    columns, so that the fp64 two-lattice oracle (304 B/cell) stays near 2 GB."""
    s = dict(cfg)
    s["nx"] = min(cfg["nx"], max_nx)
    s["nz"] = min(cfg["nz"], max_nz)
    return s


def time_oracle(cfg: dict, steps: int, warmup: int, budget_s: float = 15.0, max_nx: int = 256,
                max_nz: int = 64):
    """Time the oracle as it stands on the host cores.  `steps` = 0: as many steps as fit the
    time budget (at least 2).  Returns (MLUPS, ms per step, steps, cores, sample text)."""
    import oracle

    s = oracle_sample_config(cfg, max_nx, max_nz)
    cores = os.cpu_count() or 1
    try:
        cores = len(os.sched_getaffinity(0))
    except Exception:
        pass
    env_threads = os.environ.get("OMP_NUM_THREADS")
    if env_threads:
        cores = min(cores, int(env_threads))
    o = oracle.Oracle.from_config(s)
    o.init_from_config(s)
    if s.get("stats_every", 0) > 0:
        o.stats_accumulate(s["stats_every"])
    n_cells = wl.n_cells(s)
    t0 = time.perf_counter()
    o.step(max(1, warmup))
    per = (time.perf_counter() - t0) / max(1, warmup)
    if steps <= 0:
        steps = int(max(2, min(500, budget_s / max(per, 1e-6))))
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    o.stats_read()
    mlups = n_cells * steps / dt / 1e6
    sample = (f"{s['nx']}x{s['ny']}x{s['nz']} periodic x-z sub-slab of {cfg['name']} "
              f"({n_cells} cells, same physics/BCs/canopy, full ny), {steps} oracle steps, "
              f"fp64 two-lattice, gcc -O2 -fopenmp")
    return mlups, dt / steps * 1e3, steps, cores, sample


def run_reference(args, cfg):
    """--impl reference: the oracle alone, rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    steps = args.steps
    # bounded sample: each step is one oracle time step of a 128 x ny x 32 slab (~0.3 s)
    mlups, ms, steps_done, cores, sample = time_oracle(cfg, steps, args.warmup, max_nx=128, max_nz=32)
    ran = oracle_sample_config(cfg, 128, 32)
    conf = workload_config(cfg, args, None)
    # the lattice the oracle actually advanced (a bounded x-z sub-slab of the workload, full ny)
    conf["lattice"] = [ran["nx"], ran["ny"], ran["nz"]]
    conf["cells"] = wl.n_cells(ran)
    conf["full_workload_lattice"] = [cfg["nx"], cfg["ny"], cfg["nz"]]
    conf["storage"] = "two_lattice fp64 (oracle)"
    conf["l2"] = "oracle on host cores; no GPU cache involved"
    conf["parallelism"] = f"{cores} host threads (OpenMP)"
    line = {
        "impl": "reference", "metric": METRIC, "value": round(mlups, 3), "unit": UNIT,
        "n_gpus": args.gpus, "steps": steps_done, "warmup": args.warmup,
        "ms_per_step": round(ms, 4), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": conf,
        "cpu_baseline": {"value": round(mlups, 3), "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": round(mlups, 3), "unit": UNIT, "h2d_bytes_per_step": 0,
                "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def workload_config(cfg, args, variant):
    pops_gb = wl.n_cells(cfg) * 76 * (1 if cfg["storage"] in ("aa", "aax") else 2) / 1e9
    c = {
        "workload": f"{cfg['name']}: {cfg['note']}",
        "lattice": [cfg["nx"], cfg["ny"], cfg["nz"]], "cells": wl.n_cells(cfg),
        "storage": cfg["storage"], "stats_every": cfg.get("stats_every", 0),
        "bottom": cfg["bottom"], "top": cfg["top"], "nu": cfg["nu"], "Cs": cfg["Cs"],
        "Cd": cfg["Cd"], "seed": cfg["seed"],
        "l2": f"no flush: populations are {pops_gb:.2f} GB per pass, larger than the 126 MB L2"
              if pops_gb > 0.2 else "L2-resident workload (populations fit the 126 MB L2): "
              "the DRAM roofline fraction is not meaningful here",
        "parallelism": "1 GPU" if args.gpus == 1 else f"{args.gpus} independent replicas",
    }
    if variant:
        c["kernel_variant"] = variant
    return c


def max_over_ranks(values, world: int, device):
    """Element-wise MAX over the ranks of the default process group (times of independent
    replicas: the job is as slow as its slowest rank).  world == 1: the values themselves."""
    import torch
    import torch.distributed as dist

    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def aggregate_mlups(n_cells: int, steps: int, ms: float, world: int) -> float:
    """Whole-job MLUPS of `world` replicas that each advanced n_cells x steps in `ms` (max)."""
    return world * n_cells * steps / (ms * 1e-3) / 1e6


# ---------------------------------------------------------------------------------------------
# the CUDA leg
# ---------------------------------------------------------------------------------------------
def run_b200(args, cfg):
    import numpy as np
    import torch
    import torch.distributed as dist

    import paper_2206_15454_b200 as lb

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    K, W = args.steps, args.warmup
    N = wl.n_cells(cfg)
    every = cfg.get("stats_every", 0)
    sim = lb.Lbm.from_config(cfg, vec=args.vec, device=dev)   # storage scheme from cfg["storage"]
    if args.shape:
        tx, ty = (int(v) for v in args.shape.split("x"))
        sim.set_launch_shape(tx, ty)
    if args.tma is not None:
        tm = [int(v) for v in args.tma.split(",")]
        sim.set_tma(tm[0], tm[1] if len(tm) > 1 else 0)
    if args.sweep is not None:
        sim.set_sweep(args.sweep)
    sim.init(cfg["seed"] + rank)
    sim.stats_accumulate(every)
    stream = torch.cuda.current_stream(dev)

    # ---- device-resident throughput: W warm-up steps, then exactly K timed steps ----
    # roofline leg: the step kernel alone, each launch bracketed by a pair of CUDA events that the
    # library records on its launch stream.  On lattices whose step takes milliseconds the
    # brackets sit INSIDE the K timed steps (the same launches give `value` and
    # `roofline.achieved`, so kernel_ms <= ms_per_step by construction; two event records per
    # >= 3 ms step cost nothing measurable).  Smaller lattices are timed without brackets (a pair
    # of event records is comparable to their launch gaps, and lbm_step replays CUDA graphs
    # there) and bracketed in a second K-step pass.
    same_pass = N * BYTES_PER_CELL / 6.5e12 > 1e-3 and K <= 4096
    sim.step(W)
    barrier()
    sampler = ClockSampler(local)
    sampler.begin()
    l0 = sim.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if same_pass:
        sim.set_kernel_timing(True)
    e0.record(stream)
    sim.step(K)
    e1.record(stream)
    barrier()
    launches = sim.launch_count - l0
    ms = e0.elapsed_time(e1)
    clocks = sampler.result()
    stats, nsamp = sim.stats_read()
    if every > 0 and (nsamp != (W + K) // every or not np.isfinite(stats).all()):
        raise RuntimeError(f"statistics check failed: nsamples={nsamp}, finite={np.isfinite(stats).all()}")
    if not same_pass:
        sim.set_kernel_timing(True)
        sim.step(min(K, 4096))
    k_ms, k_n = sim.kernel_timing_read()
    sim.set_kernel_timing(False)
    kernel_ms = k_ms / max(1, k_n)

    # ---- end to end through the C ABI with host buffers ----
    rho_h = torch.empty(sim.shape, dtype=torch.float32).pin_memory()
    u_h = torch.empty((3,) + sim.shape, dtype=torch.float32).pin_memory()
    sim.get_macros_host(rho_h, u_h)          # a valid field to restart from (untimed)
    e2e_steps = K
    barrier()
    t0 = time.perf_counter()
    sim.set_macros_host(rho_h, u_h)          # H2D of the step inputs, then f = f_eq(rho, u)
    sim.stats_accumulate(max(1, every))
    out = None
    for _ in range(e2e_steps):
        sim.step(1)
        out, _n = sim.stats_read()           # D2H of the step's result; synchronises
    barrier()
    e2e_s = time.perf_counter() - t0
    if not np.isfinite(out).all():
        raise RuntimeError("end-to-end leg produced non-finite statistics")
    h2d = (rho_h.numel() + u_h.numel()) * 4 / e2e_steps
    d2h = cfg["ny"] * (lb.NSTAT * 8 + 16) + 4

    # ---- max over ranks, sum of work ----
    ms, e2e_ms, kernel_ms = max_over_ranks([ms, e2e_s * 1e3, kernel_ms], world, dev)
    variant = sim.variant
    sim.close()
    del sim, rho_h, u_h
    torch.cuda.empty_cache()

    if rank == 0:
        peak, peak_src = measured_peak()
        mlups = aggregate_mlups(N, K, ms, world)
        e2e_mlups = aggregate_mlups(N, e2e_steps, e2e_ms, world)
        achieved = BYTES_PER_CELL * N / (kernel_ms * 1e-3) / 1e9
        traffic, traffic_src = args.traffic, "command line (--traffic)"
        key = (cfg["name"], cfg["storage"])
        if traffic is None and key in NCU_TRAFFIC_BYTES_PER_CELL:
            bpc, where = NCU_TRAFFIC_BYTES_PER_CELL[key]
            traffic = round(bpc * N)
            traffic_src = f"{where}: {bpc} B/cell x {N} cells"
        elif traffic is None:
            traffic_src = None
        line = {
            "metric": METRIC, "value": round(mlups, 1), "unit": UNIT, "n_gpus": world,
            "steps": K, "warmup": W, "ms_per_step": round(ms / K, 5), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": workload_config(cfg, args, variant),
            "algorithmic_gbs": round(mlups * BYTES_PER_CELL / 1e3 / world, 1),
            "frac_of_nominal_8tbs": round(mlups * BYTES_PER_CELL / 1e3 / world / 8000.0, 4),
            "roofline": {"bound": "hbm", "kernel": "lbm::step_kernel (" + variant + ")",
                         "achieved": round(achieved, 1), "peak": peak, "unit": "GB/s",
                         "frac": round(achieved / peak, 4), "traffic": traffic,
                         "traffic_source": traffic_src,
                         "peak_source": peak_src, "bytes_per_cell": BYTES_PER_CELL,
                         "kernel_ms": round(kernel_ms, 5), "launches_timed": k_n,
                         "timed_in": "the K timed steps themselves" if same_pass else
                                     "a second K-step pass (the timed pass runs unbracketed)"},
            "e2e": {"value": round(e2e_mlups, 1), "unit": UNIT,
                    "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "steps": e2e_steps,
                    "what": "lbm_set_macros_host(pinned rho,u) + steps x [lbm_step(1) + lbm_stats_read]"},
            "gpu_launches": int(launches),
            "clocks": clocks,
        }
        if not args.no_cpu and world == 1:
            cm, _cms, _cs, cores, sample = time_oracle(cfg, 0, 1)
            line["cpu_baseline"] = {"value": round(cm, 2), "unit": UNIT, "cores": cores,
                                    "kind": "oracle", "sample": sample}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_sharded(args, cfg):
    """--sharded: ONE lattice of nx x ny x (N nz) cut into N z slabs (two-lattice storage unless
    --storage says aa / aax), one
    halo exchange per step over torch.distributed, overlapped with the interior update
    (DESIGN.md "Multi-GPU").  Opt-in: north_star asks for one GPU, so the default --gpus N path
    stays N replicas; on this run's hardware the NCCL leg could only be exercised with N = 1
    (self exchange through the second stream) and emulated rings."""
    import numpy as np
    import torch
    import torch.distributed as dist

    import paper_2206_15454_b200 as lb
    from paper_2206_15454_b200 import slab

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    g = dict(cfg)
    g["nz"] = cfg["nz"] * world
    g["storage"] = args.storage or "two_lattice"
    K, W = args.steps, args.warmup
    N = wl.n_cells(cfg)
    every = cfg.get("stats_every", 0)
    s = slab.SlabLbm(g, rank, world, device=dev, storage=g["storage"])
    s.init(cfg["seed"])
    s.stats_accumulate(every)
    s.step(W)
    barrier()
    sampler = ClockSampler(local)
    sampler.begin()
    stream = torch.cuda.current_stream(dev)
    l0 = s.sim.launch_count
    same_pass = N * BYTES_PER_CELL / 6.5e12 > 1e-3 and 3 * K <= 4096
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if same_pass:
        s.sim.set_kernel_timing(True)
    e0.record(stream)
    s.step(K)
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    launches = s.sim.launch_count - l0
    clocks = sampler.result()
    st = s.stats_read()
    if not np.isfinite(st).all():
        raise RuntimeError("sharded run produced non-finite statistics")
    nk = K
    if not same_pass:
        nk = min(K, 1300)
        s.sim.set_kernel_timing(True)
        s.step(nk)
    k_ms, _k_n = s.sim.kernel_timing_read()
    s.sim.set_kernel_timing(False)
    kernel_ms = k_ms / nk                      # boundary-plane + interior launches of one step

    # end to end: host fields of the slab -> device, then K x [step + statistics read (all-reduce + D2H)]
    rho_h = torch.empty(s.sim.shape, dtype=torch.float32).pin_memory()
    u_h = torch.empty((3,) + s.sim.shape, dtype=torch.float32).pin_memory()
    s.sim.get_macros_host(rho_h, u_h)
    barrier()
    t0 = time.perf_counter()
    s.sim.set_macros_host(rho_h, u_h)
    s.exchange()
    s.stats_accumulate(max(1, every))
    out = None
    for _ in range(K):
        s.step(1)
        out = s.stats_read()
    barrier()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    if not np.isfinite(out).all():
        raise RuntimeError("end-to-end leg produced non-finite statistics")
    ms, e2e_ms, kernel_ms = max_over_ranks([ms, e2e_ms, kernel_ms], world, dev)
    variant = s.sim.variant
    if rank == 0:
        peak, peak_src = measured_peak()
        mlups = aggregate_mlups(N, K, ms, world)
        achieved = BYTES_PER_CELL * N / (kernel_ms * 1e-3) / 1e9
        cfgd = workload_config(g, args, variant)
        cfgd["parallelism"] = (f"one lattice in {world} z slab(s), ring halo exchange of 2 x 5 x nx x ny fp32 "
                               "per step on a second stream, overlapped with the interior update")
        line = {
            "metric": METRIC, "value": round(mlups, 1), "unit": UNIT, "n_gpus": world, "steps": K,
            "warmup": W, "ms_per_step": round(ms / K, 5), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": cfgd,
            "algorithmic_gbs": round(mlups * BYTES_PER_CELL / 1e3 / world, 1),
            "frac_of_nominal_8tbs": round(mlups * BYTES_PER_CELL / 1e3 / world / 8000.0, 4),
            "roofline": {"bound": "hbm", "kernel": "lbm::step_kernel (" + variant + "), boundary + interior launches",
                         "achieved": round(achieved, 1), "peak": peak, "unit": "GB/s",
                         "frac": round(achieved / peak, 4), "traffic": None, "traffic_source": None,
                         "peak_source": peak_src, "bytes_per_cell": BYTES_PER_CELL,
                         "kernel_ms": round(kernel_ms, 5),
                         "timed_in": "the K timed steps themselves" if same_pass else "a second pass"},
            "e2e": {"value": round(aggregate_mlups(N, K, e2e_ms, world), 1), "unit": UNIT,
                    "h2d_bytes_per_step": int((rho_h.numel() + u_h.numel()) * 4 / K),
                    "d2h_bytes_per_step": int(cfg["ny"] * lb.NSTAT * 8 + 8), "steps": K,
                    "what": "lbm_set_macros_host(pinned slab fields) + steps x [slab step + stats read (all-reduce)]"},
            "halo_bytes_per_step": 2 * 5 * cfg["nx"] * cfg["ny"] * 4,
            "gpu_launches": int(launches), "clocks": clocks, "mode": "sharded"}
        if not args.no_cpu and world == 1:
            cm, _cms, _cs, cores, sample = time_oracle(cfg, 0, 1)
            line["cpu_baseline"] = {"value": round(cm, 2), "unit": UNIT, "cores": cores,
                                    "kind": "oracle", "sample": sample}
        print(json.dumps(line))
    s.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None,
                    help="timed steps; default: the count BASELINE.json states for the config "
                         "(cfg5: 500, cfg4: 1000), 200 for the small ones")
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", choices=["b200", "reference"], default="b200")
    ap.add_argument("--config", default="cfg5", help="cfg1..cfg5 (BASELINE.json:configs[0..4])")
    ap.add_argument("--storage", choices=["aa", "aax", "two_lattice"], default=None,
                    help="override the config's storage scheme")
    ap.add_argument("--stats-every", type=int, default=None, help="override the config's stats cadence")
    ap.add_argument("--shape", default=None, help="thread-block shape override TXxTY (tuning)")
    ap.add_argument("--tma", default=None,
                    help="A/B: step kinds on the TMA path, 'mode[,rows]' (bit 0 AA even, 1 AA odd, 2 pull)")
    ap.add_argument("--vec", type=int, choices=[0, 1, 2, 4], default=0,
                    help="A/B: cells per thread (0 = the library's choice)")
    ap.add_argument("--sweep", type=int, choices=[0, 1], default=None,
                    help="A/B: 0 = every step walks the lattice forward, 1 = alternating direction (default)")
    ap.add_argument("--traffic", type=float, default=None,
                    help="ncu dram bytes (read+write) per step-kernel launch, from profiles/, to quote in the line")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--boxes", action="store_true",
                    help="geometry handle with the paper's turbulence-trip boxes in place (PAPER.md:L226): "
                         "times the geometry variants of the kernels")
    ap.add_argument("--geometry", action="store_true",
                    help="geometry handle (LBM_SOLID_MASK) with an all-fluid mask: the cost of the per-block flag alone")
    ap.add_argument("--sharded", action="store_true",
                    help="one lattice cut into N z slabs with a halo exchange per step (opt-in)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    cfg = wl.get(args.config)
    if args.steps is None:
        # BASELINE.json:configs[3,4] state the timed step counts (1000, 500); the reference arm's
        # steps are oracle steps on a bounded slab (~0.3 s each), kept to a few minutes
        args.steps = 20 if args.impl == "reference" else (
            cfg["steps"] if cfg["name"] in ("cfg4", "cfg5") else 200)
    if args.storage:
        cfg["storage"] = args.storage
    if args.stats_every is not None:
        cfg["stats_every"] = args.stats_every
    if args.boxes:
        from paper_2206_15454_b200.run_paper_cases import trip_boxes
        cfg["solid"] = trip_boxes(cfg)
        cfg["note"] += ", trip boxes in place (geometry kernels)"
    if args.geometry:
        cfg["geometry"] = True
        cfg["note"] += ", geometry handle with an all-fluid mask"
    if args.impl == "reference":
        return run_reference(args, cfg)
    if args.sharded:
        return run_sharded(args, cfg)
    return run_b200(args, cfg)


if __name__ == "__main__":
    sys.exit(main())
