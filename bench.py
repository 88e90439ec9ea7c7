#!/usr/bin/env python
"""bench.py -- throughput of the coupled LBM + immersed-boundary hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

A "step" is one pass of the whole hot path: ib_compute_membrane_forces ->
ib_spread -> lbm_step(forcing) -> ib_interpolate_advance, through the C-ABI of libplb.  The
default workload is BASELINE.json's config 4 (512 x 128 x 1024 shear channel, 1024 platelets,
657,408 nodes): the coupled configuration the north_star's targets are stated on; it fits one
GPU (10.2 GB of lattice).  Prints ONE JSON line (rank 0).

Multi-GPU (--gpus N under torchrun): the path has no exchange step in this build ("replicas
only"): every rank runs the same workload on its own GPU, no data-path collective;
value = units all ranks processed / max-over-ranks time ("scaling": "weak").

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores on a bounded
sample of the same workload; it is a deliberately plain program, a reported baseline only.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "coupled LBM+IB MLUPS (fp32 D3Q19)"
UNIT = "MLUPS"
BYTES_PER_CELL = 2 * 19 * 4          # algorithmic bytes of S3 per cell per step
FALLBACK_HBM_GBS = 6650.0            # B200_PROFILING.md fallback if MEASURED_PEAKS.json is absent
NOMINAL_HBM_GBS = 8000.0


def parse_args(argv=None):
    p = argparse.ArgumentParser()
    p.add_argument("--gpus", type=int, default=1)
    p.add_argument("--steps", type=int, default=500, help="timed coupled steps (default: config 4's own 500)")
    p.add_argument("--warmup", type=int, default=5)
    p.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5])
    p.add_argument("--impl", default="ours", choices=["ours", "reference"])
    p.add_argument("--spread-mode", default="auto", choices=["auto", "scatter", "aggregate", "gather"],
                   help="form of the S2 kernel (ib_set_spread_mode); auto = the library's own choice")
    p.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg")
    p.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg")
    p.add_argument("--dist-dry-run", action="store_true",
                   help="CPU test of the N>1 plumbing (gloo): fake per-rank times, real barrier/max/aggregation")
    return p.parse_args(argv)


def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))


# ---------------------------------------------------------------------------------------------
# workload naming / sampling
# ---------------------------------------------------------------------------------------------
def describe(w):
    s = "C%s %dx%dx%d" % (w.name[1:], w.nx, w.ny, w.nz)
    if w.n_meshes:
        s += ", %d platelets (%d nodes, %d edges)" % (w.n_meshes, w.n_nodes, w.n_edges)
    else:
        s += ", no immersed boundary"
    return s


def cpu_sample(config):
    """Bounded sample of the bench workload for the oracle legs: the same recipe (tau, wall speed,
    mesh shape, platelet number density, channel height) on a smaller footprint."""
    from paper_1312_2234_b200 import workloads as wl
    if config == 4:
        return wl.config4(nx=128, ny=128, nz=128, n_meshes=32), "C4 recipe on a 128x128x128 footprint, 32 platelets (same number density and channel height)"
    if config == 3:
        return wl.config3(nx=128, ny=64, nz=128, n_meshes=4), "C3 recipe on a 128x64x128 footprint, 4 platelets"
    if config == 5:
        return wl.config5(n=256, grid_xz=8, layers=2, subdiv=4), "C5 recipe with 128 of the 8192 platelets"
    if config == 2:
        return wl.config2(n=128), "C2 recipe at 128^3"
    return wl.config1(), "C1 whole"


def aggregate(cells_per_rank, steps, world, max_seconds):
    """whole-job MLUPS: the cell updates of all ranks over the slowest rank's time"""
    return cells_per_rank * steps * world / max_seconds / 1e6


def max_over_ranks(x, device):
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def barrier(device):
    import torch
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        if device.type == "cuda":
            dist.barrier(device_ids=[device.index])
        else:
            dist.barrier()
    if device.type == "cuda":
        torch.cuda.synchronize(device)


# ---------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md)
# ---------------------------------------------------------------------------------------------
class ClockSampler:
    """SM clock and throttle reasons of one GPU, sampled every 20 ms by a thread (NVML, the same
    counters `nvidia-smi --query-gpu=clocks.sm,clocks.max.sm,clocks_event_reasons.*` prints);
    falls back to an `nvidia-smi -lms` child process when pynvml is missing.  Sampling runs from
    start() to stop(); mark() opens the timed region, only samples after it are reported."""
    SMI_FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
                  "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
                  "clocks_event_reasons.sw_power_cap")
    NAMES = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")

    def __init__(self, gpu_index):
        import threading
        self.samples = []          # (t, sm_mhz, set of reasons)
        self.sm_max = None
        self.t_mark = None
        self.how = None
        self._stop = threading.Event()
        self._thread = None
        self._proc = None
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = gpu_index
            if vis:
                ids = [v.strip() for v in vis.split(",") if v.strip()]
                if gpu_index < len(ids) and ids[gpu_index].isdigit():
                    phys = int(ids[gpu_index])
            h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            bits = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}

            def poll():
                while not self._stop.is_set():
                    try:
                        mhz = float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM))
                        r = int(pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h))
                        self.samples.append((time.perf_counter(), mhz, {n for n, b in bits.items() if r & b}))
                    except Exception:
                        pass
                    self._stop.wait(0.02)
            self._thread = threading.Thread(target=poll, daemon=True)
            self._thread.start()
            self.how = "nvml, 20 ms"
        except Exception:
            self._start_smi(gpu_index)

    def _start_smi(self, gpu_index):
        import threading
        try:
            self._proc = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), "--query-gpu=" + self.SMI_FIELDS,
                                           "--format=csv,noheader,nounits", "-lms", "50"],
                                          stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self._proc = None
            return

        def read():
            for line in self._proc.stdout:
                parts = [p.strip() for p in line.split(",")]
                if len(parts) < 7:
                    continue
                try:
                    mhz, mx = float(parts[0]), float(parts[1])
                except ValueError:
                    continue
                self.sm_max = mx
                self.samples.append((time.perf_counter(), mhz,
                                     {n for n, v in zip(self.NAMES, parts[3:7]) if v.lower().startswith("active")}))
        self._thread = threading.Thread(target=read, daemon=True)
        self._thread.start()
        self.how = "nvidia-smi -lms 50"

    def mark(self):
        self.t_mark = time.perf_counter()

    def stop(self):
        t_end = time.perf_counter()
        self._stop.set()
        if self._proc is not None:
            self._proc.terminate()
            try:
                self._proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self._proc.kill()
        if self._thread is not None:
            self._thread.join(timeout=5)
        t0 = self.t_mark if self.t_mark is not None else 0.0
        inside = [s for s in self.samples if t0 <= s[0] <= t_end]
        out = {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": [], "samples": len(inside), "how": self.how}
        if inside:
            sm = sorted(s[1] for s in inside)
            reasons = set()
            for s in inside:
                reasons |= s[2]
            out.update(sm_mhz=sm[len(sm) // 2], reasons=sorted(reasons))
        return out


def hbm_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json, copy bandwidth)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(config):
    """DRAM bytes per launch of the LBM kernel (dram__bytes_read.sum + dram__bytes_write.sum of one
    ncu --set full capture), from the committed summary profiles/lbm_dram_traffic.txt, or None.
    Line format:  C<config> <bytes per launch>  # which capture"""
    try:
        for line in open(os.path.join(ROOT, "profiles", "lbm_dram_traffic.txt")):
            parts = line.split("#")[0].split()
            if len(parts) >= 2 and parts[0] == "C%d" % config:
                return float(parts[1])
    except Exception:
        pass
    return None


# ---------------------------------------------------------------------------------------------
# the oracle legs (host cores)
# ---------------------------------------------------------------------------------------------
def time_oracle(config, steps, warmup):
    """The CPU oracle as it stands, on all host cores, on a bounded sample of the workload."""
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    os.environ.setdefault("OMP_NUM_THREADS", str(cores))
    threads = int(os.environ["OMP_NUM_THREADS"])
    from oracle import orc
    w, what = cpu_sample(config)
    ora = orc.Oracle.from_workload(w)
    for s in range(warmup):
        ora.coupled_step(w.force_sigma, w.force_seed, s)
    t0 = time.perf_counter()
    for s in range(warmup, warmup + steps):
        ora.coupled_step(w.force_sigma, w.force_seed, s)
    dt = time.perf_counter() - t0
    ora.close()
    return {"value": w.cells * steps / dt / 1e6, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": "%s; %d coupled steps (%d cells, %d nodes) in %.2f s" % (what, steps, w.cells, w.n_nodes, dt)}, dt, w


def oracle_single_thread(config, steps=10):
    """the oracle timed once with ONE thread too, on >= 10 steps (a child process:
    the OpenMP team size is read when the library loads).  Returns MLUPS or None."""
    env = dict(os.environ, OMP_NUM_THREADS="1")
    try:
        out = subprocess.run([sys.executable, os.path.abspath(__file__), "--impl", "reference", "--config", str(config),
                              "--steps", str(steps), "--warmup", "1"], env=env, capture_output=True, text=True, timeout=600)
        return float(json.loads(out.stdout.strip().splitlines()[-1])["value"])
    except Exception:
        return None


def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return 0
    from paper_1312_2234_b200 import workloads as wl
    full = wl.CONFIGS[args.config].__doc__ or ""
    cb, dt, w = time_oracle(args.config, args.steps, args.warmup)
    line = {
        "impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "C%d" % args.config, "sample": cb["sample"]},
        "cpu_baseline": cb,
        "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ---------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------
def run_dist_dry(args):
    """CPU-only check of the N>1 plumbing with gloo: each rank pretends its timed region took
    (rank + 1) * 10 ms; barrier, max-over-ranks and aggregation are the real code."""
    import torch
    import torch.distributed as dist
    rank, world, _ = dist_env()
    if world > 1:
        dist.init_process_group("gloo", init_method="env://")
    dev = torch.device("cpu")
    barrier(dev)
    fake = 0.010 * (rank + 1)
    tmax = max_over_ranks(fake, dev)
    barrier(dev)
    if rank == 0:
        cells = 1000
        print(json.dumps({"metric": METRIC, "value": aggregate(cells, args.steps, world, tmax), "unit": UNIT,
                          "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                          "ms_per_step": 1e3 * tmax / args.steps, "scaling": "weak", "dry_run": True}))
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1312_2234_b200 import binding as plb
    from paper_1312_2234_b200 import build as plb_build
    from paper_1312_2234_b200 import workloads as wl

    rank, world, local_rank = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libplb has no CPU fallback")
    if rank == 0 or world == 1:
        plb_build.build()
    device = torch.device("cuda", local_rank if world > 1 else 0)
    torch.cuda.set_device(device)
    if world > 1:
        dist.init_process_group("nccl", init_method="env://", device_id=device)
    barrier(device)

    w = wl.config(args.config)
    sim = plb.Simulation.from_workload(w, device=str(device))
    coupled = w.n_meshes > 0
    if coupled:
        sim.set_spread_mode(args.spread_mode)
    K, W = args.steps, args.warmup
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def one_step(s, marks=None):
        if coupled:
            if marks is not None: marks[0].record()
            plb.ib_compute_membrane_forces(sim.h, w.force_sigma, w.force_seed, s)
            if marks is not None: marks[1].record()
            plb.ib_spread(sim.h, sim.forcing)
            if marks is not None: marks[2].record()
            plb.lbm_step(sim.h, sim.forcing)
            if marks is not None: marks[3].record()
            plb.ib_interpolate_advance(sim.h)
            if marks is not None: marks[4].record()
        else:
            if marks is not None: marks[2].record()
            plb.lbm_step(sim.h, None)
            if marks is not None: marks[3].record()

    def reset():
        """back to the initial state (SURVEY.md 8(d) protocol: warm-up, reset, then time)"""
        u = None if w.u0 is None else torch.as_tensor(w.u0, dtype=torch.float32).to(device).contiguous()
        sim.set_equilibrium(None, u, w.noise_amp, w.noise_seed)
        if coupled:
            sim.write_nodes(np.ascontiguousarray(w.mesh_xyz.reshape(-1, 3)))
        torch.cuda.synchronize(device)

    # ---- device-resident leg: inputs already in HBM, CUDA events on the launching stream
    clocks = ClockSampler(device.index)
    for s in range(W):
        one_step(s)
    reset()
    marks = [[ev() for _ in range(5)] for _ in range(K)]
    t_beg, t_end = ev(), ev()
    barrier(device)
    launches0 = sim.launch_count()
    clocks.mark()
    t_beg.record()
    for s in range(K):
        one_step(W + s, marks[s])
    t_end.record()
    barrier(device)
    clk = clocks.stop()
    launches = sim.launch_count() - launches0
    # ---- the state the timed run produced: sticky error flags, non-finite / non-positive cells,
    # mass (P1: halfway bounce-back and the Guo force conserve it exactly), nodes inside the channel
    state = {"status": "ok", "steps_from_initial_state": K}
    try:
        sim.status()
    except plb.PlbError as err:
        state["status"] = "error %d: %s" % (err.code, err)
    state["bad_cells"] = int(sim.check_finite())
    rho_end, u_end = sim.read_macros()
    state["mean_rho_minus_1"] = float(rho_end.double().mean().item() - 1.0)
    state["max_speed"] = float(u_end.abs().max().item())
    if coupled:
        X_end = sim.read_nodes()
        state["nodes_finite"] = bool(np.isfinite(X_end).all())
        state["max_node_displacement"] = float(np.abs(X_end - w.mesh_xyz.reshape(-1, 3)).max())
        state["spread_form"] = {0: "auto", 1: "scatter", 2: "aggregate", 3: "gather"}[sim.spread_mode()]
    del rho_end, u_end
    seconds = max_over_ranks(t_beg.elapsed_time(t_end) * 1e-3, device)
    value = aggregate(w.cells, K, world, seconds)
    lbm_ms = sum(m[2].elapsed_time(m[3]) for m in marks) / K
    split = {"lbm_step": lbm_ms}
    if coupled:
        split.update(ib_compute_membrane_forces=sum(m[0].elapsed_time(m[1]) for m in marks) / K,
                     ib_spread=sum(m[1].elapsed_time(m[2]) for m in marks) / K,
                     ib_interpolate_advance=sum(m[3].elapsed_time(m[4]) for m in marks) / K)
    step_ms = 1e3 * t_beg.elapsed_time(t_end) * 1e-3 / K
    ib_share = (sum(split.values()) - lbm_ms) / sum(split.values())

    # ---- end-to-end leg: the membrane state crosses the C-ABI as HOST buffers every step
    e2e = None
    if not args.no_e2e:
        e2e = run_e2e(sim, w, K, W, world, device, plb, one_step)

    # ---- roofline of the dominant kernel (lbm_step_kernel: 152 B per cell per launch)
    peak, peak_src = hbm_peak()
    achieved = BYTES_PER_CELL * w.cells / (lbm_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": "lbm_step_vec_kernel<MODE,4,128,4,WALLS> (lbm_step)", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": ncu_traffic(args.config),
                "traffic_source": "static: profiles/lbm_dram_traffic.txt (one ncu --set full capture of this kernel; "
                                  "not measured in this run)",
                "peak_source": peak_src,
                "algorithmic_bytes_per_launch": BYTES_PER_CELL * w.cells, "avg_launch_ms": lbm_ms,
                "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS,
                "lbm_only_mlups": w.cells / (lbm_ms * 1e-3) / 1e6}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": 1e3 * seconds / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": describe(w), "cells": w.cells, "nodes": w.n_nodes, "tau": w.tau,
                   "l2": "inputs exceed L2 (%.2f GB of populations per step)" % (BYTES_PER_CELL * w.cells / 1e9),
                   "multi_gpu": "replicas only (no exchange step in this build)", "notes": w.notes},
        "clocks": clk, "e2e": e2e, "gpu_launches": launches, "roofline": roofline,
        "coupled_steps_per_s": K * world / seconds, "split_ms": split, "ib_share": ib_share, "state_check": state,
        "step_ms_rank0": step_ms,
    }
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cb, _, _ = time_oracle(args.config, 100 if args.config == 4 else 20, 2)
        cb["value_1_thread"] = oracle_single_thread(args.config)
        line["cpu_baseline"] = cb
    elif rank == 0:
        line["cpu_baseline"] = None
    if rank == 0:
        print(json.dumps(line))
    sim.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_e2e(sim, w, K, W, world, device, plb, one_step):
    """Same metric through the C-ABI with HOST buffers: every step the node positions go in from
    pinned host memory (ib_write_nodes) and come back out (ib_read_nodes), copies inside the timed
    region.  Without meshes (C2) the step's result read back is the density field."""
    import numpy as np
    import torch
    coupled = w.n_meshes > 0
    if coupled:
        n = sim.n_nodes
        pinned = torch.empty((n, 3), dtype=torch.float64).pin_memory()
        X = pinned.numpy()
        plb.ib_read_nodes(sim.h, X)
        h2d = d2h = n * 24
    else:
        pinned = torch.empty(w.cells, dtype=torch.float32).pin_memory()
        rho = torch.empty(w.cells, dtype=torch.float32, device=device)
        h2d, d2h = 0, w.cells * 4

    def e2e_step(s):
        if coupled:
            plb.ib_write_nodes(sim.h, X)
            one_step(s)
            plb.ib_read_nodes(sim.h, X)
        else:
            one_step(s)
            plb.lbm_read_macros(sim.h, rho, None)
            pinned.copy_(rho, non_blocking=False)

    for s in range(3):
        e2e_step(s)
    barrier(device)
    t0 = time.perf_counter()
    for s in range(K):
        e2e_step(s)
    barrier(device)
    dt = max_over_ranks(time.perf_counter() - t0, device)
    return {"value": aggregate(w.cells, K, world, dt), "unit": UNIT, "h2d_bytes_per_step": h2d,
            "d2h_bytes_per_step": d2h, "ms_per_step": 1e3 * dt / K,
            "what": "ib_write_nodes(pinned host) -> 4 coupled calls -> ib_read_nodes(pinned host), per step"
                    if coupled else "lbm_step -> lbm_read_macros -> density field to pinned host, per step"}


def main(argv=None):
    args = parse_args(argv)
    if args.dist_dry_run:
        return run_dist_dry(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
