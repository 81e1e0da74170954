#!/usr/bin/env python
"""bench.py -- SWE FP64 cell-updates/s on B200 (BASELINE.json metric) + HBM roofline fraction.

A "step" is one pass of the whole hot path (gather, reconstruction, HLLC
fluxes, sources, friction, update, CFL reduction) over the whole mesh = one solver time step.
Default workload: BASELINE.json configs[3] (river, 13,005,000 cells) -- the largest single-GPU
config and one of the ">= 4M-cell meshes" the north_star's roofline target is quoted on; its
2.5 GB of device data are far larger than the 126 MB L2, so no L2 flush is needed between steps.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl reference]

The line also carries a "wet" record: BASELINE.json configs[2] (lake at rest, 4,000,000 cells, every
cell wet) timed the same way in the same process -- the regime in which every cell does the method's
work and the kernel is furthest from the HBM roof.  roofline.frac charges 156 algorithmic bytes to the
cells of active tiles and 64 bytes to the cells of all-dry tiles (counted on the device during the
timed steps), so it cannot exceed ~1; the fixed-156 figure is kept as frac_fixed_156.

N > 1 (torchrun): the path does not shard ("replicas only"): every rank runs the same
workload independently, value = all ranks' cell-updates / max-over-ranks device time.
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

from paper_2010_14416_b200 import workloads as W  # noqa: E402

ALGO_BYTES_PER_CELL = 156.0   # 132 B read + 24 B written per cell-update
METRIC = "SWE FP64 cell-updates/s on 1 B200; achieved HBM GB/s vs peak"   # BASELINE.json "metric"
UNIT = "cell-updates/s"


def make_workload(name: str):
    if name == "config1":
        return W.config1()
    if name == "config2":
        return W.config2()
    if name == "config3":
        return W.config3()
    if name == "config4":
        return W.config4()
    if name.startswith("sweep_"):
        return W.config5(name[len("sweep_"):])
    raise SystemExit(f"unknown workload {name}")


def make_sample(name: str):
    """Bounded sample of the same workload for the CPU oracle: same recipe, fewer squares."""
    if name == "config4":
        return W.config4(nx=1275, ny=319), "config4 recipe at 1275x319 squares (813,450 cells)"
    if name == "config3":
        return W.config3(nx=1000, ny=500), "config3 recipe at 1000x500 squares (1,000,000 cells)"
    if name.startswith("sweep_") and W.SWEEP_NY[name[6:]] > 316:
        return W.config5("0.5M"), "config5 recipe at 0.5M cells"
    return make_workload(name), "the full workload"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for ts, r in self.rows if t0 - 0.05 <= ts <= t1 + 0.15 and len(r) >= 7] or \
               [r for _, r in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = sorted(float(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(r[3 + k].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "reasons": reasons,
                "samples": len(rows), "power_w_max": max(float(r[2]) for r in rows)}


def time_oracle(w, steps: int, warmup: int, threads=None):
    """The oracle as it stands on the host cores: returns (cell-updates/s, threads used)."""
    from oracle.swe_oracle import OracleSolver
    o = OracleSolver.from_workload(w)
    one_thread = None
    if threads is None:   # pick the thread count that is actually fastest on this box
        best = (0.0, 1)
        for n in sorted({1, 2, 4, 8, 16, 32, os.cpu_count() or 1}):
            if n > (os.cpu_count() or 1):
                continue
            o.set_threads(n)
            o.compute_dt()
            o.run(1)                       # spin the thread team up
            t0 = time.perf_counter()
            o.run(3)
            r = 3 * w.ncells / (time.perf_counter() - t0)
            if n == 1:
                one_thread = r
            if r > best[0]:
                best = (r, n)
        threads = best[1]
        o.set_state(w.h, w.hu, w.hv)
    o.set_threads(threads)
    o.compute_dt()
    o.run(warmup)
    t0 = time.perf_counter()
    done = o.run(steps)
    dt = time.perf_counter() - t0
    time_oracle.one_thread = one_thread        # 3-step probe with a single thread
    return done * w.ncells / dt, threads, dt


def run_reference(args, rank: int, world: int):
    """--impl reference: the oracle, as it stands, on the box's host cores (rank 0 only), with the
    warm-up and step counts it was asked for (a step of the bounded sample takes milliseconds)."""
    if rank != 0:
        return
    sample, what = make_sample(args.workload)
    steps = max(1, args.steps)
    value, threads, secs = time_oracle(sample, steps, args.warmup)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": args.workload, "sample": what},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": what},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def max_over_ranks(values, world: int, device="cpu"):
    """Element-wise max of a list of floats over all ranks (the job time is the slowest rank's)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def job_throughput(cells_per_rank: int, steps: int, world: int, ms_max: float) -> float:
    """Replicas only: every rank steps its own copy; units of all ranks / slowest rank's time."""
    return float(cells_per_rank) * steps * world / (ms_max * 1e-3)


STATE_BYTES_DRY = 64.0        # an all-dry tile's update is the identity: its 32-byte records in and out


def roofline_record(n, kernel_ms, active_share, list_share, step_bytes, tiles, peak, peak_src, quiet_share=None,
                    kernel_name=None, stolen_share=None):
    """HBM roofline of one launch of the step kernel (= one time step of the whole mesh).

    frac cannot exceed ~1 for a correct kernel: it charges the SURVEY's 156 algorithmic bytes only
    to the cells of tiles that did the method's work in the timed steps, 64 bytes (record in and
    out) to the cells of all-dry tiles that were moved, whose update is the identity, and nothing to
    the cells of quiet tiles, whose records are in place in both state buffers and are not touched
    (all three counted on the device).
    traffic = the bytes this launch requested from memory according to the library's own table
    sizes and the same counters (swe_get_step_bytes), not a stored constant."""
    sec = kernel_ms * 1e-3
    qs = quiet_share or 0.0
    algo = (ALGO_BYTES_PER_CELL * active_share + STATE_BYTES_DRY * max(0.0, 1.0 - active_share - qs)) * n
    fixed = ALGO_BYTES_PER_CELL * n
    return {"bound": "hbm", "achieved": algo / sec / 1e9, "peak": peak, "unit": "GB/s",
            "frac": algo / sec / 1e9 / peak, "traffic": step_bytes,
            "traffic_kind": "bytes requested per launch, from the library's table sizes and this run's "
                            "device counters (swe_get_step_bytes); ncu dram__bytes cross-check in profiles/",
            "achieved_traffic": step_bytes / sec / 1e9, "frac_traffic": step_bytes / sec / 1e9 / peak,
            "algorithmic_bytes_per_launch": algo, "algorithmic_bytes_per_cell_active_tile": ALGO_BYTES_PER_CELL,
            "algorithmic_bytes_per_cell_dry_tile": STATE_BYTES_DRY, "algorithmic_bytes_per_cell_quiet_tile": 0.0,
            "active_tile_share": active_share, "edge_list_share": list_share, "quiet_tile_share": quiet_share,
            "stolen_tile_share": stolen_share,
            # cells of tiles that did the method's arithmetic, per second (value counts every cell of the mesh)
            "active_cell_updates_per_s": active_share * n / sec,
            "achieved_fixed_156": fixed / sec / 1e9, "frac_fixed_156": fixed / sec / 1e9 / peak,
            "frac_of_nominal_8TBs": algo / sec / 1e9 / 8000.0,
            "kernel": kernel_name or f"swe_step_kernel<{tiles['tile_cells']}>", "peak_source": peak_src}


def measure_device(B, w, args, dev, order, loop, barrier, world, sampler=None):
    """W warm-up steps, then exactly K timed steps in one swe_run, CUDA events on the mesh's stream."""
    import torch
    n = w.ncells
    t_build = time.perf_counter()
    kern = {"tiled": B.KERNEL_TILED, "edge": B.KERNEL_EDGE_TWO_PASS}[args.kernel]
    m = B.SweMesh.from_workload(w, ordering=order, loop_mode=loop, block_size=args.block, kernel=kern).bind_device(dev)
    t_build = time.perf_counter() - t_build
    m.set_state(w.h, w.hu, w.hv)
    m.run(args.warmup)
    for _ in range(2 if args.steps % 2 else 1):   # untimed: instantiates every CUDA graph the timed
        m.run(args.steps)                          # call will replay (graphs are keyed by buffer parity)
    m.sync()
    launches0 = m.get_launch_info()["kernel_launches"]
    st0 = m.get_stats()
    if sampler is not None:
        sampler.start()
        time.sleep(0.25)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0 = time.time()
    ev0.record(m.stream)
    m.run(args.steps)
    ev1.record(m.stream)
    barrier()
    t1 = time.time()
    ms = ev0.elapsed_time(ev1)
    clocks = sampler.stop(t0, t1) if sampler is not None else None
    info = m.get_launch_info()
    tiles = m.get_tile_info()
    launches = info["kernel_launches"] - launches0 - 1          # minus the get_stats reduction above
    st = m.get_stats()
    tile_steps = float(tiles["ntiles"] * args.steps)
    # share of (tile, step) pairs that were not all dry / whose edge list was read
    active_share = (st["active_tile_steps"] - st0["active_tile_steps"]) / tile_steps
    list_share = (st["edge_list_fetches"] - st0["edge_list_fetches"]) / tile_steps
    quiet_share = (st["quiet_tile_steps"] - st0["quiet_tile_steps"]) / tile_steps
    stolen_share = (st["stolen_tile_steps"] - st0["stolen_tile_steps"]) / tile_steps
    step_bytes = m.get_step_bytes(active_share * tiles["ntiles"], list_share * tiles["ntiles"],
                                  quiet_share * tiles["ntiles"])
    return dict(quiet_share=quiet_share, stolen_share=stolen_share, mesh=m, ms=ms, clocks=clocks, info=info, tiles=tiles, launches=launches, stats=st,
                active_share=active_share, list_share=list_share, step_bytes=step_bytes, t_build=t_build)


def run_gpu(args, rank: int, world: int, local_rank: int):
    import torch
    import torch.distributed as dist
    from paper_2010_14416_b200 import binding as B

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: CUDA is not available and there is no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = f"cuda:{local_rank}"

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    w = make_workload(args.workload)
    n = w.ncells
    order = {"hilbert": B.ORDER_HILBERT, "rcm": B.ORDER_RCM, "identity": B.ORDER_IDENTITY}[args.ordering]
    loop = {"auto": B.LOOP_AUTO, "graph": B.LOOP_GRAPH, "persistent": B.LOOP_PERSISTENT,
            "launch": B.LOOP_LAUNCH, "cluster": B.LOOP_CLUSTER}[args.loop]
    # ---- device-resident leg of the headline workload -------------------------------------
    r = measure_device(B, w, args, dev, order, loop, barrier, world, ClockSampler(local_rank))
    m, ms, info, tiles, stats = r["mesh"], r["ms"], r["info"], r["tiles"], r["stats"]

    # ---- end-to-end leg through the C ABI with host buffers: set_state + run(K) + get_state ----
    pin = [torch.empty(n, dtype=torch.float64).pin_memory() for _ in range(6)]
    hin = [p.numpy() for p in pin[:3]]
    hout = [p.numpy() for p in pin[3:]]
    for dst, src in zip(hin, (w.h, w.hu, w.hv)):
        dst[:] = src
    barrier()
    e0 = time.perf_counter()
    m.set_state(*hin)
    m.run(args.steps)
    m.get_state_into(*hout)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - e0
    m.destroy()
    del pin, hin, hout

    # ---- all-wet leg: BASELINE.json configs[2] (lake at rest, 4M cells, every cell does the
    # method's work) timed the same way in the same process, so that the record carries the
    # regime in which the kernel is furthest from the HBM roof ------------------------------
    wet = None
    if args.wet and args.workload != "config3":
        w3 = make_workload("config3")
        r3 = measure_device(B, w3, args, dev, order, loop, barrier, world)
        r3["mesh"].destroy()
        wet = (w3, r3)

    vals = [ms, e2e_s * 1e3] + ([wet[1]["ms"]] if wet else [])
    vals = max_over_ranks(vals, world, dev)
    ms, e2e_ms = vals[0], vals[1]
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    total_updates = float(n) * args.steps * world
    value = job_throughput(n, args.steps, world, ms)
    peak, peak_src = load_peaks()
    kernel_ms = ms / args.steps                       # one step kernel launch per step
    if args.cpu_baseline:
        sample, what = make_sample(args.workload)
        cpu_value, cpu_threads, _ = time_oracle(sample, 10 if sample.ncells > 300000 else 100, 2)
    else:                                   # profiling / sweep runs: the oracle leg is skipped and says so
        cpu_value, cpu_threads, what = None, 0, "skipped (--no-cpu-baseline)"

    def l2_policy(cells):
        return "inputs larger than L2 (no flush)" if cells * 164 > 2 * 126e6 \
            else "working set fits in L2; a time loop re-reads its own output, no flush"

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "name": w.name, "cells": n, "nodes": w.nnodes,
                   "ordering": args.ordering, "loop_mode": info["loop_mode"],
                   "grid": info["grid"], "block": info["block"], "tile_cells": tiles["tile_cells"],
                   "edge_evaluations_per_cell": round(tiles["edges_per_cell"], 4),
                   "smem_bytes_per_block": tiles["smem_bytes"], "l2_policy": l2_policy(n),
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "mesh_build_s": round(r["t_build"], 2), "wet_fraction_end": 1.0 - stats["n_dry"] / n,
                   "n_clamped": stats["n_clamped"],
                   "counts": "every cell of the mesh per step; all-dry tiles whose neighbourhood was dry a step ago "
                             "(roofline.quiet_tile_share) are left untouched because their update is the identity and "
                             "both state buffers hold it: the state after K steps is bit for bit what computing every "
                             "cell gives (tests/test_gpu_parity.py); 'wet' is the regime without any shortcut"},
        "roofline": roofline_record(n, kernel_ms, r["active_share"], r["list_share"], r["step_bytes"],
                                    tiles, peak, peak_src, r["quiet_share"],
                                    "swe_edge_pass_kernel + swe_cell_pass_kernel" if args.kernel == "edge" else None,
                                    r["stolen_share"]),
        "cpu_baseline": {"value": cpu_value, "unit": UNIT, "cores": cpu_threads, "kind": "oracle",
                         "sample": what, "value_1_thread": getattr(time_oracle, "one_thread", None),
                         "host_cores": os.cpu_count()},
        "e2e": {"value": total_updates / (e2e_ms * 1e-3), "unit": UNIT,
                "h2d_bytes_per_step": 24.0 * n / args.steps, "d2h_bytes_per_step": 24.0 * n / args.steps,
                "job": "swe_set_state(pinned host) + swe_run(K) + swe_get_state(pinned host); "
                       "bytes are per job / K"},
        "gpu_launches": r["launches"], "clocks": r["clocks"],
    }
    if wet:
        w3, r3 = wet
        ms3 = vals[2]
        line["wet"] = {
            "workload": "config3", "name": w3.name, "cells": w3.ncells, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms3 / args.steps,
            "value": job_throughput(w3.ncells, args.steps, world, ms3), "unit": UNIT,
            "wet_fraction_end": 1.0 - r3["stats"]["n_dry"] / w3.ncells, "l2_policy": l2_policy(w3.ncells),
            "grid": r3["info"]["grid"], "block": r3["info"]["block"], "gpu_launches": r3["launches"],
            "roofline": roofline_record(w3.ncells, ms3 / args.steps, r3["active_share"], r3["list_share"],
                                        r3["step_bytes"], r3["tiles"], peak, peak_src, r3["quiet_share"],
                                        None, r3["stolen_share"]),
        }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--workload", default="config4")
    ap.add_argument("--ordering", default="hilbert", choices=["hilbert", "rcm", "identity"])
    ap.add_argument("--loop", default="auto", choices=["auto", "graph", "persistent", "launch", "cluster"])
    ap.add_argument("--block", type=int, default=0, help="cells per tile = threads per block (0 = default)")
    ap.add_argument("--kernel", default="tiled", choices=["tiled", "edge"],
                    help="tiled = the fused tile kernel (default); edge = the edge-centric two-pass alternative (A/B only)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", dest="cpu_baseline", action="store_false",
                    help="skip the oracle-on-host-cores leg (sweeps and runs under ncu; the default line carries it)")
    ap.add_argument("--no-wet", dest="wet", action="store_false",
                    help="skip the all-wet leg (config3) that the default run times beside the headline workload")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_gpu(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
