#!/usr/bin/env python
"""Benchmark of the hot path: cell-updates/s of the fp64 two-stage MHD step and the
fraction of the B200 HBM roofline reached by the dominant (stage) kernels.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl reference]

Workload (default ``random_uniform_4096``): BASELINE.json configs[3], the
configuration the north_star quotes its target on -- uniform periodic grid of
16x16x16 blocks of 8^3 cells (2,097,152 cells), seeded Gaussian perturbations.
Both state buffers (2 x 453 MB) are far larger than the 126 MB L2, so no L2 flush
is needed between timed steps.  A "step" is one full two-stage step: stage 1,
ghost fill, stage 2, ghost fill, dt bookkeeping.  The stage kernels also write their outer
cell layers into the face ghosts of same-level neighbours, so on this uniform periodic grid the
ghost fills enqueue nothing: 3 kernel launches per step (stage, stage, tick).

One JSON line is printed by rank 0.  N > 1 runs N independent replicas ("replicas
only"): the path has no sharding and no collective.
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
sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402

METRIC = "cell-updates/sec (fp64 MHD step)"
UNIT = "cell-updates/s"

WORKLOADS = {
    "alfven_8": lambda: wl.alfven(),
    "orszag_tang_512": lambda: wl.orszag_tang(),
    "brio_wu_amr_352": lambda: wl.brio_wu_amr(),
    "random_uniform_512": lambda: wl.random_uniform((8, 8, 8)),
    "random_uniform_1024": lambda: wl.random_uniform((16, 8, 8)),
    "random_uniform_2048": lambda: wl.random_uniform((16, 16, 8)),
    "random_uniform_4096": lambda: wl.random_uniform((16, 16, 16)),
    "random_uniform_8192": lambda: wl.random_uniform((32, 16, 16)),
    "random_uniform_16384": lambda: wl.random_uniform((32, 32, 16)),
    "random_uniform_32768": lambda: wl.random_uniform((32, 32, 32)),
    "magnetosphere": lambda: wl.magnetosphere(),
    # the paper's fast-wave test at its 1-GPU size m = 6 (Table 2/3: 8^3 roots, one octant refined = 960 blocks;
    # 8^3-cell blocks here, 10^3 in the paper), HLL-type "Linde" flux (Q-F4), CFL 0.8
    "fast_wave_960_linde": lambda: wl.fast_wave((8, 8, 8), flux_type=1),
    "fast_wave_960": lambda: wl.fast_wave((8, 8, 8)),
    # the paper's operational time stepping (L391-397): one stage, first order, CFL 0.85
    "random_uniform_4096_1stage": lambda: dict(wl.random_uniform((16, 16, 16)), n_stage=1, n_order=1, cfl=0.85),
    "magnetosphere_1stage": lambda: dict(wl.magnetosphere(), n_stage=1, n_order=1, cfl=0.85),
}
DEFAULT_WORKLOAD = "random_uniform_4096"

# algorithmic bytes per cell and stage launch: the 12^3 x 8 tile read once
# (216 B/cell) + 64 B/cell written; stage 2 also reads U^n of the physical cells (64).  PUSH: the
# face ghosts the same launch writes into same-level neighbours (6 faces x 128 cells x 64 B / 512
# cells = 96 B/cell, the face-slab part of the 152 B/cell a stored-ghost fill writes); counted
# only for the blocks that push (all of them on a uniform periodic grid).
STAGE1_BYTES_PER_CELL = 216 + 64
STAGE2_BYTES_PER_CELL = 216 + 64 + 64
PUSH_BYTES_PER_CELL = 96
FILL_BYTES_PER_CELL = 304      # one stored-ghost fill: 152 read + 152 written per cell of a filled block


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def _source_hash():
    """Hash of the sources of the stage kernels (the kernels `roofline` is about): ties a committed ncu
    capture to a build."""
    import hashlib
    h = hashlib.sha256()
    for f in ("batl_stage_fused.cu", "batl_device.cuh", "mhd_physics.cuh", "batl_grid.hpp"):
        h.update(open(os.path.join(ROOT, "paper_2501_06717_b200", "csrc", f), "rb").read())
    return h.hexdigest()[:12]


def _traffic(kernels, workload=None):
    """Mean DRAM bytes (read + write) per launch of `kernels` from the newest committed `ncu --set full`
    capture (profiles/r*_traffic.csv).  ncu cannot run inside a timed run, so the figure is quoted only
    when the capture was taken on the sources of this build (the csv carries their hash) and on the
    workload being run (the captures are of the default workload); else None."""
    import csv
    import glob
    if workload is not None and workload != DEFAULT_WORKLOAD:
        return None, f"the committed capture is of {DEFAULT_WORKLOAD}: not quoted for {workload}"
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_traffic.csv")))
    if not files:
        return None, "no capture"
    try:
        rows = list(csv.DictReader(open(files[-1])))
        if not rows or rows[0].get("source_hash") != _source_hash():
            return None, os.path.basename(files[-1]) + " is of another build (see profiles/): not quoted"
        tot = [int(r["dram_bytes_read"]) + int(r["dram_bytes_write"]) for r in rows if r["kernel"] in kernels]
        return (sum(tot) / len(tot), os.path.basename(files[-1])) if tot else (None, "kernel not in capture")
    except Exception as e:  # malformed file: say so, do not guess
        return None, f"unreadable capture: {e}"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(mx)) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def _initial_state(cfg, blocks):
    return wl.initial_conserved(cfg, blocks)


# --------------------------------------------------------------------------------------
def oracle_rate(cfg, target_s=15.0, max_steps=60):
    """cell-updates/s of the CPU oracle as it stands (never tuned) on the workload itself:
    one calibration step, then as many steps as fit in about target_s seconds."""
    import oracle
    o = oracle.Oracle(cfg)
    W = wl.initial_primitive(cfg, o.blocks())
    o.set_primitive(W)
    t0 = time.perf_counter()
    o.step(1)
    t1 = time.perf_counter() - t0
    n = int(max(1, min(max_steps, round(target_s / max(t1, 1e-3)))))
    t0 = time.perf_counter()
    o.step(n)
    dt = time.perf_counter() - t0
    return o.n_blocks * 512 * n / dt, dt, n, oracle.max_threads()


def max_over_ranks(value, device, world):
    """Maximum of a per-rank scalar over all ranks (the timing rule for N > 1)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    tt = torch.tensor([float(value)], device=device, dtype=torch.float64)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores, same metric, same workload (one
    oracle step of the named workload per bench step; --reference-blocks NX NY NZ shrinks the block
    grid of the random_uniform recipe, and the line then names the workload it ran)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    name = args.workload
    if args.reference_blocks:
        nb = tuple(args.reference_blocks)
        name = "random_uniform_%d" % (nb[0] * nb[1] * nb[2])
        cfg = wl.random_uniform(nb)
    else:
        cfg = WORKLOADS[name]()
    import oracle
    o = oracle.Oracle(cfg)
    o.set_primitive(wl.initial_primitive(cfg, o.blocks()))
    cells = o.n_blocks * 512
    for _ in range(args.warmup):
        o.step(1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.step(1)
    dt = time.perf_counter() - t0
    rate = cells * args.steps / dt
    n_stage, n_order = int(cfg.get("n_stage", 2)), int(cfg.get("n_order", 2))
    sample = f"{name}: {o.n_blocks} blocks, {cells} cells, 1 full oracle step per bench step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(1, args.steps),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": _config(name, cfg, o.n_blocks, cells, n_stage, n_order, 1, None),
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def _config(name, cfg, n_blocks, cells, n_stage, n_order, world, state_bytes):
    """The `config` object: the same keys for both arms, so that the driver can compare them."""
    c = {"workload": name, "blocks": n_blocks, "cells": cells, "block": "8^3+2 ghost layers",
         "scheme": "2-stage Rusanov, MC limiter" if n_stage == 2 and n_order == 2 else f"{n_stage}-stage Rusanov, order {n_order}",
         "cfl": cfg["cfl"], "parallelism": f"replicas x{world}"}
    if state_bytes is not None:
        c["l2"] = "state buffers (2 x %.0f MB) exceed the 126 MB L2; no flush" % (state_bytes / 1e6)
    return c


def run_gpu(args):
    import torch
    import torch.distributed as dist
    import paper_2501_06717_b200 as batl

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = WORKLOADS[args.workload]()
    if args.sharded and world > 1:
        return run_sharded(args, cfg, dev, world, rank, barrier)
    g = batl.Grid(cfg)
    cells = g.n_blocks * 512
    U0 = _initial_state(cfg, g.blocks())
    stream = torch.cuda.Stream(device=dev)
    g.bind(dev, stream)
    h_in = torch.from_numpy(U0).pin_memory()
    h_out = torch.empty_like(h_in).pin_memory()
    d_in = h_in.to(dev)
    g.set_state(d_in)
    stream.synchronize()

    # ---- device-resident timing: inputs already in HBM -------------------------------
    for _ in range(args.warmup):
        g.step(1)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    n0 = g.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record(stream)
    g.step_async(args.steps)
    ev1.record(stream)
    barrier()
    ms = ev0.elapsed_time(ev1)
    launches = g.launch_count() - n0
    clocks = sampler.stop() if rank == 0 else None
    w, t_sim, dt_last = g.step(0)
    ms = max_over_ranks(ms, dev, world)
    value = world * cells * args.steps / (ms * 1e-3)

    # ---- per-kernel durations (CUDA events on the bound stream around every launch) ----
    g.set_state(d_in)
    g.step(2)
    g.phase_timers(True)
    n_prof = min(args.steps, 10)
    g.step(n_prof)
    ph = g.phase_timers(False)
    n_stage = int(cfg.get("n_stage", 2))
    n_order = int(cfg.get("n_order", 2))
    stage_ms_per_launch = ph["stage_ms"] / (n_stage * n_prof)
    # faces whose ghosts the stage kernel writes itself (same-level neighbour) / blocks left to the fill kernel
    _, dlev = g.neighbors()
    face_dirs = [12, 14, 10, 16, 4, 22]                 # -x +x -y +y -z +z in dir = (di+1) + 3(dj+1) + 9(dk+1)
    dl = np.asarray(dlev)[:, face_dirs]
    pushed = float((dl == 0).mean())
    if int(cfg.get("prolong_order", 1)) == 1 and not int(cfg.get("flux_correction", 0)):
        # first-order prolongation is pushed too: a face with finer neighbours is 4 x 128 fine ghost cells
        pushed += 4.0 * float((dl == -1).mean())
    filled = g.kernel_counts()["fill_list"] / g.n_blocks
    s1 = STAGE1_BYTES_PER_CELL + PUSH_BYTES_PER_CELL * pushed
    s2 = STAGE2_BYTES_PER_CELL + PUSH_BYTES_PER_CELL * pushed
    alg_bytes = (0.5 * (s1 + s2) if n_stage == 2 else s1) * cells
    step_bytes = (s1 + s2 if n_stage == 2 else s1) + n_stage * FILL_BYTES_PER_CELL * filled
    achieved = alg_bytes / (stage_ms_per_launch * 1e-3) / 1e9
    peak, peak_src = _peaks()
    traffic, traffic_src = _traffic(("stage<1>", "stage<2>") if n_stage == 2 else ("stage<3>",), args.workload)
    roofline = {
        "bound": "hbm", "kernel": "stage kernels (stage 1 + stage 2, mean per launch; they also write the face ghosts of same-level neighbours)",
        "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
        "frac_of_nominal_8TBs": achieved / 8000.0, "peak_source": peak_src,
        "algorithmic_bytes_per_launch": alg_bytes,
        "algorithmic_bytes_per_cell": {"stage1": s1, "stage2": s2 if n_stage == 2 else None, "whole_step": step_bytes,
                                       "faces_pushed": pushed, "blocks_on_fill_list": filled},
        "ms_per_launch": stage_ms_per_launch,
        "traffic": traffic, "traffic_source": traffic_src,
        "phase_ms_per_step": {k: v / n_prof for k, v in ph.items()},
        "whole_step_hbm_frac": step_bytes * (cells * args.steps / (ms * 1e-3)) / (peak * 1e9),
    }

    # ---- end to end through the C ABI with HOST buffers ---------------------------------
    # Every step: batl_set_state from pinned host memory (H2D 134 MB at 4,096 blocks, ghost fill), mhd_step,
    # batl_get_state into pinned host memory (D2H).  One pipeline is bound by the two serial PCIe copies
    # (2 x 2.7 ms at the ~50 GB/s per direction measured on this box against a 0.5 ms step); several grids
    # driven by one host thread each (ctypes releases the GIL) let the copies of one overlap the step and the
    # opposite copy of the others.  Three keep both directions of the link busy (95 % of the copy bound; two
    # reach 83 %).  Both figures are reported; `value` is the multi-grid one.
    n_e2e = max(1, min(args.steps, 20))
    n_pipe = max(1, args.e2e_pipelines)

    def pipeline(grid, out, n, gate=None):
        if gate is not None:
            gate.wait()
        for _ in range(n):
            grid.set_state(h_in)         # H2D of the step's input (pinned), ghost fill
            grid.step(1)
            grid.get_state(out=out)      # D2H of the step's result (pinned)

    pipeline(g, h_out, 1)                                      # warm-up of the host path
    barrier()
    t0 = time.perf_counter()
    pipeline(g, h_out, min(n_e2e, 5))
    barrier()
    serial_s = max_over_ranks(time.perf_counter() - t0, dev, world) / min(n_e2e, 5)
    more = []
    for _ in range(n_pipe - 1):
        gq = batl.Grid(cfg)
        gq.bind(dev, torch.cuda.Stream(device=dev))
        hq = torch.empty_like(h_in).pin_memory()
        pipeline(gq, hq, 1)
        more.append((gq, hq))
    barrier()
    gate = threading.Barrier(n_pipe)
    ths = [threading.Thread(target=pipeline, args=(gq, hq, n_e2e, gate)) for gq, hq in more]
    t0 = time.perf_counter()
    for th in ths:
        th.start()
    pipeline(g, h_out, n_e2e, gate)
    for th in ths:
        th.join()
    barrier()
    e2e_s = max_over_ranks(time.perf_counter() - t0, dev, world)
    for gq, _ in more:
        gq.close()
    e2e = {"value": world * cells * n_pipe * n_e2e / e2e_s, "unit": UNIT, "steps": n_pipe * n_e2e,
           "h2d_bytes_per_step": int(h_in.numel() * 8), "d2h_bytes_per_step": int(h_out.numel() * 8),
           "pipeline": f"{n_pipe} grids, one host thread each: the copies of one overlap the step and the opposite "
                       "copy of the others",
           "single_pipeline_value": world * cells / serial_s}

    if rank == 0:
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            r, secs, n_cpu, cores = oracle_rate(cfg)
            cpu = {"value": r, "unit": UNIT, "cores": cores, "kind": "oracle",
                   "sample": f"the same workload ({args.workload}, {cells} cells), {n_cpu} oracle steps, {secs:.1f} s"}
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": _config(args.workload, cfg, g.n_blocks, cells, n_stage, n_order, world, g.state_bytes),
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
            "kernels": g.kernel_counts(),
            "roofline": roofline, "cpu_baseline": cpu,
            "sim": {"t": t_sim, "dt_last": dt_last, "warn": w},
        }
        print(json.dumps(out))
    g.close()
    if world > 1:
        dist.destroy_process_group()


def run_sharded(args, cfg, dev, world, rank, barrier):
    """--sharded (opt-in, N > 1): ONE grid split over the N GPUs (row f4: contiguous Morton segments, ghost
    writes through mapped peer buffers, a barrier per stage and an all-reduce(min) of dt per step), i.e.
    strong scaling.  The default N > 1 run stays N independent replicas (north_star: no sharding).  This
    path has run with emulated ranks and with two processes sharing one GPU (tests/test_sharded.py); no
    multi-GPU box was available to measure it."""
    import torch
    import torch.distributed as dist
    from paper_2501_06717_b200 import dist as bd
    stream = torch.cuda.Stream(device=dev)
    g = bd.make_rank(cfg, dev, stream)
    cells = g.n_blocks * 512
    U0 = _initial_state(cfg, g.blocks())
    g.set_state(torch.from_numpy(U0).to(dev))
    st = bd.ShardedStepper([g], bd.NcclTransport())
    st.step(args.warmup)
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = g.launch_count()
    ev0.record(stream)
    st.step(args.steps)
    ev1.record(stream)
    barrier()
    ms = max_over_ranks(ev0.elapsed_time(ev1), dev, world)
    if rank == 0:
        n_stage = int(cfg.get("n_stage", 2))
        print(json.dumps({
            "metric": METRIC, "value": cells * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": dict(_config(args.workload, cfg, g.n_blocks, cells, n_stage, int(cfg.get("n_order", 2)), world,
                                   g.state_bytes), parallelism=f"one grid sharded over {world} GPUs (Morton segments)"),
            "gpu_launches": int(g.launch_count() - n0), "kernels": g.kernel_counts(),
        }))
    g.close()
    dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-pipelines", type=int, default=3,
                    help="grids in flight in the end-to-end leg (host buffers, copies inside the timed region)")
    ap.add_argument("--sharded", action="store_true",
                    help="N > 1: one grid sharded over the GPUs (strong scaling) instead of N replicas; see run_sharded")
    ap.add_argument("--reference-blocks", type=int, nargs=3, default=None,
                    help="--impl reference: run the random_uniform recipe on this block grid instead of the named workload")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
