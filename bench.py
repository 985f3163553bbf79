#!/usr/bin/env python
"""bench.py — particle-steps/s of the PIC particle step (gather + Boris + Esirkepov + resort).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

One "step" = one pass of the whole hot path (pic_step(1)) over all particles
of the workload.  Default workload = BASELINE.json configs[1] (128^3 TSC thermal plasma, 16 ppc,
33.5 M particles), the configuration the metric is quoted on.  Prints ONE JSON line (rank 0).

N > 1: the path is single-GPU by contract (north_star); ranks run independent replicas of the
workload ("replicas only"), no data-path collective; value = particles of all
ranks * K / max-over-ranks device time.
--impl reference: the fp64 single-threaded oracle timed on the host cores on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "particle-steps/s (gather+Boris+Esirkepov+resort)"
UNIT = "particle-steps/s"
PARTICLE_BYTES = 64.0      # float4 pos + float4 mom, read + write (SURVEY.md §8(d), 64 B basis)
GRID_BYTES_PER_CELL = 36.0  # E+B read once (24 B) + J written once (12 B) per cell per step
LEAVER_BYTES = 36.0 * 0.015
# Yee update: the METHOD moves 60 B per cell (E, B, J read once = 36 B, E, B written once = 24 B).  The
# fields are kept in padded arrays only (the form the step kernel's TMA reads), so the kernel writes them once; the
# halo cells it writes on top are not counted.
FIELD_UPDATE_BYTES_PER_CELL = 60.0


def algorithmic_bytes_per_particle_step(wl, n_particles: int) -> float:
    """B_alg = 64 + 36 * cells/particles + 0.54 (1.5 % leavers x 36 B)."""
    return PARTICLE_BYTES + GRID_BYTES_PER_CELL * wl.n_cells / n_particles + LEAVER_BYTES


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            f = [v.strip() for v in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample_rate(wl, n_sample: int, n_steps: int = 1):
    """Time the oracle (as it stands, single-threaded fp64) on the first n_sample particles of the
    workload with the full-size fields.  Returns (particle-steps/s, seconds, n_sample)."""
    import torch
    import oracle
    from paper_2110_08650_b200 import workloads as W
    fields = W.make_fields(wl)
    per_slab = wl.grid[0] * wl.grid[1] * wl.ppc
    chunk = next(iter(W.particle_chunks(wl, max_chunk=max(n_sample, per_slab))))
    sel = torch.randperm(chunk.n, generator=torch.Generator().manual_seed(7))[:n_sample]
    orc = oracle.Oracle(wl.grid, wl.cell, wl.dt, wl.supercell, wl.shape_order)
    orc.load_particles(*(getattr(chunk, k)[sel].numpy() for k in ("x", "y", "z", "ux", "uy", "uz", "w")),
                       species=chunk.species[sel].numpy())
    orc.set_fields(fields.numpy())
    t0 = time.perf_counter()
    rc = orc.step(n_steps)
    dt = time.perf_counter() - t0
    assert rc == 0
    return orc.n * n_steps / dt, dt, orc.n


def oracle_field_update_rate(grid=(128, 128, 64), reps=3):
    """The fp64 numpy oracle of the Yee update (oracle/yee_oracle.py), as it stands, on a bounded grid."""
    import numpy as np
    from oracle import yee_oracle as Y
    rng = np.random.default_rng(0)
    shp = (grid[2], grid[1], grid[0])
    F = [rng.normal(size=shp) for _ in range(6)]
    J = [rng.normal(size=shp) for _ in range(3)]
    t0 = time.perf_counter()
    for _ in range(reps):
        F = Y.yee_update(F, J, 0.5)
    dt = time.perf_counter() - t0
    return {"value": reps * grid[0] * grid[1] * grid[2] / dt, "unit": "cell-updates/s", "cores": 1, "kind": "oracle",
            "sample": f"{reps} updates of a {grid[0]}x{grid[1]}x{grid[2]} grid ({dt:.1f} s), numpy fp64"}


def reduce_max_over_ranks(values, device, world: int):
    """MAX over ranks of a list of floats (device time of the slowest rank decides); identity at N=1."""
    import torch
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def whole_job_value(world: int, particles_per_rank: int, steps: int, seconds: float) -> float:
    """Replicas only: every rank steps its own copy of the workload; units of all ranks / slowest time."""
    return world * particles_per_rank * steps / seconds


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step = one oracle step
    over a bounded sample of the workload (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2110_08650_b200 import workloads as W
    wl = W.CONFIGS[args.workload]
    n_sample = {1: 400_000, 2: 200_000, 3: 130_000}[wl.shape_order]
    for _ in range(args.warmup):
        oracle_sample_rate(wl, n_sample // 8)
    t_tot, n_tot = 0.0, 0
    for _ in range(args.steps):
        _, dt, n = oracle_sample_rate(wl, n_sample)
        t_tot += dt
        n_tot += n
    value = n_tot / t_tot
    sample = f"{n_sample} particles of {wl.name} per step (random subset of the first z-slabs), full-size fields"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_tot / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "grid": list(wl.grid), "shape_order": wl.shape_order, "ppc": wl.ppc,
                   "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def measure_e2e(args, wl, n, K, fields, fresh, barrier, dev, world):
    """The same metric through the C ABI with HOST buffers: every step copies the inputs from pinned
    host memory, loads, steps once and reads J and the particles back to the host."""
    import torch
    from paper_2110_08650_b200 import workloads as W
    e2e_steps = min(K, args.e2e_steps)
    names = ("x", "y", "z", "ux", "uy", "uz", "w", "species")
    host = {k: [] for k in names}
    for chunk in W.particle_chunks(wl, device=dev, max_chunk=1 << 23):
        for k in names:
            host[k].append(getattr(chunk, k).cpu())
    host = {k: torch.cat(v).pin_memory() for k, v in host.items()}
    host_fields = fields.cpu().pin_memory()
    dev_in = {k: torch.empty_like(v, device=dev) for k, v in host.items()}
    dev_fields = torch.empty_like(fields)
    out_keys = ("x", "y", "z", "ux", "uy", "uz")
    host_out = {k: torch.empty(n, dtype=host[k].dtype).pin_memory() for k in out_keys}
    host_J = torch.empty((3,) + tuple(fields.shape[1:]), dtype=torch.float32).pin_memory()
    h2d = sum(v.numel() * v.element_size() for v in host.values()) + host_fields.numel() * 4
    d2h = sum(v.numel() * v.element_size() for v in host_out.values()) + host_J.numel() * 4

    def e2e_step():
        p = fresh()
        for k in names:
            dev_in[k].copy_(host[k], non_blocking=True)
        dev_fields.copy_(host_fields, non_blocking=True)
        p.load_particles(*(dev_in[k] for k in names))
        p.set_fields(dev_fields)
        p.step(1)
        host_J.copy_(p.get_current(), non_blocking=True)
        P = p.get_particles(n)
        for k in out_keys:
            host_out[k].copy_(P[k], non_blocking=True)
        torch.cuda.synchronize()
        p.destroy()

    e2e_step()                      # warm-up (page-locking, allocator)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_value = whole_job_value(world, n, e2e_steps, reduce_max_over_ranks([e2e_s], dev, world)[0])
    out = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps}

    # The same per-step traffic with two contexts on two streams (each its own workspace, device and pinned buffers):
    # the jobs are independent — every e2e step above is a fresh load already — so step k+1's host-to-device copies
    # run beside step k's device-to-host copies (PCIe is full duplex).  Reported beside `value`, not instead of it.
    try:
        from paper_2110_08650_b200.binding import workspace_bytes
        streams = [torch.cuda.Stream(dev), torch.cuda.Stream(dev)]
        wss = [None, torch.empty(workspace_bytes(wl.grid, wl.supercell, wl.shape_order, n) + 256, dtype=torch.uint8, device=dev)]
        din = [dev_in, {k: torch.empty_like(v) for k, v in dev_in.items()}]
        dfl = [dev_fields, torch.empty_like(dev_fields)]
        hout = [host_out, {k: torch.empty_like(v).pin_memory() for k, v in host_out.items()}]
        hJ = [host_J, torch.empty_like(host_J).pin_memory()]
        live = [None, None]

        def issue(i):
            b = i & 1
            if live[b] is not None:         # the buffers of set b are free once its last job is through
                streams[b].synchronize()
                live[b].destroy()
            with torch.cuda.stream(streams[b]):
                p = fresh(workspace=wss[b], stream=streams[b])
                for k in names:
                    din[b][k].copy_(host[k], non_blocking=True)
                dfl[b].copy_(host_fields, non_blocking=True)
                p.load_particles(*(din[b][k] for k in names))
                p.set_fields(dfl[b])
                p.step(1)
                hJ[b].copy_(p.get_current(), non_blocking=True)
                P = p.get_particles(n)
                for k in out_keys:
                    hout[b][k].copy_(P[k], non_blocking=True)
            live[b] = p

        torch.cuda.synchronize()
        issue(0); issue(1)                  # warm-up of both sets
        torch.cuda.synchronize()
        barrier()
        M = 2 * e2e_steps
        t0 = time.perf_counter()
        for i in range(M):
            issue(i)
        torch.cuda.synchronize()
        barrier()
        pipe_s = time.perf_counter() - t0
        for p in live:
            if p is not None:
                p.destroy()
        out["pipelined_value"] = whole_job_value(world, n, M, reduce_max_over_ranks([pipe_s], dev, world)[0])
        out["pipelined"] = ("%d independent steps on two contexts and two streams: the host-to-device copies of one overlap "
                            "the device-to-host copies of the other; same bytes per step" % M)
    except torch.cuda.OutOfMemoryError:
        out["pipelined_value"] = None
    return out


def measure_other(args, wl, dev, peak):
    """One of the other BASELINE.json workloads, device-resident: load, 3 warm-up steps, a few timed steps."""
    import torch
    from paper_2110_08650_b200 import workloads as W
    from paper_2110_08650_b200.binding import Pic, workspace_bytes
    n = W.n_particles(wl)
    t_load = time.perf_counter()
    ws = torch.empty(workspace_bytes(wl.grid, wl.supercell, wl.shape_order, n) + 256, dtype=torch.uint8, device=dev)
    pic = Pic(wl.grid, wl.cell, wl.dt, wl.supercell, wl.shape_order, max_particles=n, device=dev, workspace=ws)
    pic.set_option("cell_kernel", args.cell_kernel)
    pic.set_option("direct_below", args.direct_below)
    pic.set_option("sparse_nosort", args.sparse_nosort)
    for k in ("tma", "deposit", "two_phase"):
        pic.set_option(k, getattr(args, k))
    for kv in args.opt:
        k, v = kv.split("=")
        pic.set_option(k, int(v))
    for chunk in W.particle_chunks(wl, device=dev, max_chunk=1 << 23):
        pic.load_particles(chunk.x, chunk.y, chunk.z, chunk.ux, chunk.uy, chunk.uz, chunk.w, chunk.species)
        pic.sync()
    del chunk
    fields = W.make_fields(wl, device=dev)
    pic.set_fields(fields)
    t_load = time.perf_counter() - t_load
    steps = args.other_steps
    pic.step(3)
    pic.sync()
    pic.set_option("timing", 1)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ev0.record(pic.stream)
    pic.step(steps)
    ev1.record(pic.stream)
    torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1) / steps
    kernel_ms, n_kernel = pic.get_timing()
    kernel_ms /= max(n_kernel, 1)
    st = pic.get_stats()
    # the Yee update on this grid (not part of the metric)
    for _ in range(2):
        pic.update_fields()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record(pic.stream)
    for _ in range(5):
        pic.update_fields()
    f1.record(pic.stream)
    torch.cuda.synchronize()
    fu_ms = f0.elapsed_time(f1) / 5
    pic.destroy()
    del pic, ws, fields
    b_alg = algorithmic_bytes_per_particle_step(wl, n)
    return {"grid": list(wl.grid), "shape_order": wl.shape_order, "particles": n, "steps": steps, "warmup": 3,
            "ms_per_step": ms, "value": n / (ms * 1e-3), "unit": UNIT, "step_kernels_ms": kernel_ms,
            "bytes_per_particle_step": b_alg, "frac": b_alg * n / (kernel_ms * 1e-3) / 1e9 / peak,
            "frac_whole_step": b_alg * n / (ms * 1e-3) / 1e9 / peak,
            "leavers_per_step": st["leavers_last"], "max_supercell_population": st["max_count"], "error_word": st["error"],
            "field_update_ms": fu_ms,
            "field_update_frac_60B": FIELD_UPDATE_BYTES_PER_CELL * wl.n_cells / (fu_ms * 1e-3) / 1e9 / peak,
            "exact_shortcuts": "sparse supercells only (option rest_skip, default on; results bit-identical, tested): warps of "
                               "particles at rest in a supercell whose E/B tile is all zero are not stepped",
            "load_and_setup_s": t_load}


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2110_08650_b200 import workloads as W
    from paper_2110_08650_b200.binding import Pic, workspace_bytes

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; the product has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    wl = W.CONFIGS[args.workload]
    if args.grid:      # reduced-grid copy of the workload (experiments only; the default is the full config)
        wl = wl.scaled(tuple(int(v) for v in args.grid.split(",")))
    n = W.n_particles(wl)
    K, Wm = args.steps, max(args.warmup, 3)
    ws = torch.empty(workspace_bytes(wl.grid, wl.supercell, wl.shape_order, n) + 256, dtype=torch.uint8, device=dev)

    def fresh(host_inputs=None, workspace=None, stream=None):
        pic = Pic(wl.grid, wl.cell, wl.dt, wl.supercell, wl.shape_order, max_particles=n, device=dev,
                  workspace=ws if workspace is None else workspace, stream=stream)
        pic.set_option("tma", args.tma)
        pic.set_option("deposit", args.deposit)
        pic.set_option("segment", args.segment)
        pic.set_option("two_phase", args.two_phase)
        pic.set_option("cell_kernel", args.cell_kernel)
        pic.set_option("crowd_first", args.crowd_first)
        pic.set_option("sparse_nosort", args.sparse_nosort)
        pic.set_option("direct_below", args.direct_below)
        pic.set_option("field_update", args.self_consistent)
        for kv in args.opt:
            k, v = kv.split("=")
            pic.set_option(k, int(v))
        return pic

    # ---------------------------------------------------------------- device-resident throughput
    fields = W.make_fields(wl, device=dev)

    def load(p, w=wl):
        for chunk in W.particle_chunks(w, device=dev, max_chunk=1 << 23):
            p.load_particles(chunk.x, chunk.y, chunk.z, chunk.ux, chunk.uy, chunk.uz, chunk.w, chunk.species)
            p.sync()

    def timed_run(p, n_warm, n_steps):
        """n_warm untimed steps, then exactly n_steps steps between CUDA events on the library's stream."""
        p.step(n_warm)
        p.sync()
        p.set_option("timing", 1)
        l0 = p.launch_count()
        barrier()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(p.stream)
        p.step(n_steps)
        ev1.record(p.stream)
        barrier()
        ms = ev0.elapsed_time(ev1)
        kernel_ms, n_kernel = p.get_timing()
        p.set_option("timing", 0)
        return ms, kernel_ms / max(n_kernel, 1), p.launch_count() - l0

    # headline: median of `--repeats` runs, each from a freshly loaded state
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    runs = []
    pic = None
    for r in range(max(args.repeats, 1)):
        if pic is not None:
            pic.destroy()
        pic = fresh()
        load(pic)
        pic.set_fields(fields)
        ms_r, k_r, launches = timed_run(pic, Wm, K)
        ms_r, k_r = reduce_max_over_ranks([ms_r, k_r], dev, world)
        runs.append((ms_r, k_r))
    clocks = sampler.stop() if rank == 0 else None
    stats = pic.get_stats()
    runs_sorted = sorted(runs)
    ms_max, kernel_ms_avg = runs_sorted[len(runs_sorted) // 2]
    value = whole_job_value(world, n, K, ms_max * 1e-3)

    # the same workload late in its run (the static fields bunch the plasma: BASELINE.md): steps 80-100 of 100
    late = None
    if args.late_run and rank == 0 and world == 1 and wl.steps >= 40:
        n_late = min(20, wl.steps // 5)
        ms_l, k_l, _ = timed_run(pic, max(wl.steps - n_late - Wm - K, 0), n_late)
        st_l = pic.get_stats()
        late = {"steps": f"{wl.steps - n_late}-{wl.steps} of the workload's {wl.steps}", "ms_per_step": ms_l / n_late,
                "value": n * n_late / (ms_l * 1e-3), "kernel_ms": k_l, "max_supercell_population": st_l["max_count"],
                "leavers_per_step": st_l["leavers_last"]}

    # ---------------------------------------------------------------- the Yee field update alone
    fu = None
    if args.field_update_reps > 0 and rank == 0:
        R = args.field_update_reps
        for _ in range(3):
            pic.update_fields()
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        f0.record(pic.stream)
        for _ in range(R):
            pic.update_fields()
        f1.record(pic.stream)
        torch.cuda.synchronize()
        fu_ms = f0.elapsed_time(f1) / R
        peak_f, _ = measured_peaks()
        fu_bytes = FIELD_UPDATE_BYTES_PER_CELL * wl.n_cells
        fu = {"kernel": "pic_yee_kernel (B half, E, B half fused; padded array in, padded array out)",
              "ms_per_update": fu_ms, "cells": wl.n_cells, "bytes_per_cell": FIELD_UPDATE_BYTES_PER_CELL,
              "bound": "hbm", "achieved": fu_bytes / (fu_ms * 1e-3) / 1e9, "peak": peak_f, "unit": "GB/s",
              "frac": fu_bytes / (fu_ms * 1e-3) / 1e9 / peak_f,
              "l2": ("working set %.0f MB %s the 126 MB L2" % (fu_bytes / 1e6, "exceeds" if fu_bytes > 126e6 else "fits")),
              "updates_per_s_cells": wl.n_cells / (fu_ms * 1e-3),
              "share_of_self_consistent_step": fu_ms / (ms_max / K if args.self_consistent else fu_ms + ms_max / K)}
        if not args.no_cpu_baseline:
            fu["cpu_baseline"] = oracle_field_update_rate()
    pic.destroy()

    e2e = measure_e2e(args, wl, n, K, fields, fresh, barrier, dev, world) if args.e2e_steps > 0 else None

    # ---------------------------------------------------------------- the other workloads of BASELINE.json:configs
    others = None
    if args.all_configs and rank == 0 and world == 1 and not args.grid:
        del ws, fields
        torch.cuda.empty_cache()
        others = {}
        peak_o, _ = measured_peaks()
        for name in ("tiny_thermal", "lwfa", "khi", "khi_hotspot", "pqs_large"):
            if name == wl.name:
                continue
            try:
                others[name] = measure_other(args, W.CONFIGS[name], dev, peak_o)
            except Exception as exc:      # a workload that does not fit this box is reported, not fatal
                others[name] = {"error": f"{type(exc).__name__}: {exc}"[:200]}
            torch.cuda.empty_cache()

    if rank == 0:
        peak, peak_src = measured_peaks()
        b_alg = algorithmic_bytes_per_particle_step(wl, n)
        achieved = b_alg * n / (kernel_ms_avg * 1e-3) / 1e9
        traffic, ncu_extra = None, {}
        tpath = os.path.join(ROOT, "profiles", "step_kernel_traffic.json")
        if os.path.exists(tpath):
            with open(tpath) as f:
                tj = json.load(f)
            if tj.get("workload") == wl.name:
                traffic = tj.get("dram_bytes_per_launch")
                ncu_extra = {k: tj[k] for k in ("warp_instructions_per_launch", "shared_pipe_busy_pct",
                                                "issue_slots_busy_pct", "warps_per_sm", "registers_per_thread") if k in tj}
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            n_s = {1: 4_000_000, 2: 2_400_000, 3: 1_600_000}[wl.shape_order]
            v, dt, ns = oracle_sample_rate(wl, n_s)
            cpu = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
                   "sample": f"{ns} particles of {wl.name} x 1 step ({dt:.1f} s), full-size fields, single thread of "
                             f"{len(os.sched_getaffinity(0))} available"}
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": wl.name, "grid": list(wl.grid), "shape_order": wl.shape_order, "ppc": wl.ppc,
                       "particles_per_gpu": n, "supercell": list(wl.supercell), "dt": wl.dt,
                       "parallelism": "replicas only" if world > 1 else "single GPU",
                       "l2": f"inputs larger than L2: {n * 72 / 1e6:.0f} MB of particle state per step vs 126 MB",
                       "tma": args.tma, "deposit": "fixed-point int32 pair" if args.deposit else "float atomics",
                       "leavers_per_step": stats["leavers_last"], "self_consistent": args.self_consistent},
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": traffic, "peak_source": peak_src,
                         "kernel": "pic_step_kernel (resort of the previous step fused into its prologue) "
                                   "+ pic_sort_kernel for sparse supercells",
                         "kernel_ms": kernel_ms_avg, "bytes_per_particle_step": b_alg,
                         "frac_of_8000_GBps": achieved / 8000.0,
                         "kernel_share_of_step": kernel_ms_avg / (ms_max / K),
                         "binding_resource": "latency at 8 warps/SM (238 registers/thread, 114 KB shared memory per CTA): "
                                             "0.46 instructions per cycle per scheduler, FMA pipe 35 %, shared-memory pipe "
                                             "61 % (ncu: profiles/r02_phase_budget.md); HBM is the bound the metric names, not "
                                             "the one the kernel hits: its FP32 work alone is 0.94 ms per step (0.36 of the "
                                             "roofline), its issue floor 1.27 ms",
                         "ncu": ncu_extra},
            "repeats": {"n": len(runs), "ms_per_step": [r[0] / K for r in runs], "headline": "median",
                        "each_from": "a freshly loaded state, warm-up steps first"},
            "late_run": late,
            "all_configs": others,
            "cpu_baseline": cpu,
            "e2e": e2e,
            "field_update": fu,
            "gpu_launches": launches, "clocks": clocks,
        }))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--workload", default="thermal_128")
    ap.add_argument("--grid", default="", help="nx,ny,nz: run a reduced-grid copy of the workload")
    ap.add_argument("--tma", type=int, default=1)
    ap.add_argument("--deposit", type=int, default=1, help="1 fixed-point integer atomics, 0 float CAS atomics")
    ap.add_argument("--segment", type=int, default=3, help="work-item length in quarters of the mean cell population")
    ap.add_argument("--two-phase", type=int, default=1, help="1: per-cell stencil in registers (two-phase items), 0: gather per particle from the shared tile")
    ap.add_argument("--cell-kernel", type=int, default=0, help="1: dense supercells go to pic_cell_kernel (third generation), 0: round-1 kernels")
    ap.add_argument("--direct-below", type=int, default=768, help="supercells with fewer particles take the per-particle (sparse) kernel")
    ap.add_argument("--opt", action="append", default=[], help="key=value: any further pic_set_option (experiments)")
    ap.add_argument("--sparse-nosort", type=int, default=1, help="1: all-sparse steps skip the re-sort (one sort in 16 steps; N >= 2: one in N)")
    ap.add_argument("--crowd-first", type=int, default=0, help="1: the step kernels start crowded supercells first")
    ap.add_argument("--repeats", type=int, default=5, help="the headline is the median of this many runs, each from a fresh load")
    ap.add_argument("--late-run", type=int, default=1, help="1: also time the last 20 steps of the workload's own step count")
    ap.add_argument("--all-configs", type=int, default=1, help="1: also measure the other BASELINE.json workloads (key all_configs)")
    ap.add_argument("--other-steps", type=int, default=5, help="timed steps per workload of --all-configs")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--field-update-reps", type=int, default=20,
                    help="also time this many launches of the Yee field update alone (0 = skip); not part of the metric")
    ap.add_argument("--self-consistent", type=int, default=0,
                    help="1: every timed step ends with the Yee field update (option field_update); the metric's "
                         "configuration is 0, static fields")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
