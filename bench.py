#!/usr/bin/env python
"""bench.py -- MLUPs/s and HBM-roofline fraction of the fused LBM stream-collide step on B200.

Workload (BASELINE.json configs[4], the paper's own benchmark box): D3Q19, BGK, fully
periodic cube L^3 (default 512^3, far beyond the 126 MB L2) with no boundary nodes, perturbed-equilibrium
initial state (workloads.perturbed_equilibrium, seeded).  A "step" is one lbm_step(1): one launch of the
fused stream_collide kernel over the whole box.  The metric is BASELINE.json's: D3Q19 MLUPs/s per DDF
storage format and achieved HBM GB/s vs the measured peak.  The JSON line's `value` is the headline
format (FP16S, the paper's fastest); every format is listed under `formats`.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--size L] [--formats FP32,FP16S,...]
    python bench.py --workload cavity|poiseuille|karman [--size L]   # the boxes with boundaries of configs[1..3]
    python bench.py --impl reference     # the CPU oracle, as it stands, on a bounded sample

--workload periodic (default) is the headline.  The others time the same lbm_step on the set-ups of BASELINE.json
configs[2] (lid-driven cavity L^3, default 256), configs[1] (Poiseuille channel L^3 with walls on the y faces and a
body force, default 256) and configs[3] (Karman street 4L x L x L/4 with a cylinder and an equilibrium rim, default
L = 256, i.e. 1024 x 256 x 64), inputs from workloads/: same JSON line, same roofline accounting (2 q s + 1 bytes per
cell), clocks and cpu_baseline.

N > 1 (torchrun): by default every rank runs an independent replica of the box ("weak" scaling, no data-path
collective: the paper's path is one GPU), timed as the max over ranks.  --decomposition slab
instead runs ONE box L x L x (L n_gpus) cut into z-slabs with the halo exchange of paper_2112_08926_b200/slab.py after
every step; with one GPU it runs the same plan as two slabs on that device.
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

import workloads as wl  # noqa: E402

METRIC = "D3Q19 MLUPs/s per DDF format (headline: FP32 arithmetic / FP16S storage); HBM GB/s vs peak"
HEADLINE = "FP16S"
SEED = 20211208
TAU = 0.6


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md, 6.65 TB/s)"


def recorded_traffic(fmt_name, size, workload="periodic"):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of the stream_collide kernel from the
    committed `ncu --set full` captures: profiles/dram_traffic.csv, columns velset,format,L,bytes_per_launch,profile
    [,workload].  The value is RECORDED, not measured in this run (ncu cannot run inside a timed region): the line
    carries the profile id beside it.  The LAST matching row wins (newest profile).  (None, None) if no capture
    exists for this format / size / workload."""
    path = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    if not os.path.exists(path):
        return None, None
    found = (None, None)
    for line in open(path):
        p = [c.strip() for c in line.split(",")]
        if len(p) >= 5 and p[0] == "D3Q19" and p[1] == fmt_name and p[2] == str(size) and (p[5] if len(p) > 5 else "periodic") == workload:
            try:
                found = (float(p[3]), p[4])
            except ValueError:
                pass
    return found


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def mark(self):
        return time.time()

    def stop(self):
        if self.proc:
            self.proc.terminate()

    def summary(self, windows):
        sm, smax, reasons, power = [], 0.0, set(), 0.0
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for t, line in self.rows:
            if not any(a <= t <= b for a, b in windows):
                continue
            p = [s.strip() for s in line.split(",")]
            try:
                sm.append(float(p[0])); smax = max(smax, float(p[1])); power = max(power, float(p[2]))
            except Exception:
                continue
            for n, v in zip(names, p[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax or None,
                "power_w_max": power or None, "samples": len(sm), "reasons": sorted(reasons)}


def dist_setup(n_gpus):
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        import torch
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    return world, rank, local


def max_over_ranks(ms, device="cuda"):
    """A step is over when the slowest rank is done: MAX over ranks of a per-rank time (any backend)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_mlups(world, cells_per_rank, steps, ms):
    """Replicas only: every rank updates its own box; the job's throughput is all ranks'
    cell updates over the slowest rank's time."""
    return world * cells_per_rank * steps / (ms * 1e-3) / 1e6


def rank_seed(rank):
    return SEED + rank


def make_workload(kind, L, Q, seed):
    """The synthetic input of one rank: a workloads.Workload and a one-line description."""
    nz = 1 if Q == 9 else L
    if kind == "periodic":
        w = wl.perturbed_equilibrium(L, L, nz, seed=seed, tau=TAU, velset=Q)
        what = (f"configs[4] bandwidth sweep: D{2 if Q == 9 else 3}Q{Q} periodic {'square' if Q == 9 else 'cube'} "
                f"{L}^{2 if Q == 9 else 3}, perturbed equilibrium (seed {SEED}), tau {TAU}")
    elif kind == "cavity":
        w = wl.lid_driven_cavity(L, velset=Q)
        what = f"configs[2] lid-driven cavity {L}^3, wall shell, lid u = 0.1, Re = 1000 (tau {w.tau:.4f}), fluid at rest"
    elif kind == "poiseuille":
        w = wl.poiseuille_channel(L, L, L, velset=Q)
        what = f"configs[1] Poiseuille channel {L}^3, walls on the y faces, Guo force, tau {w.tau}, fluid at rest"
    else:
        w = wl.karman_vortex_street(4 * L, L, max(L // 4, 1), radius=L / 16.0, velset=Q)
        what = (f"configs[3] Karman street {w.nx}x{w.ny}x{w.nz}, cylinder R = {L / 16.0:g}, equilibrium rim u = 0.05, "
                f"Re = 200 (tau {w.tau:.4f})")
    return w, what


def run_ours(args):
    import torch

    import paper_2112_08926_b200 as lbm

    world, rank, local = dist_setup(args.gpus)
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
    K, W, Q, kind = args.steps, args.warmup, args.velset, args.workload
    L = args.size if args.size else (512 if kind == "periodic" else 256)
    formats = args.formats.split(",")
    if kind != "periodic":
        formats = [f for f in formats if not f.startswith("FP64")] or formats
    peak, peak_src = measured_peak()

    # synthetic input.  Default: the seeded host arrays of workloads/, pinned (they are the end-to-end leg's input)
    # and copied to the device.  --device-init (periodic sweep sizes whose host arrays would be tens of GB): the same
    # recipe drawn on the device by torch's seeded generator; no end-to-end leg then.
    host_input = not (args.device_init and kind == "periodic")
    flags, force = None, None
    if host_input:
        w, what = make_workload(kind, L, Q, rank_seed(rank))
        nx, ny, nz, tau = w.nx, w.ny, w.nz, w.tau
        N = w.n_cells
        flags = w.flags if w.flags.any() else None
        force = w.force if any(float(v) != 0.0 for v in w.force) else None
        rho_h = torch.from_numpy(w.rho).pin_memory()
        u_h = torch.from_numpy(w.u).pin_memory()
        rho_d, u_d = rho_h.cuda(), u_h.cuda()
        rho_out = torch.empty(N, dtype=torch.float32).pin_memory()
        u_out = torch.empty((3, N), dtype=torch.float32).pin_memory()
    else:
        nx, ny, nz, tau = L, L, (1 if Q == 9 else L), TAU
        N = nx * ny * nz
        what = (f"configs[4] bandwidth sweep: D{2 if Q == 9 else 3}Q{Q} periodic {'square' if Q == 9 else 'cube'} "
                f"{L}^{2 if Q == 9 else 3}, perturbed equilibrium drawn cell by cell on the device (lbm_init_generated, seed {SEED}), tau {TAU}")
        rho_d = u_d = None                                   # drawn cell by cell on the device: lbm_init_generated

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    windows = []

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    results, launches_total = {}, 0
    for name in formats:
        sim = lbm.Simulation(nx, ny, nz, Q, name, tau, force=force, cells_per_thread=args.cells_per_thread,
                             collision=lbm.TRT if args.collision == "TRT" else lbm.BGK)
        if flags is not None:
            sim.set_flags(flags)
        if rho_d is None and not name.startswith("FP64"):
            sim.init_generated(rank_seed(rank))
        elif rho_d is None:                                   # FP64 arithmetic: fields drawn by torch (they fit beside the DDFs)
            gen = torch.Generator(device="cuda").manual_seed(rank_seed(rank))
            r_t = 1.0 + 1e-3 * torch.randn(N, device="cuda", generator=gen)
            u_t = (0.05 / 3 ** 0.5) * (2.0 * torch.rand((3, N), device="cuda", generator=gen) - 1.0)
            if Q == 9:
                u_t[2] = 0.0
            sim.init(r_t, u_t)
            del r_t, u_t
        else:
            sim.init(rho_d, u_d)
        sim.step(W)
        barrier()
        n0 = lbm.launch_count()
        t0 = sampler.mark()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        sim.step(K)                       # K launches of stream_collide on torch's current stream
        e1.record()
        barrier()
        windows.append((t0, sampler.mark()))
        ms = max_over_ranks(e0.elapsed_time(e1))
        launches = lbm.launch_count() - n0
        launches_total += launches
        if N <= (1 << 30):
            rho_chk, _ = sim.read_rho_u_device()
            assert bool(torch.isfinite(rho_chk).all()), name
            del rho_chk
        else:                                                 # the largest cubes: a few thousand probes instead of 16 B per cell
            prho, _ = sim.read_rho_u_at(np.linspace(0, N - 1, 4096).astype(np.int64))
            assert bool(np.isfinite(prho).all()), name
        # end to end through the public API with HOST buffers: init (H2D) + K steps + read-out (D2H)
        e2e_ms = None
        if host_input:
            barrier()
            t_e2e = time.perf_counter()
            sim.init(rho_h.numpy(), u_h.numpy())
            sim.step(K)
            sim.read_rho_u(out=(rho_out.numpy(), u_out.numpy()))
            torch.cuda.synchronize()
            e2e_ms = max_over_ranks((time.perf_counter() - t_e2e) * 1e3)
        bpc = lbm.bytes_per_cell(Q, name)
        mlups = whole_job_mlups(world, N, K, ms)
        gbs = N * bpc / (ms / K * 1e-3) / 1e9         # per GPU, per launch
        results[name] = {"mlups": round(mlups, 1), "ms_per_step": round(ms / K, 4), "bytes_per_cell": bpc,
                         "hbm_gbs": round(gbs, 1), "frac_of_peak": round(gbs / peak, 4),
                         "e2e_mlups": round(whole_job_mlups(world, N, K, e2e_ms), 1) if e2e_ms else None, "kernel": sim.kernel_name,
                         "launches": launches}
        sim.close()
        del sim
        torch.cuda.empty_cache()
    sampler.stop()
    if rank != 0:
        return
    head = HEADLINE if HEADLINE in results else formats[0]
    r = results[head]
    clocks = sampler.summary(windows)
    traffic, prof = recorded_traffic(head, L, kind) if Q == 19 else (None, None)
    traffic_src = (f"recorded: ncu --set full capture profiles/{prof} (dram__bytes_read.sum + dram__bytes_write.sum of one launch), "
                   "not measured in this run") if traffic else None
    line = {
        "metric": METRIC, "value": r["mlups"], "unit": "MLUPs/s", "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{what}; {args.collision}; headline storage format {head}",
                   "cells": N, "l2_policy": "inputs larger than L2 (two DDF buffers of "
                                            f"{N * Q * (4 if head == 'FP32' else 2) / 1e9:.2f} GB each, no flush needed)"
                                            if 2 * N * Q * (4 if head == 'FP32' else 2) > 2.5e8 else
                                            "box smaller than twice the 126 MB L2: partly L2-resident, not a roofline quote",
                   "parallelism": f"{world} independent replica(s)"},
        "formats": results,
        "speedup_16bit_vs_fp32": (round(results[head]["mlups"] / results["FP32"]["mlups"], 3)
                                  if "FP32" in results and head != "FP32" else None),
        "roofline": {"bound": "hbm", "kernel": r["kernel"], "achieved": r["hbm_gbs"], "peak": peak, "unit": "GB/s",
                     "frac": r["frac_of_peak"], "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": N * r["bytes_per_cell"]},
        "e2e": {"value": r["e2e_mlups"], "unit": "MLUPs/s", "h2d_bytes_per_step": 16 * N / K,
                "d2h_bytes_per_step": 16 * N / K,
                "what": f"lbm_init(host rho,u) + lbm_step({K}) + lbm_read_rho_u(host), wall clock, pinned host buffers"},
        "gpu_launches": launches_total, "clocks": clocks,
    }
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(head, budget_s=args.cpu_seconds, collision=args.collision, kind=kind)
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def run_slab(args):
    """--decomposition slab: ONE periodic box L x L x (L * n_gpus), cut
    into z slabs, one per rank, every step followed by the exchange of the face-crossing directions in the stored
    format (paper_2112_08926_b200/slab.py; NCCL point-to-point).  Weak scaling: L^3 owned cells per GPU.  With one
    GPU the same plan runs as two half-height slabs of an L^3 box on that device (device copies instead of NCCL): the
    cost of the ghost planes and of the copies, not a multi-GPU number."""
    import torch

    import paper_2112_08926_b200 as lbm
    from paper_2112_08926_b200 import slab as sl

    world, rank, local = dist_setup(args.gpus)
    torch.cuda.set_device(local)
    K, W, Q = args.steps, args.warmup, args.velset
    if Q == 9 or args.workload != "periodic":
        raise SystemExit("--decomposition slab: the periodic D3Q19 / D3Q27 box only")
    L = args.size if args.size else 512
    formats = [f for f in args.formats.split(",") if not f.startswith("FP64")]
    peak, peak_src = measured_peak()
    coll = lbm.TRT if args.collision == "TRT" else lbm.BGK
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    windows, results, launches_total = [], {}, 0
    dist = None
    if world > 1:
        import torch.distributed as dist

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for name in formats:
        if world > 1:
            box = sl.DistSlab(L, L, L * world, Q, name, TAU, collision=coll)
            slabs = [box.slab]
        else:
            box = sl.LocalSlabs(L, L, L, 2, Q, name, TAU, collision=coll)
            slabs = box.slabs
        for k, s in enumerate(slabs):                         # owned planes drawn on the device, ghosts by one exchange
            s.sim.init_generated(rank_seed(rank) + 1000 * k)
        if world > 1:
            sl.exchange_distributed(box.slab.current(), box.slab.plan, rank, world, dist)
        else:
            box.exchange()
        box.step(W)
        barrier()
        n0 = lbm.launch_count()
        t0 = sampler.mark()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        box.step(K)                                           # K x (stream_collide on every local slab + exchange)
        e1.record()
        barrier()
        windows.append((t0, sampler.mark()))
        ms = max_over_ranks(e0.elapsed_time(e1))
        launches = lbm.launch_count() - n0
        launches_total += launches
        prho, _ = slabs[0].sim.read_rho_u_at(np.linspace(0, slabs[0].sim.N - 1, 4096).astype(np.int64))
        assert bool(np.isfinite(prho).all()), name
        owned = L ** 3                                        # per GPU
        computed = sum(s.sim.N for s in slabs)          # ghost planes included
        bpc = lbm.bytes_per_cell(Q, name)
        up, down = sl.crossing_directions(Q)
        halo = (len(up) + len(down)) * L * L * slabs[0].es * len(slabs)
        gbs = computed * bpc / (ms / K * 1e-3) / 1e9
        results[name] = {"mlups": round(world * owned * K / (ms * 1e-3) / 1e6, 1), "ms_per_step": round(ms / K, 4),
                         "bytes_per_cell": bpc, "hbm_gbs": round(gbs, 1), "frac_of_peak": round(gbs / peak, 4),
                         "halo_bytes_sent_per_gpu_per_step": halo, "kernel": slabs[0].sim.kernel_name, "launches": launches}
        box.close()
        del box, slabs
        torch.cuda.empty_cache()
    sampler.stop()
    if rank != 0:
        return
    head = HEADLINE if HEADLINE in results else formats[0]
    r = results[head]
    line = {
        "metric": METRIC, "value": r["mlups"], "unit": "MLUPs/s", "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": (f"ONE periodic D3Q{Q} box {L}x{L}x{L * world} in {world} z-slabs of {L} planes + 2 ghost planes, "
                                f"one per GPU, halo exchange (NCCL point-to-point) every step" if world > 1 else
                                f"periodic D3Q{Q} box {L}^3 as two z-slabs of {L // 2} planes + 2 ghost planes on ONE GPU, "
                                "halo exchange by device copies every step (the decomposition's overhead, not a multi-GPU number)")
                               + f"; perturbed equilibrium drawn on the device, tau {TAU}; {args.collision}; headline storage format {head}",
                   "cells": L ** 3 * world, "l2_policy": "inputs larger than L2" if L >= 256 else "partly L2-resident",
                   "parallelism": f"z-slab decomposition over {world} GPU(s)"},
        "formats": results,
        "roofline": {"bound": "hbm", "kernel": r["kernel"], "achieved": r["hbm_gbs"], "peak": peak, "unit": "GB/s",
                     "frac": r["frac_of_peak"], "traffic": None, "peak_source": peak_src,
                     "what": "per GPU; counts the ghost planes' cells (computed, then overwritten) and the whole step incl. the exchange"},
        "e2e": {"value": None, "unit": "MLUPs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                "what": "no end-to-end leg in this mode (input drawn on the device); see the default run"},
        "gpu_launches": launches_total, "clocks": sampler.summary(windows),
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_run(fmt_name, L, steps, warmup, collision="BGK", kind="periodic", threads=0):
    """Time the CPU oracle, as it stands, on a sample of the workload with edge L (see make_workload).
    Returns (mlups, cores, seconds, cells)."""
    import oracle
    cores = oracle.set_threads(threads or os.cpu_count() or 1)
    w, _ = make_workload(kind, L, 19, SEED)
    sim = oracle.from_workload(w, wl.FORMATS[fmt_name])
    if collision == "TRT":
        sim.set_collision(oracle.TRT)
    sim.step(warmup)
    t0 = time.perf_counter()
    sim.step(steps)
    dt = time.perf_counter() - t0
    return w.n_cells * steps / dt / 1e6, cores, dt, w.n_cells


def cpu_baseline(fmt_name, budget_s=15.0, collision="BGK", kind="periodic"):
    """The oracle on a BOUNDED sample of the same workload (128^3 periodic / cavity / channel, 256 x 64 x 16 Karman
    box: beyond the LLC), on all host cores and on one, step counts sized from a 1-step probe so that the two timed
    parts take about `budget_s` seconds together."""
    L = 64 if kind == "karman" else 128
    probe, cores, dt, cells = oracle_run(fmt_name, L, 1, 1, collision, kind)
    steps = max(2, min(200, int(0.6 * budget_s / max(dt, 1e-3))))
    mlups, cores, dt, cells = oracle_run(fmt_name, L, steps, 0, collision, kind)
    steps1 = max(1, min(50, int(0.4 * budget_s / max(dt / steps * cores, 1e-3))))
    mlups1, _, dt1, _ = oracle_run(fmt_name, L, steps1, 0, collision, kind, threads=1)
    return {"value": round(mlups, 2), "unit": "MLUPs/s", "cores": cores, "kind": "oracle",
            "one_core": round(mlups1, 2), "cpu_model": cpu_model(),
            "sample": f"D3Q19 {collision} {fmt_name} storage, {kind} box of {cells} cells of the same recipe, "
                      f"{steps} steps in {dt:.1f} s on {cores} threads, {steps1} steps in {dt1:.1f} s on one"}


def run_reference(args):
    """--impl reference: for this tier the reference arm is the CPU oracle (there is no reference code)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    K, W = args.steps, args.warmup
    L = 128
    probe, cores, dt1, _ = oracle_run(HEADLINE, L, 1, 0, args.collision)
    K_eff = max(1, min(K, int(120.0 / max(dt1, 1e-3))))       # keep the whole run within a few minutes
    mlups, cores, dt, _ = oracle_run(HEADLINE, L, K_eff, min(W, 2), args.collision)
    sample = (f"D3Q19 {args.collision} {HEADLINE} storage, {L}^3 periodic sample box of the {args.size or 512}^3 workload, "
              f"{K_eff} timed steps, {dt:.1f} s, {cores} OpenMP threads")
    line = {"impl": "reference", "metric": METRIC, "value": round(mlups, 2), "unit": "MLUPs/s",
            "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": K_eff, "warmup": min(W, 2),
            "ms_per_step": round(dt / K_eff * 1e3, 3), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"configs[4] bandwidth sweep: D3Q19 {args.collision} periodic cube, perturbed equilibrium "
                                   f"(seed {SEED}), tau {TAU}, storage format {HEADLINE}; CPU oracle on a bounded sample",
                       "sample": sample},
            "cpu_baseline": {"value": round(mlups, 2), "unit": "MLUPs/s", "cores": cores, "kind": "oracle", "sample": sample,
                             "cpu_model": cpu_model()},
            "e2e": {"value": round(mlups, 2), "unit": "MLUPs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--size", type=int, default=0, help="cube edge L (default 512; 256 for the boxes with boundaries)")
    ap.add_argument("--workload", default="periodic", choices=["periodic", "cavity", "poiseuille", "karman"],
                    help="periodic = the headline (configs[4]); the others: the boxes with boundaries of configs[1..3]")
    ap.add_argument("--formats", default="FP32,FP16S,FP16C,P16_0S,P16_1S,P16_2C,FP64,FP64_FP32")
    ap.add_argument("--velset", type=int, default=19, choices=[9, 19, 27], help="sweep only; the headline is D3Q19")
    ap.add_argument("--device-init", action="store_true", help="draw the input on the device (big sweep sizes)")
    ap.add_argument("--cells-per-thread", type=int, default=0, help="0 = library default")
    ap.add_argument("--collision", default="BGK", choices=["BGK", "TRT"], help="sweep only; the headline is BGK (TRT: DESIGN.md R13)")
    ap.add_argument("--decomposition", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: independent boxes (default) or ONE box cut into z-slabs with a halo exchange per step")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    elif args.decomposition == "slab":
        run_slab(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
