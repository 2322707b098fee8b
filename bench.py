#!/usr/bin/env python
"""bench.py -- throughput of the Kratos hydro hot path on B200 (cell-updates/s and % of HBM roofline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload C5|C4|C3|C5-256] [--precision mixed|fp64|single] [--integrator heun|vanleer]
                    [--slabs R | --decomposition slab]

A "step" is one full Heun step (both stages: ghost rules, primitive recovery, PLM, HLLC, fp64 update,
fused CFL reduction) of one synthetic block.  Default workload: BASELINE.json config 5 (512^3 periodic,
gamma 1.001, Mach-1 random-phase velocity field, mixed precision) -- the configuration the metric is
quoted on.  Prints ONE JSON line (rank 0).

Multi-GPU: the path does not shard in this build (BASELINE.json: one GPU, no collectives), so
--gpus N runs N independent replicas ("replicas only"); torch.distributed is
used for the barrier and the max-over-ranks time only.

--slabs R cuts the block into R z slabs that exchange their ghost planes through communication boundaries
(paper_2501_02317_b200/slab.py), all in this process on this GPU, advanced in lock step:
what the decomposition costs on one device (the R stage launches of a step run one after the other).  Under torchrun,
--decomposition slab gives every rank one slab of the ONE block instead of a replica ("scaling": "strong"; NCCL
all-reduces for the time step and the ordering, CUDA IPC for the neighbours' ghost arrays).

--impl reference times the oracle (oracle/kratos_oracle.c, as it stands) on the host cores on a
bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "cell-updates/sec per B200 (3D hydro step) and % of HBM roofline"
UNIT = "cell-updates/s"
BYTES_PER_CELL = {"stage1": 80.0, "stage2": 120.0}  # algorithmic HBM bytes per cell
# van Leer, mixed precision: predictor 40 B read + 20 B written, corrector 20 + 40 read + 40 written
BYTES_PER_CELL_VL = {"stage1": 60.0, "stage2": 100.0}
# all-fp32 "Single" mode: the state is stored as floats, half the traffic of the Heun stages
BYTES_PER_CELL_SINGLE = {"stage1": 40.0, "stage2": 60.0}


def workload(name: str):
    from paper_2501_02317_b200 import inputs
    if name == "C5":
        return inputs.turbulence_3d(512, seed=5, nsteps=20), "C5 3D decaying turbulence 512^3 periodic gamma=1.001"
    if name == "C5-256":
        return inputs.turbulence_3d(256, seed=5, nsteps=20), "C5 recipe at 256^3"
    if name == "C5-128":
        return inputs.turbulence_3d(128, seed=5, nsteps=20), "C5 recipe at 128^3"
    if name == "C4":
        return inputs.point_blast_3d(256, nsteps=50), "C4 3D point blast 256^3 outflow gamma=5/3"
    if name == "C1":
        return inputs.riemann_1d(1, 256), "C1 1D two-state problem, 256 cells, Free boundaries, gamma=1.4 (seed 1)"
    if name == "C2":
        return inputs.advected_wave_2d(512), "C2 2D advected density wave 512^2 periodic gamma=5/3"
    if name == "C3":
        return inputs.shear_layer_2d(2048, seed=3, nsteps=100), "C3 2D shear layer 2048^2 periodic gamma=5/3"
    if name == "implosion":
        return inputs.implosion_2d(2048, nsteps=100), "Liska-Wendroff implosion 2048^2, reflecting walls, gamma=1.4 (PAPER Sec. 4.4)"
    raise SystemExit(f"unknown workload {name}")


def kernel_name(variant: int, prec: int, stage: int, ndim: int, vanleer: bool = False) -> str:
    """Name of the stage kernel the library launches, from the variant the handle resolved."""
    from paper_2501_02317_b200 import binding as b
    ft = {0: "float", 1: "double", 2: "float"}[prec]
    if vanleer:
        if variant == b.KERNEL_TMA:
            return "stage_tma<1,1>" if stage == 1 else "stage_tma<2,2>"
        return ("vl::predict<%s>" if stage == 1 else "vl::correct<%s>") % ft
    if variant == b.KERNEL_TMA:
        return f"stage_tma<{stage},0,float>" if prec == 2 else f"stage_tma<{stage}>"
    if variant == b.KERNEL_STRIP:
        return f"stage_strip<{stage},float>" if prec == 2 else f"stage_strip<{stage}>"
    if variant == b.KERNEL_PAIRED:
        return f"stage_pair<{stage},{ndim}>"
    if variant == b.KERNEL_TILED:
        return f"stage_tiled<{ft},{stage},{ndim}>"
    return f"stage_simple<{ft},{stage},float>" if prec == 2 else f"stage_simple<{ft},{stage}>"


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_traffic(workload_name: str, precision: str, integrator: str, kernel: str):
    """(DRAM bytes per launch (read + write), where it was measured) of `kernel` from the committed
    ncu --set full captures (profiles/traffic.csv: one row per captured launch, keyed by workload, precision,
    integrator and the kernel name this file prints; `source` names the summary and `commit` the code it was
    captured on), or (None, None) when that combination was never captured.  The number is a property of the
    kernel at that commit, not of this run: the line says so in `traffic_source`."""
    import csv
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        with open(path) as f:
            for row in csv.DictReader(f):
                if (row["workload"] == workload_name and row["precision"] == precision
                        and row["integrator"] == integrator and row["bench_kernel"] == kernel):
                    return (float(row["dram_read_bytes"]) + float(row["dram_write_bytes"]),
                            f"profiles/{row['source']} (ncu --set full, commit {row['commit']})")
    except Exception:
        pass
    return None, None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [l for (t, l) in self.lines if t0 - 0.05 <= t <= t1 + 0.15] or [l for (_, l) in self.lines]
        sm, mx, reasons = [], [], set()
        for l in rows:
            p = [x.strip() for x in l.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0])); mx.append(float(p[1]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), p[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def time_oracle(pr_small, steps: int, warmup: int):
    """Oracle on the host cores: `steps` Heun steps (incl. its own CFL pass) of a bounded sample."""
    import oracle
    U = pr_small.U.copy()
    for _ in range(warmup):
        oracle.run(U, pr_small.gamma, pr_small.bc, pr_small.cfl, 1)
    t0 = time.time()
    oracle.run(U, pr_small.gamma, pr_small.bc, pr_small.cfl, steps)
    dt = time.time() - t0
    return pr_small.ncell * steps / dt, dt, oracle.num_threads()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2501_02317_b200 import inputs
    n = 96
    pr = inputs.turbulence_3d(n, seed=5) if args.workload.startswith("C5") else workload(args.workload)[0]
    sample = f"C5 recipe at {n}^3, {args.steps} timed Heun steps after {args.warmup} warm-up (oracle as it stands, OpenMP)"
    if not args.workload.startswith("C5"):
        sample = f"{pr.name} full size, {args.steps} steps"
    value, dt, cores = time_oracle(pr, args.steps, args.warmup)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload(args.workload)[1] if args.workload != "C5" else
                   "C5 3D decaying turbulence 512^3 periodic gamma=1.001", "precision": "fp64 (oracle)",
                   "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_ours(args):
    import numpy as np
    import torch
    from paper_2501_02317_b200 import binding, inputs, replicas

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist = dist_mod
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    pr, wl_name = workload(args.workload)
    prec = {"mixed": binding.PREC_MIXED, "fp64": binding.PREC_FP64, "single": binding.PREC_SINGLE}[args.precision]
    nx, ny, nz = pr.shape
    ncell = pr.ncell
    stream = torch.cuda.Stream()
    variant = {"auto": binding.KERNEL_AUTO, "simple": binding.KERNEL_SIMPLE, "tiled": binding.KERNEL_TILED,
               "paired": binding.KERNEL_PAIRED, "tma": binding.KERNEL_TMA}[args.kernel]
    vanleer = args.integrator == "vanleer"
    bpc = dict(BYTES_PER_CELL_SINGLE if prec == binding.PREC_SINGLE else BYTES_PER_CELL)
    if vanleer:
        bpc = dict(BYTES_PER_CELL_VL) if prec == binding.PREC_MIXED else {"stage1": 80.0, "stage2": 120.0}
    step_bytes = bpc["stage1"] + bpc["stage2"]
    h = binding.KratosHydro(nx, ny, nz, pr.gamma, pr.bc, precision=prec, stream=stream, kernel=variant,
                            integrator=binding.INTEGRATOR_VANLEER if vanleer else binding.INTEGRATOR_HEUN)
    if args.zchunk > 0:
        h.set_zchunk(args.zchunk)
    resolved = h.get_kernel()
    host = torch.from_numpy(pr.U).pin_memory()            # pinned host copy (e2e leg)
    with torch.cuda.stream(stream):
        dev = host.to("cuda", non_blocking=True)
        h.set_state(dev)
        stream.synchronize()
        del dev

        def barrier():
            torch.cuda.synchronize()
            if dist is not None:
                dist.barrier()
            torch.cuda.synchronize()

        # ---- device-resident throughput -------------------------------------------------------
        t = h.run(pr.cfl, args.warmup, 0.0)
        sampler = ClockSampler(local_rank)
        sampler.start()
        time.sleep(0.25)
        barrier()
        # kernel times: CUDA events around the stage launches inside the timed region -- of every step where a step takes
        # milliseconds, of every 4th step on the small grids (the event records themselves cost ~15 us per step)
        prof_every = 1 if ncell >= (1 << 25) else 4
        h.set_profiling(prof_every)
        l0 = h.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        w0 = time.time()
        e0.record(stream)
        t = h.run(pr.cfl, args.steps, t)
        e1.record(stream)
        barrier()
        w1 = time.time()
        ms = e0.elapsed_time(e1)
        launches = h.launch_count() - l0
        timing = h.get_timing()
        h.set_profiling(False)
        clocks = sampler.stop(w0, w1)
        value, job_s = replicas.job_value(ncell, args.steps, ms * 1e-3)   # max over ranks of the device time
        ms = job_s * 1e3
        hits = h.floor_hits()

        # ---- end to end: host buffers through the public API, copies inside the timed region -------
        e2e_steps = max(1, min(args.steps, args.e2e_steps))
        streamed = (resolved == binding.KERNEL_TMA and prec == binding.PREC_MIXED and not vanleer and nz >= 64
                    and not args.e2e_serial)
        e2e_mode = "whole block in, one step, whole block out (serial)"
        h2d_step = d2h_step = 40 * ncell
        st = host2 = None
        if streamed:
            # the block streams through the GPU in z chunks (outofcore.HostStepper): upload, kernels and download overlap
            from paper_2501_02317_b200 import outofcore
            try:
                h.set_state(host)
                dt_e = h.cfl_dt(pr.cfl)
                st = outofcore.HostStepper(nx, ny, nz, pr.gamma, pr.bc, chunk=args.e2e_chunk, p_ref=h.get_reference_pressure())
                host2 = torch.empty_like(host).pin_memory()
                st.step(host, host2, dt_e)                   # untimed: creates the chunk blocks
            except (RuntimeError, MemoryError) as exc:       # e.g. no room for a second pinned copy of the state
                sys.stderr.write(f"bench.py: streamed end-to-end leg not available ({exc}); using the serial one\n")
                if st is not None:
                    st.destroy()
                st, streamed = None, False
        if streamed:
            a, b = host2, host
            dt_e = st.next_dt(pr.cfl)
            st.h2d_bytes = st.d2h_bytes = 0
            barrier()
            w2 = time.time()
            for _ in range(e2e_steps):
                st.step(a, b, dt_e)                          # H2D of every chunk (+ overlap), its Heun step, D2H of its planes
                dt_e = st.next_dt(pr.cfl)                    # from the rate maxima the chunks' stage 2 reduced
                a, b = b, a
            barrier()
            e2e_s = time.time() - w2
            h2d_step, d2h_step = st.h2d_bytes // e2e_steps, st.d2h_bytes // e2e_steps
            e2e_mode = (f"streamed in z chunks of {st.chunk} planes (+{outofcore.HALO} planes of overlap on cut sides), two buffers "
                        "on two streams: upload, kernels and download overlap (paper_2501_02317_b200/outofcore.py)")
            st.destroy()
            del host2
        else:
            h.set_state(host)
            h.run(pr.cfl, 1, 0.0)
            h.get_state(host)
            barrier()
            w2 = time.time()
            te = 0.0
            for _ in range(e2e_steps):
                h.set_state(host)          # H2D of this step's input from pinned memory (5 N doubles)
                te = h.run(pr.cfl, 1, te)  # one Heun step (its CFL pass included: fresh state)
                h.get_state(host)          # D2H of the step's result
            barrier()
            e2e_s = time.time() - w2
        e2e_value, e2e_s = replicas.job_value(ncell, e2e_steps, e2e_s)
    h.destroy()

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    peak, peak_src = measured_peak()
    kern = {}
    for k in ("stage1", "stage2"):
        tot_ms, n = timing[k]
        if n:
            avg = tot_ms / n
            gbs = bpc[k] * ncell / (avg * 1e-3) / 1e9
            kern[k] = {"avg_ms": avg, "launches": n, "algorithmic_bytes": bpc[k] * ncell,
                       "achieved_gbs": gbs, "frac": gbs / peak}
    dom = max(kern, key=lambda k: kern[k]["avg_ms"] * kern[k]["launches"]) if kern else None
    roofline = None
    if dom:
        kname = kernel_name(resolved, prec, int(dom[-1]), 3 if nz > 1 else (2 if ny > 1 else 1), vanleer)
        traffic, traffic_src = ncu_traffic(args.workload, args.precision, args.integrator, kname)
        roofline = {"bound": "hbm", "kernel": kname, "achieved": kern[dom]["achieved_gbs"], "peak": peak,
                    "unit": "GB/s", "frac": kern[dom]["frac"], "traffic": traffic, "traffic_source": traffic_src,
                    "peak_source": peak_src, "bytes_per_cell": bpc[dom]}
    step_frac = value / world * step_bytes / (peak * 1e9)

    # ---- oracle on the host cores, bounded sample (rank 0, N = 1 only) ---------------------------
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        # bounded sample of the same recipe: about 10-30 s of CPU work at the oracle's ~8e6 cell-updates/s on 16 cores
        n_s = 192 if nz > 1 else 2048
        st = 20
        small = inputs.turbulence_3d(n_s, seed=5) if nz > 1 else inputs.shear_layer_2d(n_s, seed=3)
        v, dt_s, cores = time_oracle(small, st, 0)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{small.name} recipe at {n_s}^{3 if nz > 1 else 2}, {st} Heun steps ({dt_s:.1f} s)"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": {0: "f32 flux / f64 state", 1: "f64", 2: "f32"}[prec], "data": "synthetic",
        "config": {"workload": wl_name, "grid": [nx, ny, nz], "precision": args.precision,
                   "scheme": "PLM-minmod + HLLC + " + ("van Leer" if vanleer else "Heun"), "kernel": args.kernel, "cfl": pr.cfl, "parallelism": f"replicas x{world}",
                   "l2": l2_note(ncell, 4 if prec == 2 else 8),
                   "floor_hits": hits},
        "hbm_roofline_frac_step": step_frac,
        "roofline": roofline, "kernels": kern,
        "kernel_timing": "CUDA events on the library's stream around the stage launches of every "
                         + ("step" if prof_every == 1 else f"{prof_every}th step") + " of the timed region",
        "cpu_baseline": cpu,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d_step, "d2h_bytes_per_step": d2h_step,
                "steps": e2e_steps, "mode": e2e_mode},
        "gpu_launches": int(launches), "clocks": clocks,
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def run_slabs(args):
    """One block as z slabs (row f-4): --slabs R in this process, or one slab per rank under torchrun."""
    import numpy as np
    import torch
    from paper_2501_02317_b200 import binding, slab

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist = dist_mod
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    if args.precision != "mixed" or args.integrator != "heun":
        raise SystemExit("communication boundaries serve the mixed-precision Heun path")
    pr, wl_name = workload(args.workload)
    nx, ny, nz = pr.shape
    ncell = pr.ncell
    stream = torch.cuda.Stream()
    nslab = world if world > 1 else args.slabs
    s = slab.SlabSolver(nx, ny, nz, pr.gamma, pr.bc, world=nslab, stream=stream)
    if args.zchunk > 0:
        for b in s.blocks.values():
            b.set_zchunk(args.zchunk)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    s.set_state(pr.U)
    t = s.run(pr.cfl, args.warmup, 0.0)
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.25)
    barrier()
    for b in s.blocks.values():
        b.set_profiling(True)
    l0 = s.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    w0 = time.time()
    e0.record(stream)
    t = s.run(pr.cfl, args.steps, t)
    e1.record(stream)
    barrier()
    w1 = time.time()
    ms = e0.elapsed_time(e1)
    launches = s.launch_count() - l0
    timing = {"stage1": [0.0, 0], "stage2": [0.0, 0]}
    for b in s.blocks.values():
        tm = b.get_timing()
        for k in timing:
            timing[k][0] += tm[k][0]
            timing[k][1] += tm[k][1]
        b.set_profiling(False)
    clocks = sampler.stop(w0, w1)
    from paper_2501_02317_b200 import replicas
    job_s = replicas.job_time(ms * 1e-3)                 # max over ranks of the device time
    value = ncell * args.steps / job_s                   # ONE block, whatever the number of slabs: strong scaling
    hits = s.floor_hits()
    # end to end: the whole block from and to host memory through the driver, one step per round trip
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    host = torch.from_numpy(pr.U).pin_memory()
    barrier()
    w2 = time.time()
    for _ in range(e2e_steps):
        s.set_state(host)                  # H2D from pinned memory: the whole block cut into slabs on the device (one
                                           # process), or the planes this rank owns only (one process per GPU)
        s.run(pr.cfl, 1, 0.0)
        if world == 1:
            s.get_state_into(host)         # slabs joined on the device, one D2H copy
            down = 40 * ncell
        else:
            got = s.get_state()
            down = sum(int(g.size) * 8 for g in got.values())
    barrier()
    e2e_s = replicas.job_time(time.time() - w2)
    # bytes that crossed the bus per step, summed over the ranks (counted from the copies, not from the grid)
    moved = s.comm.all_sum([float(s.last_upload_bytes), float(down)])
    h2d_bytes, d2h_bytes = int(moved[0]), int(moved[1])
    s.destroy()
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    peak, peak_src = measured_peak()
    planes = 2 * sum(1 for r in range(nslab) for nb in s.dec.neighbours(r) if nb is not None)
    halo_bytes = 2 * planes * 5 * nx * ny * 8            # both stages: every cut face side receives two planes of 5 fields
    kern = {}
    for k in ("stage1", "stage2"):
        tot_ms, n = timing[k]
        if n:
            per_step = tot_ms / (n / len(s.ranks) if len(s.ranks) else 1)   # the slabs of this process run one after the other
            gbs = BYTES_PER_CELL[k] * ncell / world / (per_step * 1e-3) / 1e9
            kern[k] = {"avg_ms": per_step, "launches": n, "algorithmic_bytes": BYTES_PER_CELL[k] * ncell / world,
                       "achieved_gbs": gbs, "frac": gbs / peak}
    dom = max(kern, key=lambda k: kern[k]["avg_ms"]) if kern else None
    roofline = None
    if dom:
        roofline = {"bound": "hbm", "kernel": f"stage_tma<{dom[-1]}> x {len(s.ranks)} slabs per step", "achieved": kern[dom]["achieved_gbs"],
                    "peak": peak, "unit": "GB/s", "frac": kern[dom]["frac"], "traffic": None, "traffic_source": None,
                    "peak_source": peak_src, "bytes_per_cell": BYTES_PER_CELL[dom]}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": job_s * 1e3 / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
        "dtype": "f32 flux / f64 state", "data": "synthetic",
        "config": {"workload": wl_name, "grid": [nx, ny, nz], "precision": "mixed", "scheme": "PLM-minmod + HLLC + Heun",
                   "kernel": "tma", "cfl": pr.cfl,
                   "parallelism": (f"{nslab} z slabs, one per GPU (communication boundaries, NCCL all-reduce for dt)" if world > 1 else
                                   f"{nslab} z slabs in one process on one GPU, advanced in lock step (communication boundaries)"),
                   "halo_bytes_per_step": halo_bytes,
                   "l2": f"state is {5 * 8 * ncell / 1e9:.2f} GB per copy, larger than the 126 MB L2 (no flush needed)", "floor_hits": hits},
        "hbm_roofline_frac_step": value / world * 200.0 / (peak * 1e9),
        "roofline": roofline, "kernels": kern, "cpu_baseline": None,
        "e2e": {"value": ncell * e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d_bytes, "d2h_bytes_per_step": d2h_bytes,
                "steps": e2e_steps},
        "gpu_launches": int(launches), "clocks": clocks,
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


L2_BYTES = 126e6   # B200


def l2_note(ncell, word):
    """What the config says about the L2: a step touches two copies of the state (Heun: U and the predictor).  Larger than
    the L2 per copy: every step streams from HBM, no flush needed.  Otherwise part or all of the working set stays on chip
    between steps (the steps are data-dependent, so nothing can be flushed in between without changing the run): the HBM
    fraction of such a line is not a statement about HBM."""
    copy = 5 * word * ncell
    if copy > L2_BYTES:
        return f"state is {copy / 1e9:.2f} GB per copy, larger than the 126 MB L2 (no flush needed)"
    if 2 * copy > L2_BYTES:
        return (f"state is {copy / 1e6:.0f} MB per copy: one copy fits the 126 MB L2, the step's two do not -- partly on-chip, "
                "no flush between steps (steps are data-dependent); the HBM fraction is flattered by L2 hits")
    return (f"on-chip: state is {copy / 1e6:.2f} MB per copy, the whole working set stays in the 126 MB L2; launch-bound, "
            "the HBM fraction says nothing here")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C5")
    ap.add_argument("--precision", default="mixed", choices=["mixed", "fp64", "single"],
                    help="mixed: fp32 flux / fp64 state (the headline); fp64: all-fp64; single: all-fp32 (PAPER.md:240)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--e2e-chunk", type=int, default=32, help="planes per chunk of the streamed end-to-end step")
    ap.add_argument("--e2e-serial", action="store_true", help="end-to-end leg: whole block in, step, whole block out")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--kernel", default="auto", choices=["auto", "simple", "tiled", "paired", "tma"],
                    help="stage kernel variant (default: the library's own choice)")
    ap.add_argument("--integrator", default="heun", choices=["heun", "vanleer"],
                    help="time integrator (PAPER.md Sec. 3.3); the headline metric is quoted on heun")
    ap.add_argument("--zchunk", type=int, default=0, help="planes per slab of the marching kernels (0 = auto)")
    ap.add_argument("--slabs", type=int, default=1, help="cut the block into this many z slabs in this process (row f-4)")
    ap.add_argument("--decomposition", default="replicas", choices=["replicas", "slab"],
                    help="what --gpus N > 1 means: N replicas (default, DESIGN.md section 9) or N z slabs of one block")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    elif args.slabs > 1 or (args.decomposition == "slab" and int(os.environ.get("WORLD_SIZE", "1")) > 1):
        run_slabs(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
