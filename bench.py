#!/usr/bin/env python
"""bench.py -- coupled FDTD-LLG throughput on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C]

One "step" = one full time step of the hot path (H/M half-step, E update, H/M half-step:
PAPER.md:94, 152) over the whole synthetic grid.  Default workload: BASELINE.json configs[4],
the 768^3 coupled grid named "throughput and HBM-roofline run" (the largest single-GPU
configuration; configs[1] is Maxwell-only and configs[0] is the 32^3 parity case).

Prints ONE JSON line: metric/value (Gcell-updates/s, inputs resident in HBM, CUDA-graph replay),
e2e (same metric through the public API with HOST buffers: H2D of the initial fields, K steps,
D2H of all 15 result arrays inside the timed region), roofline (dominant kernel, algorithmic
bytes / CUDA-event duration against the measured HBM peak), cpu_baseline (the oracle as it
stands, timed on this box's host cores on a bounded sample, all cores and one thread), clocks,
gpu_launches, and other_configs: the same measurement on the grids shaped like the paper's
waveguide and tunable-filter runs (BASELINE.json configs 2, 3, 4 at full size and the paper's own
1024 x 4 x 512 base case).

N > 1 (torchrun, one process per GPU): the grid is cut into z-slabs (domain
decomposition is the paper's parallelism), the halo exchange is done by peer stores inside the
update kernels over NVLink, one 8-byte NCCL max-allreduce per sub-step merges the LLG stopping
test and orders the slabs (paper_2103_12819_b200/slabs.py).  --scaling weak (default): every rank
holds one copy of the config, the copies stacked along z (the paper grows its base case in z the
same way); --scaling strong: the config's own grid cut into N slabs.  value = all
ranks' cell updates / max-over-ranks device time.

--impl reference times the CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "coupled FDTD-LLG Gcell-updates/s (fp64)"
UNIT = "Gcell-updates/s"

# algorithmic 8-byte words per cell and launch: every array
# read once and written once per sweep, stencil neighbours served on chip
WORDS = {"h_update": 9,      # E 3 + H 3 read, H 3 written
         "hm_first": 27,     # E 3 + H^n 3 + M^n 9 read, M^1 9 + H^1 3 written
         "hm_second": 39,    # + H^1 3 + M^1 9 read, M^2 9 + H^2 3 written
         "hm_iter": 39,      # r >= 3: as r = 2
         "e_update": 9,      # E 3 + H 3 read, E 3 written
         "eh_fused": 12}     # E 3 + H 3 read, E 3 + H 3 written: eq. 11 fused with the merged H update
OTHER_CONFIGS = (2, 3, 4, 6)


def _parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config number 1..5 (6: the paper's weak-scaling base case, "
                         "the tunable filter on 1024x4x512 cells)")
    ap.add_argument("--shape", default=None, help="nx,ny,nz (default: the config's full size)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-sample-shape", default="128,128,128")
    ap.add_argument("--cpu-sample-steps", type=int, default=30)
    ap.add_argument("--cpu-single-shape", default="64,64,64")
    ap.add_argument("--cpu-single-steps", type=int, default=4)
    ap.add_argument("--no-other-configs", action="store_true",
                    help="skip the extra measurements on configs 2, 3, 4, 6 (they run with the default config at N = 1)")
    ap.add_argument("--other-steps", type=int, default=50)
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = one copy of the config per rank, stacked in z; strong = the config's grid cut into N slabs")
    ap.add_argument("--no-merge-h", action="store_true", help="fdtd_llg_options.merge_h = 0 (two H half-steps everywhere)")
    ap.add_argument("--kernel-path", type=int, default=0,
                    help="fdtd_llg_options.kernel_path: 0 = staged sweeps where they apply (default), "
                         "1 = direct-load kernels, 5 = staged sweeps whatever the box size")
    ap.add_argument("--plain-graph", action="store_true",
                    help="capture the step without the conditional node (use_graph = 2), so that ncu lists "
                         "the kernels of the replayed steps too")
    ap.add_argument("--time-scheme", type=int, default=0,
                    help="0 = second-order scheme (the BASELINE metric), 1 = first-order scheme (PAPER.md:102-150)")
    return ap.parse_args()


def _shape(args):
    return tuple(int(v) for v in args.shape.split(",")) if args.shape else None


def _workload_name(w):
    return f"{w.name} {w.nx}x{w.ny}x{w.nz}"


# ------------------------------------------------------------------ clocks

class ClockSampler:
    """nvidia-smi clocks / throttle reasons of one GPU, sampled every 200 ms while running."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "200", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), [c.strip() for c in line.split(",")]))

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()

    def summary(self, t0, t1):
        rows = [r for t, r in self.rows if t0 <= t <= t1 and len(r) >= 7] or \
               [r for _, r in self.rows[-3:] if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        sm = sorted(float(r[0]) for r in rows)
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        reasons = [n for q, n in enumerate(names) if any(r[3 + q].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]),
                "power_w_max": max(float(r[2]) for r in rows), "reasons": reasons,
                "samples": len(rows)}


# ------------------------------------------------------------------ the oracle legs

def _oracle_rate(cfg, shape, steps, warmup=0, time_scheme=0):
    """Cell-updates/s of the CPU oracle (as it stands) on a reduced-shape copy of the workload."""
    from oracle import Oracle  # noqa: F401  (the one place bench.py may execute oracle/)
    from oracle.cpu_oracle import omp_threads
    from paper_2103_12819_b200 import workloads as wl
    from oracle import oracle_from_workload
    w = wl.make_config(cfg, shape=shape)
    o = oracle_from_workload(w, time_scheme=time_scheme)
    if warmup:
        o.step(warmup)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    return w, w.cells * steps / dt, dt, omp_threads()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    shape = tuple(int(v) for v in args.cpu_sample_shape.split(","))
    from paper_2103_12819_b200 import workloads as wl
    full = wl.CONFIGS[args.config].__defaults__[0] if args.shape is None else _shape(args)
    w, rate, dt, cores = _oracle_rate(args.config, shape, args.steps, args.warmup, args.time_scheme)
    sample = (f"config {args.config} structure at {shape[0]}x{shape[1]}x{shape[2]} cells, "
              f"{args.steps} steps after {args.warmup} warm-up (the full {full[0]}x{full[1]}x{full[2]} "
              f"grid is out of the oracle's reach; the rate per cell is what is compared)")
    val = rate * 1e-9
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": f"{w.name} {w.nx}x{w.ny}x{w.nz} (bounded sample of {full[0]}x{full[1]}x{full[2]})", "sample": sample,
                       "time_scheme": "first-order" if args.time_scheme else "second-order"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------ ours

def _peak():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return float(json.loads(p.read_text())["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def _ncu_traffic(kernel, workload):
    """dram bytes per launch of `kernel` from the committed ncu capture, if it was taken on this
    workload (profiles/traffic.csv: kernel,workload,dram_bytes_per_launch)."""
    f = ROOT / "profiles" / "traffic.csv"
    if not f.exists():
        return None
    for line in f.read_text().splitlines():
        c = [x.strip() for x in line.split(",")]
        if len(c) >= 3 and c[0] == kernel and c[1] == workload:
            try:
                return float(c[2])
            except ValueError:
                return None
    return None


def _oracle_single_thread(cfg, shape, steps, time_scheme):
    """The oracle on ONE thread (libgomp is told so; restored afterwards)."""
    import ctypes
    from oracle.cpu_oracle import omp_threads
    try:
        gomp = ctypes.CDLL("libgomp.so.1")
        gomp.omp_set_num_threads(1)
    except OSError:
        return None
    try:
        _, rate, dt, _ = _oracle_rate(cfg, shape, steps, time_scheme=time_scheme)
    finally:
        gomp.omp_set_num_threads(omp_threads())
    return {"value": rate * 1e-9, "unit": UNIT, "cores": 1,
            "sample": f"config {cfg} structure at {shape[0]}x{shape[1]}x{shape[2]}, {steps} steps, {dt:.1f} s"}


def _timed_steps(sim, K, W, barrier):
    """K steps of CUDA-graph replay after W warm-up steps, timed with CUDA events on the library's stream."""
    import torch
    stream = sim.stream
    sim.step(max(W, 1))
    stream.synchronize()
    barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    sim.step(K)
    e1.record(stream)
    stream.synchronize()
    torch.cuda.synchronize()
    barrier()
    return e0.elapsed_time(e1)


def _kernel_breakdown(sim, K, cells, ms_step, peak, peak_src, name):
    """roofline block: an event pair around every launch of K more steps (fdtd_llg_step_timed)."""
    from paper_2103_12819_b200.binding import MAT_BITS
    st = sim.stats()
    prof = sim.step_timed(K)
    box = st["sweep_cells"]
    mask = st["material_array_mask"]
    extra = {"h_update": bool(mask & MAT_BITS["mu_r"]),
             "hm_first": sum(bool(mask & MAT_BITS[m]) for m in ("Ms", "alpha", "gamma", "mu_r")),
             "e_update": sum(bool(mask & MAT_BITS[m]) for m in ("eps_r", "sigma"))}
    extra["hm_iter"] = extra["hm_second"] = extra["hm_first"]
    extra["eh_fused"] = extra["e_update"]
    fused = prof["eh_fused"][1] > 0        # the E phase ran by regions: fused outside the box, E only in it
    prof = dict(prof)                       # r = 2 and r >= 3 are the same kernel: one class
    a2, b2 = prof.pop("hm_second"), prof["hm_iter"]
    prof["hm_iter"] = (a2[0] + b2[0], a2[1] + b2[1])
    per_class = {}
    for cls, (cms, cnt) in prof.items():
        if cnt == 0:
            continue
        ent = {"launches": cnt, "ms_total": cms, "us_per_launch": 1e3 * cms / cnt}
        if cls in WORDS:
            # cells one launch covers: the sweep box (LLG sweeps), the whole grid (E update), the
            # complement of the box split over its slabs (H update: two half-steps per step, or
            # one merged update per step)
            if cls.startswith("hm_"):
                ncell = box
            elif cls == "e_update":
                ncell = (box if fused else cells) * K / cnt
            elif cls == "eh_fused":
                ncell = (cells - box) * K / cnt
            elif fused:
                continue            # left-over faces of a region that could not be fused: not modelled
            else:
                ncell = (cells - box) * (1 if st["merged_h"] else 2) * K / cnt
            ent["alg_bytes_per_launch"] = 8.0 * (WORDS[cls] + extra[cls]) * ncell
            ent["alg_GBps"] = ent["alg_bytes_per_launch"] / (cms / cnt * 1e-3) * 1e-9
        per_class[cls] = ent
    timed = [c for c in per_class if "alg_GBps" in per_class[c]]
    dom = max(timed, key=lambda c: per_class[c]["ms_total"])
    staged = bool(st["staged_sweeps"])
    dom_kernel = {"h_update": "k_h_update",
                  "hm_first": "k_hm_stage<FIRST>" if staged else "k_hm_sweep<FIRST>",
                  "hm_iter": "k_hm_stage<ITER>" if staged else "k_hm_sweep<ITER>",
                  "e_update": "k_eh_stage" if fused else "k_e_update",
                  "eh_fused": "k_eh_fused"}[dom]
    achieved = per_class[dom]["alg_GBps"]
    step_bytes = sum(per_class[c]["alg_bytes_per_launch"] * per_class[c]["launches"] for c in timed) / K
    traffic = _ncu_traffic(dom_kernel, name)
    return {"bound": "hbm", "kernel": dom_kernel, "achieved": achieved, "peak": peak,
            "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
            "traffic": traffic,
            "traffic_source": ("profiles/traffic.csv: dram__bytes_read.sum + dram__bytes_write.sum per launch from the "
                               "committed ncu --set full capture of this kernel on this workload (not measured in this run)"
                               if traffic is not None else None),
            "alg_bytes_per_launch": per_class[dom]["alg_bytes_per_launch"],
            "us_per_launch": per_class[dom]["us_per_launch"],
            "share_of_step": per_class[dom]["ms_total"] / sum(v["ms_total"] for v in per_class.values()),
            "how": f"CUDA events around every launch over {K} steps (fdtd_llg_step_timed, plain launches)",
            "whole_step": {"alg_bytes_per_step": step_bytes,
                           "achieved": step_bytes / (ms_step * 1e-3) * 1e-9,
                           "frac": step_bytes / (ms_step * 1e-3) * 1e-9 / peak},
            "kernels": per_class}


def _measure_other(cfg, K, W, dev, args, peak, peak_src, vis_index):
    """One of the other configs at full size: graph replay + the class breakdown, no e2e leg."""
    import torch
    from paper_2103_12819_b200 import workloads as wl
    from paper_2103_12819_b200.binding import from_workload
    w = wl.make_config(cfg, device=dev)
    name, cells = _workload_name(w), w.cells
    sim = from_workload(w, device=dev, kernel_path=args.kernel_path, merge_h=not args.no_merge_h)
    del w
    # These grids step in 0.2-3 ms: a timed region of K = 50 steps would be over before the GPU has
    # left the clock / power state of the run before it (right after the 768^3 run the SM clock is
    # still at the power-capped 1.4 GHz and a 17 ms measurement comes out 15 % low).  A pilot sets
    # the step count so that the warm-up lasts >= 0.25 s and the timed region >= 0.5 s.
    pilot = _timed_steps(sim, 10, max(W, 3), lambda: None) / 10.0
    Kt = int(min(4000, max(K, 500.0 / pilot)))
    sampler = ClockSampler(vis_index)
    sampler.start()
    t0 = time.perf_counter()
    ms = _timed_steps(sim, Kt, int(max(W, 250.0 / pilot)), lambda: None)
    t1 = time.perf_counter()
    clocks = sampler.summary(t0, t1)
    sampler.stop()
    st = sim.stats()
    roof = _kernel_breakdown(sim, K, cells, ms / Kt, peak, peak_src, name)
    K = Kt
    out = {"workload": name, "cells": cells, "magnetic_cells": st["magnetic_cells"], "steps": K, "clocks": clocks,
           "gcell_s": cells * K / (ms * 1e-3) * 1e-9, "ms_per_step": ms / K,
           "launches_per_step": st["launches_per_step"], "staged_sweeps": st["staged_sweeps"],
           "merged_h": st["merged_h"], "staged_maxwell": st["staged_maxwell"],
           "llg_iterations_per_halfstep": st["iters_total"] / max(1, st["halfsteps"]),
           "alg_bytes_per_cell_step": roof["whole_step"]["alg_bytes_per_step"] / cells,
           "whole_step_frac": roof["whole_step"]["frac"], "whole_step_GBps": roof["whole_step"]["achieved"],
           "dominant_kernel": roof["kernel"], "dominant_frac": roof["frac"],
           "dominant_traffic": roof["traffic"],
           "kernels": {k: {"us_per_launch": v["us_per_launch"], "launches": v["launches"],
                           "alg_GBps": v.get("alg_GBps")} for k, v in roof["kernels"].items()}}
    sim.close()
    del sim
    torch.cuda.empty_cache()
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2103_12819_b200 import workloads as wl
    from paper_2103_12819_b200.binding import FIELD_NAMES, from_workload

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    local %= max(1, torch.cuda.device_count())      # more ranks than GPUs: share (smoke tests, gloo)
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        # NCCL over NVLink is the product path; FDTD_LLG_DIST_BACKEND=gloo carries the 8-byte words
        # through the host instead (ranks sharing one GPU, where NCCL refuses to run)
        backend = os.environ.get("FDTD_LLG_DIST_BACKEND", "nccl")
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=dev)
        else:
            dist.init_process_group(backend)

    from paper_2103_12819_b200.replicas import barrier, max_over_ranks, whole_job_rate

    K, W = args.steps, max(args.warmup, 0)
    peak, peak_src = _peak()
    w = wl.make_config(args.config, shape=_shape(args), device=dev)
    name = _workload_name(w)
    slab, slab_error = None, None
    if world > 1:
        # z-slabs: weak = one copy of the grid per rank stacked in z, strong = the grid cut in N
        from paper_2103_12819_b200.slabs import (PERIODIC, DistSlab, SlabSetupError, cut_workload, plan_slabs,
                                                 stack_copies)
        if args.scaling == "weak":
            plan = plan_slabs(w.nz * world, world, False)[rank]
            w = stack_copies(w, plan)
            name += f" x {world} copies stacked in z"
        else:
            plan = plan_slabs(w.nz, world, w.bc[2] == PERIODIC)[rank]
            w = cut_workload(w, plan)
            name += f" cut into {world} z-slabs"
        try:
            slab = DistSlab(w, plan, dev, kernel_path=args.kernel_path, merge_h=not args.no_merge_h,
                            time_scheme=args.time_scheme)
            sim = slab.sim
        except SlabSetupError as e:
            # every rank gets this error together (slabs.DistSlab).  The measurement falls back to N
            # independent replicas of the config and SAYS SO in config.parallelism: no halo exchange,
            # no allreduce -- a timing of N single-GPU runs, not of the decomposed grid.
            slab, slab_error = None, str(e)
            del w
            torch.cuda.empty_cache()
            w = wl.make_config(args.config, shape=_shape(args), device=dev)
            name = _workload_name(w) + f" x {world} independent replicas"
    if slab is None:
        sim = from_workload(w, device=dev, kernel_path=args.kernel_path, time_scheme=args.time_scheme,
                            use_graph=2 if args.plain_graph else True, merge_h=not args.no_merge_h)
    cells = w.nx * w.ny * w.nz          # this rank's cells
    stream = sim.stream

    # host copies of the initial state for the end-to-end leg (pinned), before the device inputs go
    host_in = None
    if not args.no_e2e:
        def pin(t):
            return None if t is None else torch.empty(t.shape, dtype=t.dtype).pin_memory().copy_(t)
        host_in = {"E": [pin(t) for t in w.E], "H": [pin(t) for t in w.H],
                   "M_cell": [pin(t) for t in w.M_cell]}
    del w
    torch.cuda.empty_cache()

    vis = [v for v in os.environ.get("CUDA_VISIBLE_DEVICES", "").split(",") if v.strip()]
    sampler = ClockSampler(vis[local] if local < len(vis) else local)
    sampler.start()

    # ---- device-resident throughput
    t_a = time.perf_counter()
    if slab is None:
        ms = max_over_ranks(_timed_steps(sim, K, W, barrier), dev)      # CUDA-graph replay of K steps
        st = sim.stats()
        launches = K * st["launches_per_step"]
    else:
        slab.step(max(W, 1))
        stream.synchronize()
        barrier()
        torch.cuda.synchronize()
        l0 = sim.stats()["kernel_launches"]
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        slab.step(K)
        e1.record(stream)
        stream.synchronize()
        torch.cuda.synchronize()
        barrier()
        ms = max_over_ranks(e0.elapsed_time(e1), dev)
        st = sim.stats()
        launches = st["kernel_launches"] - l0
    value = whole_job_rate(cells, K, ms * 1e-3, world) * 1e-9

    # ---- roofline
    if slab is None:
        roofline = _kernel_breakdown(sim, K, cells, ms / K, peak, peak_src, name)
    else:
        # a connected slab has no per-launch timing hook: the whole step against the peak, with the
        # single-GPU byte model (27 + 39 (R - 1) words per half-step on the sweep box, 9 per
        # outside update, 9 for the E update; + 1 per material array a kernel reads)
        from paper_2103_12819_b200.binding import MAT_BITS
        mask, box = st["material_array_mask"], st["sweep_cells"]
        R = st["iters_total"] / max(1, st["halfsteps"])
        xm = sum(bool(mask & MAT_BITS[m]) for m in ("Ms", "alpha", "gamma", "mu_r"))
        xe = sum(bool(mask & MAT_BITS[m]) for m in ("eps_r", "sigma"))
        words = 2 * box * ((27 + xm) + (39 + xm) * max(0.0, R - 1)) \
            + (cells - box) * (1 if st["merged_h"] else 2) * (9 + bool(mask & MAT_BITS["mu_r"])) \
            + cells * (9 + xe)
        ach = 8.0 * words / (ms / K * 1e-3) * 1e-9
        roofline = {"bound": "hbm", "kernel": "whole step of one rank (z-slab run: no per-launch timing hook)",
                    "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "peak_source": peak_src,
                    "traffic": None, "alg_bytes_per_launch": 8.0 * words,
                    "how": "algorithmic bytes of one rank's step / max-over-ranks step time (CUDA events)",
                    "halo": {"bytes_per_plane": 8 * sim.shape[1] * sim.shape[2],
                             "planes_per_substep": "H_x, H_y up + H_z down per (H,M) sweep; E_x, E_y down per E update",
                             "allreduces_per_step": slab.merges / max(1, K + max(W, 1)),
                             "host_checks_per_step": slab.host_checks / max(1, K + max(W, 1))}}
    t_c = time.perf_counter()
    clocks = sampler.summary(t_a, t_c)

    # ---- end to end through the public API with HOST buffers
    e2e = None
    if host_in is not None:
        out = {nm: torch.empty(sim.shape, dtype=torch.float64).pin_memory() for nm in FIELD_NAMES}
        if not st["magnetic_cells"]:
            out = {k: v for k, v in out.items() if not k.startswith("M")}
        h2d = sum(t.numel() * 8 for g in host_in.values() for t in g if t is not None)
        d2h = sum(t.numel() * 8 for t in out.values())
        step = (lambda n: sim.step(n)) if slab is None else (lambda n: slab.step(n))
        sim.set_fields(host_in["E"], host_in["H"], host_in["M_cell"])   # warm the path once
        barrier()
        step(1)
        stream.synchronize()
        barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        sim.set_fields(host_in["E"], host_in["H"], host_in["M_cell"])   # H2D from pinned memory
        if slab is not None:
            barrier()            # every slab's ghost planes are in place before a neighbour stores into them
        step(K)
        sim.read_fields(out=out)                                         # D2H, synchronises
        torch.cuda.synchronize()
        dt = max_over_ranks(time.perf_counter() - t0, dev)
        barrier()
        e2e = {"value": whole_job_rate(cells, K, dt, world) * 1e-9, "unit": UNIT,
               "h2d_bytes_per_step": h2d / K, "d2h_bytes_per_step": d2h / K,
               "seconds": dt, "what": f"set_fields(host) + step({K}) + read_fields(host), wall clock"}
        del out, host_in
    sampler.stop()
    iters_per_half = st["iters_total"] / max(1, st["halfsteps"])
    mag = st["magnetic_cells"]
    if slab is not None:
        slab.close()
    else:
        sim.close()
    del sim
    torch.cuda.empty_cache()

    # ---- the grids shaped like the paper's waveguide / tunable-filter runs (north_star)
    other = None
    if rank == 0 and world == 1 and args.config == 5 and args.shape is None and not args.no_other_configs \
            and not args.time_scheme:
        other = {}
        for cfg in OTHER_CONFIGS:
            try:
                other[f"config{cfg}"] = _measure_other(cfg, args.other_steps, max(W, 3), dev, args, peak, peak_src,
                                                       vis[local] if local < len(vis) else local)
            except Exception as e:  # a failure here must not lose the headline line
                other[f"config{cfg}"] = {"error": repr(e)}

    # ---- CPU baseline: the oracle on a bounded sample (rank 0, N = 1), all cores and one thread
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        shp = tuple(int(v) for v in args.cpu_sample_shape.split(","))
        _, rate, dt, cores = _oracle_rate(args.config, shp, args.cpu_sample_steps, time_scheme=args.time_scheme)
        cpu = {"value": rate * 1e-9, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"config {args.config} structure at {shp[0]}x{shp[1]}x{shp[2]}, "
                         f"{args.cpu_sample_steps} steps, {dt:.1f} s",
               "host_cpus": os.cpu_count(),
               "single_thread": _oracle_single_thread(args.config, tuple(int(v) for v in args.cpu_single_shape.split(",")),
                                                      args.cpu_single_steps, args.time_scheme)}

    if rank == 0:
        # a run that fell back to independent replicas did not measure the decomposed grid: no headline
        # value (the replica rate is kept under its own key, the parallelism string says what ran)
        line = {"metric": METRIC, "value": value if slab_error is None else None, "unit": UNIT,
                "n_gpus": world, "steps": K,
                "warmup": W, "ms_per_step": ms / K, "higher_is_better": True,
                "scaling": args.scaling if (world > 1 and slab_error is None) else "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": name, "cells": cells * world,
                           "cells_per_gpu": cells, "magnetic_cells_rank0": mag,
                           "llg_iterations_per_halfstep": iters_per_half,
                           "parallelism": ("single-gpu" if world == 1 else
                                           f"z-slabs x{world}: peer stores in the update kernels + 8-byte max-allreduce per sub-step"
                                           if slab_error is None else
                                           f"REPLICAS x{world} (no exchange): the z-slab set-up failed: {slab_error}"),
                           "l2": "state far larger than L2 (no flush needed)" if cells * 48 > 4e8
                                 else "state fits L2: latency-bound case, no roofline claim",
                           "time_loop": "CUDA graph replay" if (world == 1 or slab_error is not None) else "plain launches (sub-steps)",
                           "kernel_path": args.kernel_path, "merge_h": st["merged_h"],
                           "staged_sweeps": st["staged_sweeps"], "staged_maxwell": st["staged_maxwell"],
                           "time_scheme": "first-order" if args.time_scheme else "second-order"},
                "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "clocks": clocks,
                "gpu_launches": launches, "other_configs": other,
                **({} if slab_error is None else {"replicas_value": value}),
                "context": "paper: 59x node-by-node GPU speedup (8x V100 vs 32-core Haswell, "
                           "PAPER.md:229, 277) -- another machine, context only"}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = _parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
