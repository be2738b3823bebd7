#!/usr/bin/env python
"""bench.py -- atom-steps/s of the FLARE B2 hot path on B200 (BASELINE.json metric).

A "step" is one velocity-Verlet MD step = one pass of the whole hot path (neighbour build,
descriptors, beta + Sigma quadratic forms, back-propagated forces, gather, integrator) over the
synthetic H2/Pt(111)-shaped system.  Default workload: config 3
(1 082 016 atoms, n_max 8, l_max 3, P 544, variance on, dt 0.5 fs) -- the linear-scaling regime
the paper's metric is quoted in; it fits one GPU.

    python bench.py --gpus N --steps K --warmup W [--workload c1|c2|c3|c4|c5a|c5b|c5c|tile] [--sweep none|small|full]
    python bench.py --impl reference ...   # the CPU oracle, as it stands, on a bounded sample

The timed region (K steps between two CUDA events, after W warm-up steps) is repeated `--repeats` times (default 3);
the line reports the MEDIAN repeat and lists all of them.  At N = 1 the same line also carries
`roofline` (the dominant kernel), `roofline_kernels` (every phase against its own bound), `sweep` (configs 1, 2, 4 and
the six runs of config 5, short step counts) and `cpu_baseline` (the oracle on the host cores, all cores and 1 thread).

For N > 1 (launched by torch.distributed.run) the ranks share ONE slab px x py times the C3 cell, one C3-sized domain
per GPU on a 2-D process grid with a halo exchange per step (paper_2204_12573_b200/halo.py + the device data plane
flare_domain_*; `--replicas` runs N independent copies instead); value = all ranks' atom-steps / max-over-ranks device
time.  `--decomposed` at N = 1 runs the same path with the rank as its own neighbour.  Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import csv
import datetime
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2204_12573_b200 import workloads  # noqa: E402

METRIC = "atom-steps/s on 1 B200 (FP64 FLARE B2 energy+forces+variance)"
UNIT = "atom-steps/s"
QFORM_TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r02_qform_traffic.csv")

_C5 = {"c5a": (8, 3), "c5b": (10, 4), "c5c": (12, 6)}


def make_system(name: str):
    if name == "c1":
        return workloads.config1(), "C1 fcc Pt 256 atoms (n_max 8, l_max 3, P 144), dt 1 fs, 300 K"
    if name == "c2":
        return workloads.config2(), "C2 H2/Pt(111) 1264 atoms (2 species, n_max 8, l_max 3, P 544), dt 0.5 fs, 500 K"
    if name == "c3":
        return workloads.config3(), "C3 H2/Pt(111) 1 082 016 atoms (2 species, n_max 8, l_max 3, P 544), dt 0.5 fs, 500 K"
    if name == "c4":
        return workloads.config4(), "C4 H2/Pt(111) 9 994 400 atoms (2 species, n_max 8, l_max 3, P 544), dt 0.5 fs, 500 K"
    if name in _C5:
        n_max, l_max = _C5[name]
        s = workloads.config5(n_max, l_max)
        return s, f"C5 H2/Pt(111) 1 082 016 atoms (2 species, n_max {n_max}, l_max {l_max}, P {s.P}), dt 0.5 fs, 500 K"
    if name == "tile":
        s = workloads.tile_like_c3(48, 24)
        return s, f"48x24-cell tile of the C3 construction, {s.n_atoms} atoms (P 544)"
    raise SystemExit(f"unknown workload {name}")


# ----------------------------------------------------------------------------- clocks


class ClockSampler:
    """nvidia-smi sampling DURING the timed region (B200_PROFILING.md clocks line)."""

    QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
             "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.QUERY}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            for line in open(self.path):
                p = [x.strip() for x in line.split(",")]
                if len(p) < 9:
                    continue
                try:
                    sm.append(float(p[1])); smax.append(float(p[2])); power.append(float(p[3]))
                except ValueError:
                    continue
                for nme, val in zip(names, p[5:9]):
                    if val.lower().startswith("active"):
                        reasons.add(nme)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(smax)), reasons=sorted(reasons),
                       samples=len(sm), power_w_max=float(max(power)))
        return out


# ----------------------------------------------------------------------------- CPU oracle leg


def oracle_leg(steps: int, warmup: int, budget_s: float = 20.0, threads: int | None = None) -> dict:
    """Time the oracle, as it stands, on a bounded sample of the workload: full E/F/V evaluations
    (neighbour search included) of a periodic 48x24-cell tile of the C3 construction (same slab,
    H2 coverage, basis and P=544 model shape); one evaluation = one step."""
    from oracle import flare_oracle as oracle

    s = workloads.tile_like_c3(48, 24)
    all_cores = oracle.num_threads()
    if threads is not None:
        oracle.set_num_threads(threads)
    cores = oracle.num_threads()
    try:
        for _ in range(max(0, warmup)):
            oracle.compute(s.pos, s.types, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, s.beta, s.sigma)
        t0 = time.perf_counter()
        done = 0
        for _ in range(max(1, steps)):
            oracle.compute(s.pos, s.types, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, s.beta, s.sigma)
            done += 1
            if time.perf_counter() - t0 > budget_s and budget_s > 0:
                break
        dt = time.perf_counter() - t0
    finally:
        if threads is not None:
            oracle.set_num_threads(all_cores)
    return {"value": s.n_atoms * done / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{done} full oracle_compute (E,F,V + neighbour search) of a 48x24-cell periodic tile of the "
                      f"C3 construction ({s.n_atoms} atoms, P=544); gcc -O2 -ffp-contract=off, OpenMP over atoms",
            "seconds": dt, "steps_done": done}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    leg = oracle_leg(args.steps, args.warmup, budget_s=0.0)
    ms = leg["seconds"] / leg["steps_done"] * 1e3
    line = {
        "impl": "reference", "metric": METRIC, "value": leg["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": leg["steps_done"], "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "CPU oracle on a bounded sample of C3 (see cpu_baseline.sample)"},
        "cpu_baseline": {k: leg[k] for k in ("value", "unit", "cores", "kind", "sample")},
        "e2e": {"value": leg["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ----------------------------------------------------------------------------- timing one workload on one GPU


def time_workload(s, args, local: int, steps: int, warmup: int, repeats: int, want_var: bool, barrier=None,
                  sampler=None, analysis: bool = False, **ctx_kw):
    """W warm-up steps, then `repeats` timed regions of exactly `steps` MD steps each (CUDA events on the stream the
    library launches on, a synchronise on both sides).  Returns the context and a dict of measurements."""
    import torch

    from paper_2204_12573_b200 import flare

    dev = torch.device("cuda", local)
    n = s.n_atoms
    ctx = flare.from_system(s, device=local, variance=want_var, timing=True, **ctx_kw)
    ctx.bind(n)
    dt_fs = float(s.meta.get("dt_fs", 0.5))
    pos = torch.as_tensor(s.pos, dtype=torch.float64, device=dev)
    vel = torch.as_tensor(s.vel, dtype=torch.float64, device=dev)
    types = torch.as_tensor(s.types, dtype=torch.int32, device=dev)
    ctx.set_state(pos, vel, types, s.box, s.pbc)
    del pos, vel, types
    ctx.step(dt_fs, 0, want_var)  # initial forces (setup, excluded like the paper's timing protocol P:L213)
    ctx.check()
    for _ in range(warmup):
        ctx.step(dt_fs, 1, want_var)
    ctx.check()
    sync = barrier if barrier is not None else torch.cuda.synchronize
    reps = []
    ana = None
    for rep in range(repeats):
        ctx.timings()  # reset the per-phase accumulators
        launches0 = ctx.kernel_launches()
        rebuilds0 = ctx.get_option(flare.OPT_SKIN_REBUILDS)  # synchronises
        sync()
        if sampler is not None and rep == 0:
            sampler.start()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        if analysis and want_var and s.mass.size > 1:
            for _ in range(steps):
                ctx.step(dt_fs, 1, want_var)
                ana = ctx.analyze(threshold=0.05, species_a=1, species_b=1, r_coord=1.0)  # synchronises
        else:
            ctx.step(dt_fs, steps, want_var)
        ev1.record()
        sync()
        ctx.check()
        reps.append({"ms_total": ev0.elapsed_time(ev1), "launches": ctx.kernel_launches() - launches0,
                     "phases": ctx.timings(), "skin_rebuilds": ctx.get_option(flare.OPT_SKIN_REBUILDS) - rebuilds0})
    order = sorted(range(repeats), key=lambda r: reps[r]["ms_total"])
    med = reps[order[repeats // 2]]
    return ctx, {"ms_per_step": med["ms_total"] / steps, "median": med, "reps": reps, "analysis": ana, "dt_fs": dt_fs}


# ----------------------------------------------------------------------------- rooflines


def group_stats(ctx):
    """Per quadratic-form group: rows, components P_g, compact channels Nc, neighbour pairs sum_i M_i."""
    cnt, _ = ctx.neighbors()
    rows = ctx.rows()
    groups = ctx.groups()
    starts = np.concatenate([[0], np.cumsum([r for r, _ in groups])])
    gid = np.searchsorted(starts, rows, side="right") - 1
    pairs = np.bincount(gid, weights=cnt, minlength=len(groups))
    L = ctx.l_max + 1
    out = []
    for g, (r, p) in enumerate(groups):
        if r == 0:
            continue
        # P_g = Nc (Nc + 1) / 2 * L  ->  Nc
        nc = int(round((-1 + np.sqrt(1 + 8.0 * p / L)) / 2)) if p else 0
        out.append({"rows": int(r), "P": int(p), "Nc": nc, "pairs": float(pairs[g])})
    return out


def qform_traffic(groups, want_var):
    """dram bytes of the k_qform launches of one step, from the tracked ncu --set full capture of the code at HEAD
    (profiles/r02_qform_traffic.csv: one line per captured launch with its rows, K and dram read / write bytes),
    scaled per row to this run's groups.  None when the capture does not cover a group's K."""
    if not os.path.exists(QFORM_TRAFFIC_CSV):
        return None, None
    per_row, commit = {}, None
    with open(QFORM_TRAFFIC_CSV) as fh:
        for rec in csv.DictReader(r for r in fh if not r.startswith("#")):
            if int(rec["variance"]) != int(bool(want_var)):
                continue
            key = int(rec["P"])
            per_row.setdefault(key, []).append((float(rec["dram_read_bytes"]) + float(rec["dram_write_bytes"])) / float(rec["rows"]))
            commit = rec.get("commit", commit)
    tot = 0.0
    for g in groups:
        if g["P"] not in per_row:
            return None, commit
        # the launch with the most rows of that P is the representative one (first line of each P in the file)
        tot += g["rows"] * per_row[g["P"]][0]
    return tot, commit


def kernel_rooflines(ctx, s, res, want_var, peaks, steps):
    """Every phase of the step against its own bound (north_star: ">= 50 % of the FP64/HBM roofline on the dominant
    kernels").  Flop / byte counts per SURVEY.md 8(d), on the groups' compact channels; see DESIGN.md 7."""
    gs = group_stats(ctx)
    n = s.n_atoms
    L = s.l_max + 1
    L2 = L * L
    n_max = s.n_max
    cb = 60 + 8 * n_max + 12 * L2  # per-pair basis cost (rsqrt, cospi / sincospi, Chebyshev and Y_lm recurrences)
    pairs = sum(g["pairs"] for g in gs)
    fl_a2 = sum(g["pairs"] * (cb + 2.0 * n_max * L2) for g in gs)
    fl_a3 = sum(g["rows"] * (L2 * g["Nc"] * (g["Nc"] + 1.0) + 2.0 * g["P"]) for g in gs)
    fl_a6 = sum(g["rows"] * (2.0 * g["Nc"] ** 2 * L2 + 3.0 * g["P"]) for g in gs)
    fl_a7 = sum(g["pairs"] * (cb + 4.0 * n_max * L2 + 8.0 * L2) for g in gs)
    ph = {k: v[0] / steps for k, v in res["median"]["phases"].items()}
    out = []

    def add(kernel, phase, bound, work, unit_work, peak, unit, note):
        ms = ph.get(phase, 0.0)
        ach = work / (ms * 1e-3) / unit_work if ms > 0 else None
        out.append({"kernel": kernel, "phase": phase, "bound": bound, "ms_per_step": ms, "achieved": ach, "peak": peak,
                    "unit": unit, "frac": (ach / peak if (ach and peak) else None), "work_per_step": work, "note": note})

    add("k_descriptor (a2 + a3)", "descriptor", "alu", fl_a2 + fl_a3, 1e12, peaks["dfma"], "TFLOP/s",
        "flops: pairs x (c_b + 2 n_max L^2) + rows x (L^2 Nc (Nc+1) + 2 P_g), c_b = 60 + 8 n_max + 12 L^2")
    add("k_backprop (a6 + pair forces of a7)", "backprop", "alu", fl_a6 + fl_a7, 1e12, peaks["dfma"], "TFLOP/s",
        "flops: rows x (2 Nc^2 L^2 + 3 P_g) + pairs x (c_b + 4 n_max L^2 + 8 L^2)")
    add("k_gather (a7 gather)", "gather", "hbm", pairs * (24 + 24 + 4 + 1) + n * 72.0, 1e9, peaks["hbm"], "GB/s",
        "bytes: per pair own + partner pair force 48, index 4, reverse slot 1; per atom sorted atom 32 + E, V, F out 40")
    add("k_kick_drift + k_kick (a9)", "integrate", "hbm", n * 192.0, 1e9, peaks["hbm"], "GB/s",
        "bytes: SURVEY 8(d) unfused count, 192 B per atom")
    add("neighbour phase (a1: refresh + filter of the candidate list, rebuilds as they fall)", "neighbor", "hbm",
        n * 120.0, 1e9, peaks["hbm"], "GB/s", "bytes: SURVEY 8(d) count, 120 B per atom (the phase is latency-bound)")
    return out, gs


# ----------------------------------------------------------------------------- GPU arm, decomposed (N > 1)


def process_grid(world: int):
    """Near-square px x py factorisation, px >= py (the slab is near-two-dimensional)."""
    py = int(np.floor(np.sqrt(world)))
    while world % py:
        py -= 1
    return world // py, py


def run_decomposed(args):
    """Weak scaling of the real multi-GPU path: one H2/Pt(111) slab px x py times the C3 cell, one C3-sized domain
    per GPU on a 2-D process grid, device data plane (flare_domain_*), one halo exchange per step over
    torch.distributed point-to-point (NCCL).  At N = 1 the rank is its own neighbour on all four sides (self-halo), so
    the same kernels and messages run.  Same JSON line; roofline / cpu_baseline belong to the N = 1 plain run."""
    import torch
    import torch.distributed as dist

    from paper_2204_12573_b200 import flare
    from paper_2204_12573_b200.halo import CudaEngine, DomainDecomposition

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local), timeout=datetime.timedelta(seconds=300))
    torch.cuda.set_device(local)
    want_var = not args.no_variance
    px, py = process_grid(world)
    nx, ny, nh2 = (408, 204, 41616) if args.workload != "tile" else (48, 24, 576)
    s = workloads.h2_pt111_config(3, nx * px, ny * py, nh2 * world, name=f"C3x{px}x{py}")
    ctx = flare.from_system(s, device=local, variance=want_var, timing=True)
    rc_max = float(np.max(s.r_cut))
    halo_skin = 6.0  # domains are ~1000 A wide: a thick ghost shell is cheap (0.4 % more atoms per A) and spaces the rebuilds
    Lx, Ly = float(s.box[0]), float(s.box[4])
    h = 2.0 * rc_max + halo_skin
    shell = (1.0 + 2.0 * h / (Lx / px)) * (1.0 + 2.0 * h / (Ly / py))
    eng = CudaEngine(ctx, capacity=int(1.1 * shell * s.n_atoms / world) + 65536)
    dd = DomainDecomposition(eng, s.box, s.pbc, rc_max, grid=(px, py), halo_skin=halo_skin, self_halo=(world == 1))
    dd.scatter(s.pos, s.vel, s.types)
    dt_fs = float(s.meta.get("dt_fs", 0.5))
    dd.compute(want_var)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    dd.step(dt_fs, args.warmup, want_var)
    reps = []
    sampler = ClockSampler(local)
    for rep in range(args.repeats):
        launches0, sent0, rebuilds0 = ctx.kernel_launches(), dd.bytes_sent, dd.rebuilds
        ctx.timings()
        barrier()
        if rank == 0 and rep == 0:
            sampler.start()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        dd.step(dt_fs, args.steps, want_var)
        ev1.record()
        barrier()
        ms = ev0.elapsed_time(ev1)
        if world > 1:
            t = torch.tensor([ms], dtype=torch.float64, device=torch.device("cuda", local))
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        reps.append({"ms_total": ms, "launches": ctx.kernel_launches() - launches0, "bytes": dd.bytes_sent - sent0,
                     "rebuilds": dd.rebuilds - rebuilds0, "phases": ctx.timings()})
    clocks = sampler.stop() if rank == 0 else {}
    ctx.check()
    order = sorted(range(len(reps)), key=lambda r: reps[r]["ms_total"])
    med = reps[order[len(reps) // 2]]
    if rank == 0:
        line = {
            "metric": METRIC, "value": s.n_atoms * args.steps / (med["ms_total"] * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": med["ms_total"] / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "repeats": len(reps), "repeats_ms_per_step": [r["ms_total"] / args.steps for r in reps],
            "config": {"workload": f"C3 construction tiled {px} x {py}: {s.n_atoms} atoms, one C3-sized domain per GPU on a "
                                   f"{px} x {py} process grid, halo 2 r_cut + {halo_skin} A, device data plane, one exchange per step"
                                   + (" (N = 1: self-halo, the rank is its own neighbour)" if world == 1 else ""),
                       "atoms": s.n_atoms, "P": s.P, "variance": want_var, "dt_fs": dt_fs,
                       "parallelism": f"domain decomposition {px}x{py}",
                       "owned_atoms_rank0": dd.counts["n_owned"], "local_atoms_rank0": dd.counts["n_local"],
                       "halo_bytes_per_rank_per_step": med["bytes"] / max(1, args.steps),
                       "rebuilds_in_window": med["rebuilds"], "candidate_list_rebuilds_total_rank0": ctx.get_option(6),
                       "l2": "working set far larger than L2; no flush needed"},
            "phases_ms_per_step_rank0": {k: v[0] / args.steps for k, v in med["phases"].items()},
            "clocks": clocks, "gpu_launches": med["launches"],
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# ----------------------------------------------------------------------------- GPU arm


def sweep_entries(args, local, peaks, t_start):
    """Configs 1, 2, 4 and the six runs of config 5 with short step counts, so that the driver's record holds them."""
    import torch

    out = []
    # (workload, variance, steps, warm-up, FLARE_OPT_GRAPH): configs 1 and 2 replayed from the captured step (the
    # default for small systems) and, for the per-phase kernel timeline, on plain launches
    plan = [("c1", True, 400, 20, None), ("c1", True, 200, 20, 0), ("c2", True, 200, 20, None), ("c2", True, 100, 20, 0)]
    if args.sweep == "full":
        # enough timed steps that the window holds the candidate-list rebuilds a production run pays for (one per
        # ~10 steps at 500 K, dt 0.5 fs; `skin_rebuilds_in_window` says how many fell in)
        plan += [("c5a", True, 20, 3, None), ("c5a", False, 20, 3, None), ("c5b", True, 20, 3, None),
                 ("c5b", False, 20, 3, None), ("c5c", True, 12, 3, None), ("c5c", False, 12, 3, None), ("c4", True, 12, 3, None)]
    cache = {}
    for name, var, steps, warm, graph in plan:
        if time.perf_counter() - t_start > args.sweep_budget:
            out.append({"workload": name, "variance": var, "skipped": f"sweep time budget of {args.sweep_budget:.0f} s used up"})
            continue
        try:
            if name in _C5 and "c5geo" in cache:  # the three descriptor sizes share one geometry (same seeds)
                n_max, l_max = _C5[name]
                g = cache["c5geo"]
                st = workloads.streams(5)
                s = workloads.System(f"C5_n{n_max}_l{l_max}", g.pos, g.types, g.box, g.pbc, g.mass, g.r_cut, n_max, l_max,
                                     vel=g.vel, meta=dict(g.meta))
                if (name,) in cache:
                    s.beta, s.sigma = cache[(name,)]
                else:
                    s.beta = workloads.random_beta(st["beta"], 2, s.P)
                    s.sigma = workloads.random_sigma(st["sigma"], 2, s.P)
                    cache[(name,)] = (s.beta, s.sigma)
                desc = f"C5 H2/Pt(111) 1 082 016 atoms (n_max {n_max}, l_max {l_max}, P {s.P})"
            else:
                s, desc = make_system(name)
                if name in _C5:
                    cache["c5geo"] = s
                    cache[(name,)] = (s.beta, s.sigma)
            ctx, res = time_workload(s, args, local, steps, warm, 1, var, graph=graph)
            med = res["median"]
            ph = {k: v[0] / steps for k, v in med["phases"].items()}
            flops = ctx.qform_flops(var)
            entry = {"workload": desc, "name": name, "atoms": s.n_atoms, "P": s.P, "variance": var, "steps": steps,
                     "warmup": warm, "ms_per_step": res["ms_per_step"], "value": s.n_atoms / (res["ms_per_step"] * 1e-3),
                     "unit": UNIT, "launches_per_step": med["launches"] / steps,
                     "graph_replay": bool(ctx.get_option(8) > 0),
                     "phases_ms_per_step": ph if any(ph.values()) else None,  # replayed steps record no phase events
                     "skin_rebuilds_in_window": med["skin_rebuilds"],
                     "qform_frac_algorithmic": (flops / (ph["qform"] * 1e-3) * 1e-12 / peaks["dmma"]) if ph["qform"] > 0 else None,
                     "qform_flop_count": "executed: beta dense + upper triangle of Sigma; algorithmic: SURVEY 8(d), 2 P_g^2 per atom and form",
                     "qform_frac_executed": (ctx.qform_flops(var, symmetric=True) / (ph["qform"] * 1e-3) * 1e-12 / peaks["dmma"])
                     if ph["qform"] > 0 else None,
                     "chunk_atoms": ctx.get_option(2), "workspace_bytes_per_atom": ctx.workspace_bytes(s.n_atoms) / s.n_atoms}
            if name in ("c1", "c2"):
                entry["us_per_step"] = res["ms_per_step"] * 1e3
            if any(ph.values()) and (name in _C5 or name == "c4"):
                # the same per-kernel fractions as the headline's roofline_kernels: config 5 is the one meant to show
                # the shift from the ALU kernels to the quadratic forms as P grows
                kr, _ = kernel_rooflines(ctx, s, res, var, peaks, steps)
                entry["roofline_kernels"] = [{"kernel": k["kernel"], "bound": k["bound"], "ms_per_step": k["ms_per_step"],
                                              "achieved": k["achieved"], "peak": k["peak"], "unit": k["unit"],
                                              "frac": k["frac"]} for k in kr]
            out.append(entry)
            ctx.close()
            del ctx
            torch.cuda.empty_cache()
        except Exception as exc:  # a failed sweep entry must not take the headline down with it
            out.append({"workload": name, "variance": var, "error": repr(exc)[:300]})
    return out


def run_ours(args):
    import torch

    from paper_2204_12573_b200 import flare, probes

    t_start = time.perf_counter()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local), timeout=datetime.timedelta(seconds=300))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)

    s, desc = make_system(args.workload)
    want_var = not args.no_variance
    n = s.n_atoms

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local) if rank == 0 else None
    ctx, res = time_workload(s, args, local, args.steps, args.warmup, args.repeats, want_var, barrier=barrier,
                             sampler=sampler, analysis=args.analysis,
                             chunk_atoms=args.chunk if args.chunk else None,
                             species_sparse=False if args.dense else None, skin=args.skin,
                             max_neighbors=args.max_neighbors, graph=args.graph)
    clocks = sampler.stop() if rank == 0 else {}
    dt_fs = res["dt_fs"]
    med = res["median"]
    ms_total = med["ms_total"]
    if dist is not None:
        t = torch.tensor([ms_total], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    ms_per_step = ms_total / args.steps
    value = world * n * args.steps / (ms_total * 1e-3)
    phases = med["phases"]

    # ---- end to end through the host-buffer entry points: per step H2D of the state from pinned
    # memory, one MD step, D2H of the new state and the per-atom results
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    hpos = torch.as_tensor(s.pos, dtype=torch.float64).pin_memory()
    hvel = torch.as_tensor(s.vel, dtype=torch.float64).pin_memory()
    htyp = torch.as_tensor(s.types, dtype=torch.int32).pin_memory()
    out = dict(pos=hpos.numpy(), vel=hvel.numpy(), E=torch.empty(n, dtype=torch.float64).pin_memory().numpy(),
               F=torch.empty((n, 3), dtype=torch.float64).pin_memory().numpy(),
               V=torch.empty(n, dtype=torch.float64).pin_memory().numpy() if want_var else None)

    def e2e_step():
        ctx.set_state(hpos.numpy(), hvel.numpy(), htyp.numpy(), s.box, s.pbc)
        ctx.set_forces(out["F"])  # the forces of that state, read back by the previous step
        ctx.step(dt_fs, 1, want_var)
        ctx.get_state_host(variances=want_var, out=out)  # synchronises

    ctx.set_state(hpos.numpy(), hvel.numpy(), htyp.numpy(), s.box, s.pbc)
    ctx.step(dt_fs, 0, want_var)
    ctx.get_state_host(variances=want_var, out=out)  # forces of the initial state (setup, untimed)
    e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    barrier()
    e2e_s = time.perf_counter() - t0
    if dist is not None:
        t = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    h2d = n * (24 + 24 + 4 + 24)  # positions, velocities, types, forces
    d2h = n * (24 + 24 + 8 + 24 + (8 if want_var else 0))
    e2e_value = world * n * e2e_steps / e2e_s

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline denominators: FP64 peaks measured live by the bench hooks (MEASURED_PEAKS.json has no FP64 entry);
    # HBM from MEASURED_PEAKS.json (driver-written), else the profiling guide's fallback
    peaks = {"dmma": probes.fp64_dmma_tflops(local), "dfma": probes.fp64_dfma_tflops(local), "hbm": 6650.0,
             "hbm_source": "fallback 6.65 TB/s (B200_PROFILING.md)"}
    peaks_file = os.path.join(ROOT, "MEASURED_PEAKS.json")
    derived = None
    if os.path.exists(peaks_file):
        mp = json.load(open(peaks_file))
        if mp.get("hbm_gbs"):
            peaks["hbm"] = float(mp["hbm_gbs"])
            peaks["hbm_source"] = "MEASURED_PEAKS.json hbm_gbs (measured copy)"
        # guide's rule: another dtype's measured peak x nominal ratio (FP64 45 TF : bf16 2250 TF nominal)
        derived = mp.get("bf16_tflops_sustained", 0.0) * 45.0 / 2250.0
    peaks["hbm_copy_probe_gbs"] = probes.hbm_copy_gbs(local, 1 << 30)

    # ---- roofline of the dominant kernel: the quadratic-form DMMA GEMM
    P = s.P
    sparse = bool(ctx.get_option(flare.OPT_SPECIES_SPARSE))
    kernels, gstats = kernel_rooflines(ctx, s, res, want_var, peaks, args.steps)
    flops_per_step = ctx.qform_flops(want_var)  # sum over atoms of 2 P_g^2 per form
    flops_exec = ctx.qform_flops(want_var, symmetric=True)
    # a4 reads B 8 P_g and writes c (here: W) 8 P_g + E 8; a5 shares the B tile and writes V 8
    qf_bytes_per_step = float(sum(g["rows"] * (16.0 * g["P"] + (16 if want_var else 8)) for g in gstats))
    qf_ms, qf_launches = phases["qform"]
    qf_ms_per_step = qf_ms / args.steps
    achieved = flops_per_step / (qf_ms_per_step * 1e-3) * 1e-12 if qf_ms_per_step > 0 else 0.0
    peak = peaks["dmma"]
    ach_exec = flops_exec / (qf_ms_per_step * 1e-3) * 1e-12 if qf_ms_per_step > 0 else 0.0
    traffic, traffic_commit = qform_traffic(gstats, want_var)
    roofline = {
        "bound": "tensor", "kernel": "k_qform_res / k_qform (FP64 DMMA grouped GEMM, beta + Sigma forms)",
        # headline = the flops the tensor pipe EXECUTES: all of W = beta d, but only the blocks of the symmetric
        # Sigma on and above the diagonal.  The paper-level count of SURVEY 8(d) (2 P_g^2 per atom and form, dense) is kept
        # beside it: by that count the kernel can read above the peak, because the symmetry halves the work of the second form.
        "achieved": ach_exec, "peak": peak, "unit": "TFLOP/s", "frac": ach_exec / peak if peak > 0 else None,
        "flop_count": "flops executed on the DMMA pipe: 2 P_g^2 for beta + 512 per 16 x 16 block of the upper triangle of Sigma, "
                      "per atom, on the groups actually evaluated",
        "flops_per_launch_set": flops_exec,
        "achieved_algorithmic": achieved, "frac_algorithmic": achieved / peak if peak > 0 else None,
        "flops_algorithmic": flops_per_step,
        "algorithmic_note": "SURVEY 8(d) count, 2 P_g^2 per atom and per form (dense); may exceed 1 since Sigma's symmetry is used",
        "traffic": traffic,
        "traffic_source": (f"dram__bytes_read.sum + dram__bytes_write.sum per row of the k_qform launches in "
                           f"profiles/r02_qform_traffic.csv (ncu --set full, commit {traffic_commit}), scaled to this step's rows"
                           if traffic is not None else None),
        "algorithmic_bytes": qf_bytes_per_step,
        "traffic_over_algorithmic": (traffic / qf_bytes_per_step if traffic else None),
        "groups": gstats,
        "peak_source": "FP64 DMMA issue peak measured live by the bench hook flare_probe_fp64_dmma_tflops "
                       "(MEASURED_PEAKS.json has no FP64 entry" +
                       (f"; its sustained bf16 x nominal 45/2250 gives {derived:.1f} TFLOP/s)" if derived else ")"),
        "ms_per_step": qf_ms_per_step, "launches_per_step": qf_launches / args.steps,
        "share_of_step": qf_ms_per_step / ms_per_step,
    }
    cpu = None
    if not args.no_cpu_baseline and world == 1:
        cpu = oracle_leg(3, 1, budget_s=15.0)
        one = oracle_leg(1, 0, budget_s=12.0, threads=1)
        cpu["one_thread"] = {"value": one["value"], "unit": UNIT, "cores": one["cores"], "sample": one["sample"]}
    sweep = sweep_entries(args, local, peaks, t_start) if (args.sweep != "none" and world == 1) else None
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "repeats": args.repeats, "repeats_ms_per_step": [r["ms_total"] / args.steps for r in res["reps"]],
        "config": {"workload": desc, "atoms": n, "P": P, "variance": want_var, "dt_fs": dt_fs,
                   "species_sparse": sparse, "skin_angstrom": 1e-3 * ctx.get_option(flare.OPT_SKIN),
                   "skin_rebuilds_in_window": med["skin_rebuilds"],
                   "skin_rebuilds_per_repeat": [r["skin_rebuilds"] for r in res["reps"]],
                   "max_neighbors": ctx.get_option(flare.OPT_MAX_NEIGHBORS),
                   "chunk_atoms": ctx.get_option(flare.OPT_CHUNK_ATOMS),
                   "workspace_bytes_per_atom": ctx.workspace_bytes(n) / n,
                   "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "analysis_every_step": ({"max_uncertainty": res["analysis"]["max_unc"], "n_above_0.05": res["analysis"]["n_above"],
                                            "h_coordination_hist": [int(x) for x in res["analysis"]["hist"][:4]]}
                                           if res["analysis"] else None),
                   "l2": "working set (>10 GB of descriptors per step) is far larger than the 126 MB L2; no flush needed"},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": e2e_steps, "note": "per step: flare_set_state_host + flare_set_forces_host (pinned host -> device), "
                "flare_step(1), flare_get_state_host (x, v, E, F, V device -> pinned host), host wall clock"},
        "gpu_launches": med["launches"],
        "roofline": roofline,
        "roofline_kernels": kernels,
        "peaks": peaks,
        "phases_ms_per_step": {k: v[0] / args.steps for k, v in phases.items()},
        "cpu_baseline": ({k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample", "one_thread")} if cpu else None),
        "sweep": sweep,
        "paper_context": "10.5 M atom-steps/s per Summit node of 6 V100 (P:L225), another machine and model: context only",
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--repeats", type=int, default=3, help="timed regions of --steps steps each; the median is reported")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c3")
    ap.add_argument("--chunk", type=int, default=0)
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--no-variance", action="store_true")
    ap.add_argument("--dense", action="store_true", help="switch the species-sparse evaluation (P:L155) off")
    ap.add_argument("--max-neighbors", type=int, default=None, help="row stride of the neighbour table (library default 48)")
    ap.add_argument("--skin", type=float, default=None, help="skin of the candidate neighbour list in Angstrom (0 = off)")
    ap.add_argument("--graph", type=int, default=None, help="FLARE_OPT_GRAPH: 0 = never capture a CUDA graph, 1 = always, default = automatic")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", default="full", choices=["none", "small", "full"],
                    help="also time configs 1, 2 (small) and 4, 5 (full) with short step counts into the `sweep` array")
    ap.add_argument("--sweep-budget", type=float, default=420.0, help="seconds after which remaining sweep entries are skipped")
    ap.add_argument("--analysis", action="store_true",
                    help="also run flare_analyze (maximum uncertainty + H-H coordination within 1 A) after every step "
                         "inside the timed region, like the paper's production run (P:L247-249)")
    ap.add_argument("--decomposed", action="store_true",
                    help="run the multi-GPU path (2-D domain decomposition + halo exchange through the device data plane, "
                         "paper_2204_12573_b200/halo.py): the default for N > 1; at N = 1 the rank is its own neighbour")
    ap.add_argument("--replicas", action="store_true", help="N > 1: N independent replicas of the workload instead")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    args.repeats = max(1, args.repeats)
    if args.impl == "reference":
        run_reference(args)
    elif args.decomposed or (int(os.environ.get("WORLD_SIZE", "1")) > 1 and not args.replicas):
        run_decomposed(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
