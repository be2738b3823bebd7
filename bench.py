#!/usr/bin/env python
"""bench.py -- atom-steps/s of the FLARE B2 hot path on B200 (BASELINE.json metric).

A "step" is one velocity-Verlet MD step = one pass of the whole hot path (neighbour build,
descriptors, beta + Sigma quadratic forms, back-propagated forces, gather, integrator) over the
synthetic H2/Pt(111)-shaped system.  Default workload: config 3
(1 082 016 atoms, n_max 8, l_max 3, P 544, variance on, dt 0.5 fs) -- the linear-scaling regime
the paper's metric is quoted in; it fits one GPU.

    python bench.py --gpus N --steps K --warmup W [--workload c1|c2|c3|c4|c5a|c5b|c5c|tile]
    python bench.py --impl reference ...   # the CPU oracle, as it stands, on a bounded sample

For N > 1 (launched by torch.distributed.run) every rank runs an independent replica of the
workload ("replicas only": the path has no cross-GPU exchange until the halo decomposition of
DESIGN.md section 9 exists); value = all ranks' atom-steps / max-over-ranks device time.
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
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


def make_system(name: str):
    if name == "c1":
        return workloads.config1(), "C1 fcc Pt 256 atoms (n_max 8, l_max 3, P 144), dt 1 fs, 300 K"
    if name == "c2":
        return workloads.config2(), "C2 H2/Pt(111) 1264 atoms (2 species, n_max 8, l_max 3, P 544), dt 0.5 fs, 500 K"
    if name == "c3":
        return workloads.config3(), "C3 H2/Pt(111) 1 082 016 atoms (2 species, n_max 8, l_max 3, P 544), dt 0.5 fs, 500 K"
    if name == "c4":
        return workloads.config4(), "C4 H2/Pt(111) 9 994 400 atoms (2 species, n_max 8, l_max 3, P 544), dt 0.5 fs, 500 K"
    if name in ("c5a", "c5b", "c5c"):
        n_max, l_max = {"c5a": (8, 3), "c5b": (10, 4), "c5c": (12, 6)}[name]
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


def oracle_leg(steps: int, warmup: int, budget_s: float = 20.0) -> dict:
    """Time the oracle, as it stands, on a bounded sample of the workload: full E/F/V evaluations
    (neighbour search included) of a periodic 48x24-cell tile of the C3 construction (same slab,
    H2 coverage, basis and P=544 model shape); one evaluation = one step."""
    from oracle import flare_oracle as oracle

    s = workloads.tile_like_c3(48, 24)
    cores = oracle.num_threads()
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


# ----------------------------------------------------------------------------- GPU arm, decomposed (opt-in)


def run_decomposed(args):
    """Weak scaling of the real multi-GPU path: one H2/Pt(111) slab `world` times as long as C3 along x, cut into
    `world` slabs, halo exchange every step (NCCL point-to-point).  Same JSON line; roofline / cpu_baseline omitted."""
    import torch
    import torch.distributed as dist

    from paper_2204_12573_b200 import flare
    from paper_2204_12573_b200.halo import CudaEngine, SlabDecomposition

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    want_var = not args.no_variance
    s = workloads.h2_pt111_config(3, 408 * world, 204, 41616 * world, name=f"C3x{world}")
    ctx = flare.from_system(s, device=local, variance=want_var)
    eng = CudaEngine(ctx, capacity=int(1.2 * s.n_atoms / world) + 4096)
    dd = SlabDecomposition(eng, s.box, s.pbc, float(np.max(s.r_cut)), axis=0).scatter(s.pos, s.vel, s.types)
    dt_fs = float(s.meta.get("dt_fs", 0.5))
    dd.compute(want_var)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    dd.step(dt_fs, args.warmup, want_var)
    launches0 = ctx.kernel_launches()
    sent0 = dd.bytes_sent
    sampler = ClockSampler(local)
    barrier()
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    dd.step(dt_fs, args.steps, want_var)
    ev1.record()
    barrier()
    clocks = sampler.stop() if rank == 0 else {}
    ms_total = ev0.elapsed_time(ev1)
    if world > 1:
        t = torch.tensor([ms_total], dtype=torch.float64, device=torch.device("cuda", local))
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    if rank == 0:
        line = {
            "metric": METRIC, "value": s.n_atoms * args.steps / (ms_total * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"C3 construction {world}x as long along x: {s.n_atoms} atoms on {world} slab(s), "
                                   "halo 2 r_cut, one exchange + one migration per step", "atoms": s.n_atoms, "P": s.P,
                       "variance": want_var, "dt_fs": dt_fs, "parallelism": f"slab decomposition x{world}",
                       "halo_bytes_per_rank_per_step": (dd.bytes_sent - sent0) / max(1, args.steps),
                       "l2": "working set far larger than L2; no flush needed"},
            "clocks": clocks, "gpu_launches": ctx.kernel_launches() - launches0,
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# ----------------------------------------------------------------------------- GPU arm


def run_ours(args):
    import torch

    from paper_2204_12573_b200 import flare

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)

    s, desc = make_system(args.workload)
    want_var = not args.no_variance
    n = s.n_atoms
    ctx = flare.from_system(s, device=local, variance=want_var, timing=True,
                            chunk_atoms=args.chunk if args.chunk else None,
                            species_sparse=False if args.dense else None, skin=args.skin,
                            max_neighbors=args.max_neighbors)
    ctx.bind(n)
    dt_fs = float(s.meta.get("dt_fs", 0.5))
    pos = torch.as_tensor(s.pos, dtype=torch.float64, device=dev)
    vel = torch.as_tensor(s.vel, dtype=torch.float64, device=dev)
    types = torch.as_tensor(s.types, dtype=torch.int32, device=dev)
    ctx.set_state(pos, vel, types, s.box, s.pbc)
    ctx.step(dt_fs, 0, want_var)  # initial forces (setup, excluded like the paper's timing protocol P:L213)
    ctx.check()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: W warm-up steps, then exactly K timed steps
    for _ in range(args.warmup):
        ctx.step(dt_fs, 1, want_var)
    ctx.check()
    ctx.timings()  # reset the per-phase accumulators
    launches0 = ctx.kernel_launches()
    sampler = ClockSampler(local)
    barrier()
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    analysis = None
    if args.analysis and want_var and s.mass.size > 1:
        for _ in range(args.steps):
            ctx.step(dt_fs, 1, want_var)
            analysis = ctx.analyze(threshold=0.05, species_a=1, species_b=1, r_coord=1.0)  # synchronises
    else:
        ctx.step(dt_fs, args.steps, want_var)
    ev1.record()
    barrier()
    clocks = sampler.stop() if rank == 0 else {}
    ctx.check()
    ms_total = ev0.elapsed_time(ev1)
    launches = ctx.kernel_launches() - launches0
    phases = ctx.timings()
    if dist is not None:
        t = torch.tensor([ms_total], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    ms_per_step = ms_total / args.steps
    value = world * n * args.steps / (ms_total * 1e-3)

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

    # ---- roofline of the dominant kernel: the quadratic-form DMMA GEMM
    P = s.P
    sparse = bool(ctx.get_option(flare.OPT_SPECIES_SPARSE))
    groups = [g for g in ctx.groups() if g[0] > 0]
    flops_per_step = ctx.qform_flops(want_var)  # sum over atoms of 2 P_g^2 per form
    qf_bytes_per_step = float(sum(r * 8.0 * p * (2 if want_var else 1) + r * 8.0 * p for r, p in groups))
    qf_ms, qf_launches = phases["qform"]
    qf_ms_per_step = qf_ms / args.steps
    achieved = flops_per_step / (qf_ms_per_step * 1e-3) * 1e-12 if qf_ms_per_step > 0 else 0.0
    peak = flare.measure_fp64_dmma_peak(local)
    peaks_file = os.path.join(ROOT, "MEASURED_PEAKS.json")
    derived = None
    if os.path.exists(peaks_file):
        mp = json.load(open(peaks_file))
        # guide's rule: another dtype's measured peak x nominal ratio (FP64 45 TF : bf16 2250 TF nominal)
        derived = mp.get("bf16_tflops_sustained", 0.0) * 45.0 / 2250.0
    roofline = {
        "bound": "tensor", "kernel": "k_qform (FP64 DMMA grouped GEMM, beta + Sigma forms)",
        "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak if peak > 0 else None,
        # dram__bytes_read+write of k_qform per row, from the ncu --set full capture in profiles/r01f_c3.md
        # (3 290 B per K=144 row, 5 860 B per K=544 row, variance on), scaled to one step's rows
        "traffic": (float(sum(r * {144: 3290.0, 544: 5860.0}[p] for r, p in groups))
                    if want_var and all(p in (144, 544) for _, p in groups) else None),
        "algorithmic_bytes": qf_bytes_per_step,
        "groups_rows_x_components": groups,
        "peak_source": "FP64 DMMA issue peak measured live by flare_measure_fp64_dmma_peak "
                       "(MEASURED_PEAKS.json has no FP64 entry; its sustained bf16 x nominal 45/2250 gives "
                       f"{derived:.1f} TFLOP/s)" if derived else "FP64 DMMA issue peak measured live",
        "flops_per_launch_set": flops_per_step, "ms_per_step": qf_ms_per_step,
        # the variance tiles skip the blocks of the symmetric Sigma below the diagonal: flops the kernel really needs
        "flops_needed_with_symmetry": ctx.qform_flops(want_var, symmetric=True),
        "frac_of_needed_flops": (ctx.qform_flops(want_var, symmetric=True) / (qf_ms_per_step * 1e-3) * 1e-12 / peak
                                 if qf_ms_per_step > 0 and peak > 0 else None),
        "launches_per_step": qf_launches / args.steps,
        "share_of_step": qf_ms_per_step / ms_per_step,
    }
    cpu = oracle_leg(3, 1, budget_s=25.0) if not args.no_cpu_baseline else None
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": desc, "atoms": n, "P": P, "variance": want_var, "dt_fs": dt_fs,
                   "species_sparse": sparse, "skin_angstrom": 1e-3 * ctx.get_option(flare.OPT_SKIN),
                   "max_neighbors": ctx.get_option(flare.OPT_MAX_NEIGHBORS),
                   "chunk_atoms": ctx.get_option(flare.OPT_CHUNK_ATOMS),
                   "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "analysis_every_step": ({"max_uncertainty": analysis["max_unc"], "n_above_0.05": analysis["n_above"],
                                            "h_coordination_hist": [int(x) for x in analysis["hist"][:4]]}
                                           if analysis else None),
                   "l2": "working set (>10 GB of descriptors per step) is far larger than the 126 MB L2; no flush needed"},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": e2e_steps, "note": "per step: flare_set_state_host + flare_set_forces_host (pinned host -> device), "
                "flare_step(1), flare_get_state_host (x, v, E, F, V device -> pinned host), host wall clock"},
        "gpu_launches": launches,
        "roofline": roofline,
        "phases_ms_per_step": {k: v[0] / args.steps for k, v in phases.items()},
        "cpu_baseline": {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample")} if cpu else None,
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
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c3")
    ap.add_argument("--chunk", type=int, default=0)
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--no-variance", action="store_true")
    ap.add_argument("--dense", action="store_true", help="switch the species-sparse evaluation (P:L155) off")
    ap.add_argument("--max-neighbors", type=int, default=None, help="row stride of the neighbour table (library default 48)")
    ap.add_argument("--skin", type=float, default=None, help="skin of the candidate neighbour list in Angstrom (0 = off)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--analysis", action="store_true",
                    help="also run flare_analyze (maximum uncertainty + H-H coordination within 1 A) after every step "
                         "inside the timed region, like the paper's production run (P:L247-249)")
    ap.add_argument("--decomposed", action="store_true",
                    help="N ranks share ONE system N times as long as C3 (slab decomposition + halo exchange, "
                         "paper_2204_12573_b200/halo.py) instead of running N replicas")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    elif args.decomposed:
        run_decomposed(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
