#!/usr/bin/env python
"""bench.py -- throughput of the full MPM particle-grid step (Algorithm 1 of arXiv 2404.17057) on B200.

    python bench.py --gpus N --steps K --warmup W [--workload sedov|clumps|cylinder|box|sod] [--size n]
    python bench.py --impl reference ...      # the CPU oracle, as it stands, on the host cores (bounded sample)

One "step" = one pass of the whole hot path (P2G#1, node update + BC, G2P + P2G#2, BC, G2PD + particle update +
advection + re-ordering, CFL) over all particles.  Metric: particle-steps/s (BASELINE.json).  Default workload:
config 4 of BASELINE.json (3D Sedov blast, 256^3 cells, 8 particles/cell, 134 M particles), the largest
single-GPU configuration and one of the two the >= 50 %-of-roofline target is quoted on.  Inputs are seeded and
synthetic (paper_2404_17057_b200/inputs.py).  N > 1: independent replicas, one per GPU (the path has no exchange step
on one GPU), weak scaling, no data-path collective.

Prints ONE JSON line (rank 0).  Timing: CUDA events on the solver's stream around mpm_step(K) with no host sync
inside, barrier + synchronize on both sides, max over ranks.  The particle state (> 10 GB at the default size) is
far larger than the 126 MB L2, so no L2 flush is needed between steps.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2404_17057_b200 import inputs  # noqa: E402

METRIC = "particle-steps/sec (full P2G+grid+G2P step)"
UNIT = "particle-steps/s"


def make_workload(name, size, rank=0):
    """The BASELINE.json configs; `size` overrides the grid resolution (parity / sample sizes)."""
    if name == "sedov":
        return inputs.sedov(n=size or 256, seed=4004 + rank)
    if name == "clumps":
        n = size or 128
        return inputs.clumps(n=n, num_particles=(1 << 26) * n ** 3 // 128 ** 3, seed=5005 + rank)
    if name == "cylinder":
        nx = size or 2048
        return inputs.cylinder(nx=nx, ny=nx // 2, seed=3003 + rank)
    if name == "box":
        return inputs.periodic_box(n=size or 512, seed=2002 + rank)
    if name == "sod":
        return inputs.sod(nx=size or 256, seed=1001 + rank)
    raise SystemExit(f"unknown workload {name}")


def sample_size(name):
    """Bounded sample of the same workload for the CPU oracle (about 10-30 s of single-core work)."""
    return {"sedov": 96, "clumps": 64, "cylinder": 768, "box": 1024, "sod": 256}[name]


def algorithmic_bytes(dim, n_p, n_n):
    """what one step must move (sorting, reset and keys are not credited)."""
    d = dim
    per_kernel = {
        # sweep (i): read X, V, M, write V'  +  nodes: read m, f / write mv2
        "g2p_p2g2": 8 * ((3 * d + 1) * n_p + (1 + 2 * d) * n_n),
        # sweep (ii): read X, rho, E, Q (+V', M), write X', rho', E', Q'  +  nodes: read m, mv, f, mv2
        "update": 8 * ((3 * d + 7) * n_p + (1 + 3 * d) * n_n),
        # not credited separately by section 8(d) (its reads belong to sweep (ii) in the 2-sweep floor); when this
        # kernel dominates it is reported against its own minimal traffic: read X, V, M, S, write m, mv, f
        "p2g1": 8 * ((2 * d + 2) * n_p + (1 + 2 * d) * n_n),
        "node1": 8 * (1 + 2 * d + 2 * d + 2 * d) * n_n,
        "node2": 8 * (1 + 3 * d) * n_n,
    }
    step = 8 * ((6 * d + 8) * n_p + (3 + 7 * d) * n_n)
    return per_kernel, step


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.path = tempfile.NamedTemporaryFile(prefix="clocks_", suffix=".csv", delete=False).name
        self.proc = None
        self.gpu = gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()
        sm, smax, reasons = [], [], set()
        try:
            for line in open(self.path):
                parts = [p.strip() for p in line.split(",")]
                if len(parts) < 7:
                    continue
                try:
                    sm.append(float(parts[0])); smax.append(float(parts[1]))
                except ValueError:
                    continue
                for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), parts[3:7]):
                    if val.lower().startswith("active"):
                        reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "reasons": sorted(reasons),
                "samples": len(sm)}


def measured_peak_gbs():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def ncu_traffic(kernel, workload_name, variant):
    """dram bytes per launch of the dominant kernel from the committed ncu --set full summary, if there is one."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        table = json.load(open(path))
        return table.get(variant, {}).get(workload_name, {}).get(kernel)
    except Exception:
        return None


def oracle_rate(workload, size, steps, warmup=0):
    """particle-steps/s of the CPU oracle (single thread) on a bounded sample of the workload."""
    from oracle import pyoracle as po
    w = make_workload(workload, size)
    o = po.Oracle(w["cfg"])
    o.load_particles(w["x"], w["v"], w["mass"], w["rho"], w["e"])
    if warmup:
        o.step(0.0, w["cfl"], warmup)
    t0 = time.perf_counter()
    o.step(0.0, w["cfl"], steps)
    dt = time.perf_counter() - t0
    n = w["mass"].shape[0]
    return n * steps / dt, dt, n, w["name"]


def max_over_ranks(value, world, device="cpu"):
    """max of a host float over all ranks (the contract's max-over-ranks timing); works for nccl (cuda) and gloo (cpu)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(n_per_rank, steps, ms_max, world):
    """particle-steps/s of the WHOLE job: every rank advances n_per_rank particles (weak scaling, replicas)."""
    return world * n_per_rank * steps / (ms_max * 1e-3)


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores; each step is one oracle step on a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    size = args.size or sample_size(args.workload)
    rate, dt, n, name = oracle_rate(args.workload, size, args.steps, args.warmup)
    sample = f"{name}: {n} particles x {args.steps} steps (reduced-size instance of the {args.workload} workload)"
    line = {
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": name, "particles": n, "note": "CPU oracle (oracle/mpm_oracle.c), single thread"},
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_decomposed(args):
    """--decompose: ONE problem cut into slabs along the last axis, one (or --slabs) per GPU, halo sum-exchanges and particle
    hand-over over torch.distributed (paper_2404_17057_b200/slab.py) -- strong scaling.  First correct multi-GPU path (it
    re-sorts every slab on every step); the default N > 1 run stays independent replicas."""
    import torch
    import torch.distributed as dist
    from paper_2404_17057_b200 import binding as mpm, slab

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    mpm.load()
    w = make_workload(args.workload, args.size, 0)              # every rank builds the same global problem
    n_p = int(w["mass"].shape[0])
    num_slabs = args.slabs or world
    transport = slab.DistTransport(torch.device("cuda", local)) if world > 1 else slab.LocalTransport()
    dom = slab.SlabDomain(w["cfg"], num_slabs, transport=transport, engine_factory=lambda c, s: slab.CudaSlabEngine(c, device=local))
    dom.load_particles(w["x"], w["v"], w["mass"], w["rho"], w["e"])

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()

    dom.step(w["cfl"], args.warmup)
    sampler = ClockSampler(local)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stream = dom.engines[dom.local[0]].solver.stream
    barrier()
    sampler.start()
    ev0.record(stream)
    dom.step(w["cfl"], args.steps)
    ev1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms = max_over_ranks(ev0.elapsed_time(ev1), world, "cuda")
    launches = sum(int(dom.engines[s].stats().launches) for s in dom.local)
    dim = w["cfg"]["dim"]
    n_n = int(np.prod([n if b[0] == 0 else n + 1 for n, b in zip(w["cfg"]["n"][:dim], w["cfg"]["bc"][:dim])]))
    _, step_bytes = algorithmic_bytes(dim, n_p, n_n)
    peak, _ = measured_peak_gbs()
    gbs = step_bytes * args.steps / (ms * 1e-3) / 1e9
    line = {
        "metric": METRIC, "value": n_p * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w["name"], "particles_total": n_p, "nodes": n_n, "dim": dim, "kernel_family": "tiled",
                   "parallelism": f"slab decomposition, {num_slabs} slabs over {world} GPU(s)",
                   "particles_handed_over_per_step": dom.n_migrated / max(1, args.steps + args.warmup)},
        "clocks": clocks, "gpu_launches": launches,
        "step_roofline": {"bytes_per_step": step_bytes, "achieved_gbs": gbs, "frac_of_measured_peak": gbs / (peak * world),
                          "frac_of_8TBs": gbs / (8000.0 * world)},
    }
    dom.close()
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2404_17057_b200 import binding as mpm

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    mpm.load()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()

    peak, peak_src = measured_peak_gbs()
    variant = {"tiled": mpm.VARIANT_TILED, "atomic": mpm.VARIANT_ATOMIC}[args.variant]
    accum = mpm.ACCUM_FP32 if args.grid_accum == "fp32" else mpm.ACCUM_FP64

    def resident(workload, size, steps, warmup):
        """W warm-up steps, then exactly K steps between CUDA events on the solver's stream (inputs resident in HBM);
        then a separate pass with per-kernel timers.  Returns the solver, the workload and the measurements."""
        w = make_workload(workload, size, rank)
        dim = w["cfg"]["dim"]
        n_p = int(w["mass"].shape[0])
        g = mpm.Solver(w["cfg"], sort_every=1, variant=variant, device=local, grid_accum=accum,
                       particle_stream=mpm.STREAM_BULK if args.stream == "bulk" else mpm.STREAM_CP_ASYNC,
                       p2g_mode=args.p2g_mode, particle_ids=mpm.IDS_NONE if args.particle_ids == "none" else mpm.IDS_TRACK)
        n_n = g.num_nodes
        g.load_particles(w["x"], w["v"], w["mass"], w["rho"], w["e"])
        g.step(0.0, w["cfl"], warmup, sync=False)
        st0 = g.stats()
        sampler = ClockSampler(local)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        sampler.start()
        ev0.record(g.stream)
        g.step(0.0, w["cfl"], steps, sync=False)
        ev1.record(g.stream)
        barrier()
        clocks = sampler.stop()
        ms = max_over_ranks(ev0.elapsed_time(ev1), world, "cuda")
        st = g.stats()
        launches = int(st.launches - st0.launches) - 2          # minus the stats reduction itself
        # fraction of the particles that changed cell per step inside the timed window (they take the scattered-store
        # and whole-warp P2G branches of the update kernel; a quiescent window has almost none)
        movers = (st.n_cell_changes - st0.n_cell_changes) / max(1, steps * n_p) if variant == mpm.VARIANT_TILED else None
        # per-kernel durations: separate pass, so that the timers do not perturb `ms`
        prof_steps = min(steps, 10)
        g.set_profiling(True)
        g.step(0.0, w["cfl"], prof_steps, sync=True)
        stp = g.stats()
        g.set_profiling(False)
        kms = {mpm.KERNEL_NAMES[k]: stp.kernel_ms[k] / prof_steps for k in range(7)}
        per_kernel, step_bytes = algorithmic_bytes(dim, n_p, n_n)
        step_gbs = step_bytes * steps / (ms * 1e-3) / 1e9
        # bytes section 8(d) credits that the TILED kernels do not move: with equal particle masses M is never read
        # (8 B in each sweep), and Q' is consumed by the fused P2G#1 of the next step, so it is neither written nor read
        # back except on the last step of a call (2 x 8 B): 32 B per particle, disclosed, and the fraction without them
        # reported next to the credited one
        elided = 8 * 4 * n_p if variant == mpm.VARIANT_TILED and bool(np.all(w["mass"] == w["mass"][0])) else 0
        step_roofline = {"bytes_per_step": step_bytes, "achieved_gbs": step_gbs, "frac_of_measured_peak": step_gbs / peak,
                         "frac_of_8TBs": step_gbs / 8000.0, "kernel_ms_per_step": kms,
                         "credited_but_not_moved_bytes_per_step": elided,
                         "frac_of_8TBs_without_those": (step_bytes - elided) * steps / (ms * 1e-3) / 8e12}
        return dict(g=g, w=w, dim=dim, n_p=n_p, n_n=n_n, ms=ms, clocks=clocks, launches=launches, movers=movers, kms=kms,
                    per_kernel=per_kernel, step_roofline=step_roofline, not_finite=int(st.n_nonfinite),
                    out_of_cell=int(st.n_out_of_cell))

    r = resident(args.workload, args.size, args.steps, args.warmup)
    g, w, dim, n_p, n_n, ms, kms = r["g"], r["w"], r["dim"], r["n_p"], r["n_n"], r["ms"], r["kms"]
    value = whole_job_rate(n_p, args.steps, ms, world)
    dom = max(("p2g1", "g2p_p2g2", "update", "node1", "node2"), key=lambda k: kms[k])
    achieved = r["per_kernel"][dom] / (kms[dom] * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": ncu_traffic(dom, args.workload, args.variant) if not args.size and args.grid_accum == "fp64" else None, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": r["per_kernel"][dom], "kernel_ms": kms[dom]}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if args.grid_accum == "fp64" else "f64 particles, f32 grid accumulation (separate variant)", "data": "synthetic",
        "config": {"workload": w["name"], "grid_accum": args.grid_accum, "particles_per_gpu": n_p, "nodes": n_n, "dim": dim,
                   "kernel_family": args.variant, "particle_stream": args.stream, "p2g_mode": args.p2g_mode, "parallelism": f"replicas x{world}",
                   "l2": "inputs (%.1f GB particle state) exceed the 126 MB L2; no flush" % (n_p * (2 * dim + 5) * 8 / 1e9),
                   "particle_ids": "tracked" if g.ids_tracked else "none (Algorithm 1 has no ids; read-back in storage order)",
                   "movers_per_step": r["movers"],
                   "window": "steps %d-%d after the load" % (args.warmup + 1, args.warmup + args.steps)},
        "clocks": r["clocks"], "gpu_launches": r["launches"], "roofline": roofline, "step_roofline": r["step_roofline"],
    }

    # ---- end to end through the C ABI with HOST buffers: every step copies the inputs H2D and the result D2H
    if not args.no_e2e:
        names = ("x", "v", "mass", "rho", "e")
        pinned = {k: torch.from_numpy(np.ascontiguousarray(w[k])).pin_memory() for k in names}
        out = {k: torch.empty_like(pinned[k]).pin_memory() for k in names}
        out["q"] = torch.empty_like(pinned["mass"]).pin_memory()
        esteps = max(1, min(args.e2e_steps, args.steps))
        h2d = sum(pinned[k].numel() * 8 for k in names)
        d2h = sum(out[k].numel() * 8 for k in out)
        for _ in range(1):                                                 # one untimed pass (page mapping, allocator)
            g.load_particles(pinned["x"], pinned["v"], pinned["mass"], pinned["rho"], pinned["e"], location=mpm.HOST)
            g.step(0.0, w["cfl"], 1, sync=False)
            g.read_particles(out=out, location=mpm.HOST)
        barrier()
        t0 = time.perf_counter()
        for _ in range(esteps):
            g.load_particles(pinned["x"], pinned["v"], pinned["mass"], pinned["rho"], pinned["e"], location=mpm.HOST)
            g.step(0.0, w["cfl"], 1, sync=False)
            g.read_particles(out=out, location=mpm.HOST)
        barrier()
        e2e_s = time.perf_counter() - t0
        e2e_s = max_over_ranks(e2e_s, world, "cuda")
        line["e2e"] = {"value": whole_job_rate(n_p, esteps, e2e_s * 1e3, world), "unit": UNIT, "h2d_bytes_per_step": h2d,
                       "d2h_bytes_per_step": d2h, "steps": esteps,
                       "note": "each step: mpm_load_particles(pinned host) + mpm_step(1) + mpm_read_particles(pinned host)"}
        del pinned, out
    g.close()
    del g, w, r

    # ---- second timed block: BASELINE.json config 5 (clustered contention stress, ~3 % of the particles change cell per
    # step), so that the record carries the stress configuration next to the (almost quiescent) blast window
    if args.workload == "sedov" and not args.size and not args.no_extra:
        torch.cuda.empty_cache()
        r5 = resident("clumps", 0, args.steps, args.warmup)
        r5["g"].close()
        line["extra"] = {"config5": {
            "workload": r5["w"]["name"], "particles_per_gpu": r5["n_p"], "nodes": r5["n_n"],
            "ms_per_step": r5["ms"] / args.steps, "value": whole_job_rate(r5["n_p"], args.steps, r5["ms"], world), "unit": UNIT,
            "step_roofline": r5["step_roofline"], "clocks": r5["clocks"], "movers_per_step": r5["movers"],
            "gpu_launches": r5["launches"]}}
        del r5

    # ---- the oracle on the host cores, bounded sample (reported baseline, not the target)
    if rank == 0 and not args.no_cpu_baseline:
        size = sample_size(args.workload)
        rate, dt, n, name = oracle_rate(args.workload, size, 3)
        line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"{name}: {n} particles x 3 steps in {dt:.1f} s, single thread, "
                                          f"host has {os.cpu_count()} cores"}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="sedov", choices=["sedov", "clumps", "cylinder", "box", "sod"])
    ap.add_argument("--size", type=int, default=0, help="grid resolution override (0 = BASELINE.json size)")
    ap.add_argument("--variant", default="tiled", choices=["tiled", "atomic"])
    ap.add_argument("--grid-accum", default="fp64", choices=["fp64", "fp32"],
                    help="fp32: the fp32 grid-accumulation variant of config 5 (tiled family), reported separately")
    ap.add_argument("--stream", default="cp_async", choices=["cp_async", "bulk"],
                    help="particle stream of the tile kernels: per-thread cp.async (default) or bulk copies (TMA) + mbarriers")
    ap.add_argument("--p2g-mode", type=int, default=0, choices=[0, 1, 2, 3],
                    help="0 = global reductions (default); bit 0 / bit 1: atomics-free shared-memory accumulation by cell "
                         "colour in the gather / update kernel (include/mpm.h MPM_P2G_*)")
    ap.add_argument("--particle-ids", default="none", choices=["none", "track"],
                    help="none (default): the sweeps carry no persistent particle ids (mpm.h MPM_IDS_NONE; grids with an inflow "
                         "face keep them regardless); track: 4 more bytes read and written per particle and step")
    ap.add_argument("--decompose", action="store_true",
                    help="N > 1 (or --slabs > 1): ONE problem cut into slabs over the GPUs (strong scaling) instead of replicas")
    ap.add_argument("--slabs", type=int, default=0, help="with --decompose: number of slabs (default: one per GPU)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the second timed block (config 5) of the default run")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    elif args.decompose:
        run_decomposed(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
