#!/usr/bin/env python
"""bench.py -- MLUPS / HBM roofline of the fused CLIP step on B200 (contract: see DESIGN.md "Measurement").

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--n 256] [--precision 32|64]

One "step" = one pass of the whole hot path (rows a1-a10 of SURVEY.md 8(a)) over the lattice = one LBM time step.
Workload at N=1: BASELINE.json configs[4] (throughput sweep) at 256^3, fp32, periodic, 20 seeded drops, density
ratio 1000 -- the lattice BASELINE.json's `north_star` quotes its target on.  State is 2.7 GB (>> 126 MB L2), so
no L2 flush is needed between timed steps.  Prints ONE JSON line.
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

B_MIN_WORDS = 84  # f 19R+19W, g 19R+19W, phi 1R+1W, u 3R+3W

def ncu_traffic(kernel, workload, n, precision):
    """roofline.traffic: dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed ncu
    --set full captures (profiles/r02_traffic.csv, written from the .ncu-rep files named there; commands in profiles/r02_traffic.md).
    None when no capture matches this run's kernel / workload / size / precision."""
    import csv
    path = os.path.join(ROOT, "profiles", "r02_traffic.csv")
    if not os.path.exists(path):
        return None
    for row in csv.DictReader(open(path)):
        if (row["kernel"], row["workload"], int(row["n"]), int(row["precision"])) == (kernel, workload, int(n), int(precision)):
            return float(row["dram_read_bytes"]) + float(row["dram_write_bytes"])
    return None


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def rank_seed(rank, base=2505):
    """Every rank runs its own seeded replica of the workload (weak scaling)."""
    return base + int(rank)


def whole_job_mlups(nodes_per_rank, steps, ms, world):
    """Whole-job throughput: lattice updates of ALL ranks / max-over-ranks time."""
    return world * nodes_per_rank * steps / (ms * 1e-3) / 1e6


def reduce_over_ranks(ms, e2e_s, finite, world, device):
    """MAX over ranks of the two timings, AND over ranks of the finite flag (nccl on GPU, gloo in the CPU test)."""
    if world <= 1:
        return float(ms), float(e2e_s), bool(finite)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms, e2e_s], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    fl = torch.tensor([1.0 if finite else 0.0], device=device)
    dist.all_reduce(fl, op=dist.ReduceOp.MIN)
    return float(t[0]), float(t[1]), bool(fl.item() > 0.5)


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index = index
        self.samples = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.samples.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for s in self.samples:
            parts = [x.strip() for x in s.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_baseline(n_sample, steps, warmup, seed=2505):
    """Time the oracle as it stands on the host (single thread) on a bounded sample of the same workload."""
    from oracle.clip_oracle import Oracle
    from paper_2505_12205_b200 import inputs
    case = inputs.sweep_drops(n=n_sample, seed=seed, precision=64)
    o = Oracle.from_case(case)
    o.step(warmup)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    mlups = n_sample ** 3 * steps / dt / 1e6
    return mlups, dt / steps * 1e3, f"configs[4] at {n_sample}^3 (same recipe, seed {seed}), fp64, {warmup} warm-up + {steps} timed steps"


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import clip_oracle
    clip_oracle.build()
    n_sample = 64 if (args.steps + args.warmup) <= 40 else (48 if (args.steps + args.warmup) <= 120 else 32)
    mlups, ms, sample = oracle_baseline(n_sample, args.steps, args.warmup)
    line = {
        "impl": "reference", "metric": "MLUPS", "value": mlups, "unit": "MLUPS", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"BASELINE configs[4] sweep, periodic two-phase, bounded sample {n_sample}^3 of the 256^3 lattice",
                   "l2": "n/a (CPU)"},
        "cpu_baseline": {"value": mlups, "unit": "MLUPS", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": mlups, "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


def run_ours(args):
    import torch
    import torch.distributed as dist
    import __graft_entry__ as g
    g.build()
    from paper_2505_12205_b200 import clip, inputs

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    n = args.n
    prec = args.precision
    dtype = torch.float32 if prec == 32 else torch.float64
    word = 4 if prec == 32 else 8
    # one independent lattice per rank (replicas): seed differs per rank
    if args.workload == "rt":  # BASELINE configs[2]: Rayleigh-Taylor 128 x 512 x 128, walls in y (not the headline workload)
        case = inputs.rayleigh_taylor(L=n // 2, precision=prec)
    elif args.workload == "jet":  # BASELINE configs[3]: liquid jet 192 x 192 x 1536, inlet disc, convective outlet, side walls
        case = inputs.jet(nxy=3 * n // 4, nz=args.nz or 6 * n, r_nozzle=12.0 * n / 256, precision=prec)
    elif args.workload == "jetfs":  # the paper's own jet set-up: free-slip side walls (Sec. 6)
        case = inputs.jet(nxy=3 * n // 4, nz=args.nz or 6 * n, r_nozzle=12.0 * n / 256, precision=prec)
        case["params"]["bc"] = (inputs.FREESLIP,) * 4 + (inputs.INLET, inputs.OUTLET)
    elif args.workload == "d2q9":  # 2-D lattice 16 n x 16 n on D2Q9 (Table 2 :561 times a 256 x 64 D2Q9 case)
        case = inputs.sweep2d(nx=16 * n, ny=16 * n, seed=rank_seed(rank), ndrops=20 * n // 16, rmin=6.0, rmax=20.0, precision=prec)
    else:
        case = inputs.sweep_drops(n=n, seed=rank_seed(rank), precision=prec)
    case["params"]["path"] = args.path
    case["params"]["tile_ty"], case["params"]["tile_chunks"] = args.tile_ty, args.tile_chunks
    case["params"]["cluster_y"] = args.cluster_y
    nxl, nyl, nzl = case["nx"], case["ny"], case["nz"]
    nodes = nxl * nyl * nzl
    # a stream of its own (not the legacy default stream): clip_step can then replay small lattices from a CUDA graph (clip.h)
    sim = clip.Clip(nxl, nyl, nzl, case["params"], device=dev, stream=torch.cuda.Stream(dev))
    phi0_h = torch.as_tensor(case["phi0"]).to(dtype).pin_memory()
    u0_h = torch.as_tensor(case["u0"]).to(dtype).pin_memory()
    sim.init(phi0_h, u0_h)
    torch.cuda.synchronize()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput: W warm-up steps, then exactly K timed steps
    sim.step(args.warmup)
    if nodes <= (1 << 22):
        sim.step(32)   # launch-bound lattices: 32 more untimed steps, in which the handle captures its 16-step CUDA graph
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = sim.launches
    g0 = sim.graph_steps
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(sim.stream)
    sim.step(args.steps)
    e1.record(sim.stream)
    barrier()
    ms = e0.elapsed_time(e1)
    launches = sim.launches - l0
    graph_steps = sim.graph_steps - g0
    clocks = sampler.stop() if rank == 0 else None
    phi, p, u = sim.get()
    sim.stream.synchronize()
    finite = bool(torch.isfinite(phi).all() and torch.isfinite(u).all() and torch.isfinite(p).all())

    # ---- per-kernel durations (CUDA events on the launch stream around every launch)
    prof = sim.step_profiled(args.steps)
    step_ms_prof = sum(v[0] for v in prof.values()) / args.steps
    dom = max(prof, key=lambda k: prof[k][0])

    # ---- end to end through the host-buffer call: H2D(phi0,u0) -> init -> K steps -> get -> D2H(phi,p,u)
    out_phi = torch.empty((nzl, nyl, nxl), dtype=dtype).pin_memory()
    out_p = torch.empty((nzl, nyl, nxl), dtype=dtype).pin_memory()
    out_u = torch.empty((3, nzl, nyl, nxl), dtype=dtype).pin_memory()
    bufs = (torch.empty_like(phi0_h, device=dev), torch.empty_like(u0_h, device=dev), torch.empty_like(out_phi, device=dev),
            torch.empty_like(out_p, device=dev), torch.empty_like(out_u, device=dev))
    clip.run_host(sim, phi0_h, u0_h, 2, out_phi, out_p, out_u, bufs)  # warm-up job
    barrier()
    t0 = time.perf_counter()
    h2d, d2h = clip.run_host(sim, phi0_h, u0_h, args.steps, out_phi, out_p, out_u, bufs)
    barrier()
    e2e_s = time.perf_counter() - t0

    ms, e2e_s, finite = reduce_over_ranks(ms, e2e_s, finite, world, dev)

    if rank == 0:
        peak, peak_src = measured_peak()
        mlups = whole_job_mlups(nodes, args.steps, ms, world)
        e2e_mlups = world * nodes * args.steps / e2e_s / 1e6
        b_min = 42 if args.workload == "d2q9" else B_MIN_WORDS   # D2Q9: f 9R+9W, g 9R+9W, phi 1R+1W, u 2R+2W
        step_bytes = b_min * word * nodes
        achieved = step_bytes / (step_ms_prof * 1e-3) / 1e9
        line = {
            "metric": "MLUPS", "value": mlups, "unit": "MLUPS", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32" if prec == 32 else "f64", "data": "synthetic",
            "config": {"workload": (f"BASELINE configs[2] Rayleigh-Taylor {nxl}x{nyl}x{nzl}, walls in y, fp{prec}" if args.workload == "rt" else
                                    f"BASELINE configs[3] liquid jet {nxl}x{nyl}x{nzl}, inlet disc + convective outlet + side walls, fp{prec}" if args.workload == "jet" else
                                    f"2-D periodic two-phase lattice {nxl}x{nyl} on D2Q9 (PAPER.md:568), seeded discs, rho ratio 1000, fp{prec}; B_min = 42 words/LU" if args.workload == "d2q9" else
                                    f"the paper's jet set-up {nxl}x{nyl}x{nzl}: inlet disc + convective outlet + FREE-SLIP sides (PAPER.md Sec. 6), fp{prec}" if args.workload == "jetfs" else
                                    f"BASELINE configs[4] throughput sweep at {n}^3: periodic two-phase box, 20 seeded drops, "
                                    f"rho ratio 1000, fp{prec} (north_star target lattice)"),
                       "lattice": [nxl, nyl, nzl], "l2": f"state {sim.workspace_bytes / 1e9:.2f} GB >> 126 MB L2, no flush needed",
                       "parallelism": "independent replica per GPU" if world > 1 else "single GPU",
                       "finite_after_run": finite, "steps_replayed_from_cuda_graph": int(graph_steps)},
            "gpu_launches": int(launches),
            "effective_gbs": mlups * 1e6 * b_min * word / 1e9 / world,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": ncu_traffic(dom, args.workload, n, prec) if not args.nz else None, "peak_source": peak_src,
                         "kernel": dom, "algorithmic_bytes_per_step": step_bytes,
                         "note": f"achieved = {b_min} words/LU x nodes / (sum of the step's kernel durations, CUDA events per launch)",
                         "kernels_ms_per_step": {k: v[0] / args.steps for k, v in prof.items()},
                         "frac_of_nominal_8TBs": achieved / 8000.0},
            "e2e": {"value": e2e_mlups, "unit": "MLUPS", "h2d_bytes_per_step": h2d / args.steps,
                    "d2h_bytes_per_step": d2h / args.steps,
                    "job": f"pinned host phi0,u0 -> H2D -> clip_init -> clip_step({args.steps}) -> clip_get -> D2H, wall clock"},
            "clocks": clocks,
        }
        if world == 1 and not args.no_cpu:
            cm, cms, sample = oracle_baseline(64, 20, 2)
            line["cpu_baseline"] = {"value": cm, "unit": "MLUPS", "cores": 1, "kind": "oracle", "sample": sample}
        print(json.dumps(line))
    sim.close()
    if world > 1:
        dist.destroy_process_group()


def run_slab(args):
    """`--decomp slab`: ONE periodic lattice n x n x (n * N) cut into N z slabs, one per GPU (weak scaling: n^3 owned nodes per
    GPU), exchange of one 12-word record per face node and cut side after every step (paper_2505_12205_b200/slab.py).  With N = 1
    the slab is its own neighbour: the line then shows what packing, copying and unpacking the halos costs on one GPU."""
    import torch
    import torch.distributed as dist
    import __graft_entry__ as g
    g.build()
    from paper_2505_12205_b200 import inputs, slab

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    n, prec = args.n, args.precision
    dtype = torch.float32 if prec == 32 else torch.float64
    word = 4 if prec == 32 else 8
    planes = slab.slab_plane_index(n * world, rank, world, True)
    # same recipe and drop density; every rank builds only its own planes (ghosts included) of the global field
    case = inputs.sweep_drops(shape=(n, n, n * world), seed=2505, ndrops=20 * world, precision=prec, z_planes=planes)
    case["params"]["path"] = args.path
    sl = slab.SlabClip(n, n, n * world, case["params"], rank, world, device=dev, overlap=not args.no_overlap)
    assert sl.planes == planes
    phi0_h = torch.as_tensor(case["phi0"]).to(dtype).pin_memory()
    u0_h = torch.as_tensor(case["u0"]).to(dtype).pin_memory()
    del case

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sl.sim.init(phi0_h, u0_h)
    sl.step(args.warmup)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = sl.sim.launches
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(sl.sim.stream)
    sl.step(args.steps)
    e1.record(sl.sim.stream)
    barrier()
    ms = e0.elapsed_time(e1)
    launches = sl.sim.launches - l0
    clocks = sampler.stop() if rank == 0 else None
    phi, p, u = sl.get()
    finite = bool(torch.isfinite(phi).all() and torch.isfinite(u).all() and torch.isfinite(p).all())
    # end to end: pinned host slab -> H2D -> init -> K steps with exchanges -> get -> D2H of the owned planes
    own = sl.z1 - sl.z0
    out = [torch.empty((own, n, n), dtype=dtype).pin_memory(), torch.empty((own, n, n), dtype=dtype).pin_memory(),
           torch.empty((3, own, n, n), dtype=dtype).pin_memory()]
    barrier()
    t0 = time.perf_counter()
    sl.exchanges = 0
    sl.sim.init(phi0_h, u0_h)
    sl.step(args.steps)
    for o, d in zip(out, sl.get()):
        o.copy_(d, non_blocking=True)
    barrier()
    e2e_s = time.perf_counter() - t0
    # per-kernel durations of the slab's own step (CUDA events around every launch; no exchange in between: timing only)
    prof = sl.sim.step_profiled(10)
    kernels_ms = {k: v[0] / 10 for k, v in prof.items() if v[1]}
    ms, e2e_s, finite = reduce_over_ranks(ms, e2e_s, finite, world, dev)
    if rank == 0:
        peak, peak_src = measured_peak()
        nodes = n * n * n
        mlups = whole_job_mlups(nodes, args.steps, ms, world)
        achieved = B_MIN_WORDS * word * nodes / (ms / args.steps * 1e-3) / 1e9
        h2d = (phi0_h.numel() + u0_h.numel()) * word
        d2h = sum(o.numel() for o in out) * word
        print(json.dumps({
            "metric": "MLUPS", "value": mlups, "unit": "MLUPS", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if prec == 32 else "f64", "data": "synthetic",
            "config": {"workload": f"BASELINE configs[4] recipe on ONE periodic lattice {n}x{n}x{n * world} cut into {world} z slab(s), fp{prec}",
                       "lattice": [n, n, n * world], "parallelism": f"z slabs, {slab.HALO} ghost plane per cut, neighbour send/recv of one 12-word record per face node after every step",
                       "halo_bytes_sent_per_rank_per_step": sl.halo_bytes_per_step, "local_planes": sl.nz_local,
                       "l2": f"state {sl.sim.workspace_bytes / 1e9:.2f} GB >> 126 MB L2, no flush needed", "finite_after_run": finite},
            "gpu_launches": int(launches),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                         "peak_source": peak_src, "kernel": "whole step incl. halo pack / exchange / unpack", "kernels_ms_per_step": kernels_ms,
                         "overlap": sl.halo is not None,
                         "note": "achieved = 84 words/LU x OWNED nodes / step time (CUDA events around the timed steps)"},
            "e2e": {"value": world * nodes * args.steps / e2e_s / 1e6, "unit": "MLUPS", "h2d_bytes_per_step": h2d / args.steps,
                    "d2h_bytes_per_step": d2h / args.steps,
                    "job": "pinned host slab -> H2D -> clip_init -> K x (clip_step(1) + halo exchange) -> clip_get -> D2H, wall clock"},
            "clocks": clocks}))
    sl.close()
    if world > 1:
        dist.destroy_process_group()


def run_plumbing(args):
    """`--plumbing-only`: the launch / rendezvous / reduction path of a multi-rank run without any GPU work (CPU test)."""
    import torch
    import torch.distributed as dist
    world, rank = int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0"))
    if world > 1:
        dist.init_process_group("gloo")
    ms, e2e, finite = reduce_over_ranks(1.0 + rank, 2.0 + rank, True, world, torch.device("cpu"))
    if rank == 0:
        decomp = args.decomp or ("slab" if world > 1 else "replicas")
        print(json.dumps({"plumbing_only": True, "n_gpus": world, "gpus_requested": args.gpus, "decomp": decomp, "max_ms": ms, "max_e2e_s": e2e,
                          "finite": finite}))
    if world > 1:
        dist.destroy_process_group()


def run_long(args):
    """`--long-run rt|jet`: BASELINE configs[2] / configs[3] at FULL LENGTH on the GPU (the CPU oracle would need
    days), with the checks the survey lists: finite fields, drift of sum(phi), x <-> z symmetry (RT: the initial condition is
    symmetric under the swap), inflow mass balance d(sum phi)/dt against the nozzle's flux (jet, before the liquid reaches the
    outlet), range of phi, max |u|.  Prints ONE JSON line with the time series; diagnostics are torch reductions on the device
    between clip_step calls (measurement, not the path)."""
    import torch
    import __graft_entry__ as g
    g.build()
    from paper_2505_12205_b200 import clip, inputs
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    prec = args.precision
    if args.long_run == "rt":
        case = inputs.rayleigh_taylor(L=args.n // 2, precision=prec)
        total = args.steps if args.steps_given else 20000
    elif args.long_run == "jetpaper":   # the paper's own set-up (Sec. 6.1, Table 6 row --case): 6 D x 6 D x 20 D, free-slip sides, gravity
        case = inputs.jet_paper(case=args.case, D=args.n // 8, precision=prec, W=args.width, M=args.mobility, U=args.uj)
        total = args.steps if args.steps_given else 40000
    else:
        case = inputs.jet(nxy=3 * args.n // 4, nz=6 * args.n, r_nozzle=12.0 * args.n / 256, We=args.we, precision=prec)
        total = args.steps if args.steps_given else 50000
    every = max(1, total // (200 if args.long_run == "jetpaper" else 50))
    case["params"]["path"] = args.path
    sim = clip.Clip.from_case(case, precision=prec)
    pr = case["params"]
    nx, ny, nz = case["nx"], case["ny"], case["nz"]
    phi0 = torch.as_tensor(case["phi0"]).to(dev)
    s0 = float(phi0.double().sum())
    disc = None
    if args.long_run in ("jet", "jetpaper"):
        yy, xx = torch.meshgrid(torch.arange(ny, dtype=torch.float64), torch.arange(nx, dtype=torch.float64), indexing="ij")
        disc = int((((xx - pr["inlet_c"][0]) ** 2 + (yy - pr["inlet_c"][1]) ** 2) <= pr["inlet_r"] ** 2).sum())
    series, first_bad = [], None
    t0 = time.perf_counter()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    gpu_ms = 0.0
    done = 0
    while done < total:
        n = min(every, total - done)
        e0.record(sim.stream)
        sim.step(n)
        e1.record(sim.stream)
        done += n
        phi, p, u = sim.get()
        torch.cuda.synchronize()
        gpu_ms += e0.elapsed_time(e1)
        finite = bool(torch.isfinite(phi).all() and torch.isfinite(u).all() and torch.isfinite(p).all())
        rec = {"t": done, "finite": finite}
        if finite:
            rec.update(sum_phi=float(phi.double().sum()), phi_min=float(phi.min()), phi_max=float(phi.max()), u_max=float(u.abs().max()))
            if args.long_run == "rt":
                rec["xz_asym"] = float((phi - phi.transpose(0, 2)).abs().max())
                rec["y_front_heavy"] = int((phi[:, :, :] > 0.5).any(dim=2).any(dim=0).nonzero().min())   # lowest row the heavy fluid has reached
            else:
                axis = phi[:, ny // 2, nx // 2] > 0.5
                col = axis.nonzero()
                rec["tip_z"] = int(col.max()) if col.numel() else -1
                gaps = (~axis).nonzero()
                rec["attached_len"] = int(gaps.min()) if gaps.numel() else nz      # length of the liquid column still attached to the nozzle
                rec["outlet_phi_max"] = float(phi[-1].max())
        elif first_bad is None:
            first_bad = done
        series.append(rec)
        if not finite:
            break
    wall = time.perf_counter() - t0
    last = series[-1]
    out = {"long_run": args.long_run, "lattice": [nx, ny, nz], "precision": prec, "steps_requested": total, "steps_done": done,
           "stable": first_bad is None, "first_non_finite_step_at_or_before": first_bad,
           "params": {k: (list(v) if isinstance(v, tuple) else v) for k, v in pr.items()},
           "sum_phi_0": s0, "mlups": nx * ny * nz * done / (gpu_ms * 1e-3) / 1e6, "gpu_ms_per_step": gpu_ms / max(done, 1), "wall_s": wall,
           "series": series}
    if first_bad is None:
        if args.long_run == "rt":
            out["sum_phi_rel_drift"] = (last["sum_phi"] - s0) / s0
            out["xz_asym_max"] = max(r["xz_asym"] for r in series)
        else:
            # inflow mass balance while the liquid is far from the outlet: d(sum phi)/dt against (disc nodes) x U x phi_in
            if args.long_run == "jetpaper":
                # breakup length (Fig. 18c): the attached column grows until a drop pinches off; L_b = its length just
                # before each pinch-off (local maxima of the attached length followed by a drop of more than D / 2)
                D = 2.0 * pr["inlet_r"]
                al = [r["attached_len"] for r in series]
                peaks = [al[k] for k in range(1, len(al) - 1) if al[k] >= al[k - 1] and al[k + 1] < al[k] - 0.5 * D]
                # drop sizes ("equilibrium droplet diameter d_e", Fig. 18c): connected components of phi > 1/2 in the final field
                # that do not touch the inlet plane; d_e = (6 V / pi)^(1/3), V = sum of phi over the component (host side, scipy)
                drops = []
                try:
                    from scipy import ndimage
                    ph = phi.float().cpu().numpy()
                    lab, ncomp = ndimage.label(ph > 0.5)
                    attached = set(lab[0][lab[0] > 0].ravel().tolist())
                    vol = ndimage.sum_labels(ph, lab, index=range(1, ncomp + 1))
                    drops = sorted(((6.0 * float(v) / 3.141592653589793) ** (1.0 / 3.0) / D for k, v in enumerate(vol, start=1) if k not in attached and v > 30.0), reverse=True)
                except Exception as e:  # diagnostics only
                    drops = [f"unavailable: {e}"]
                out["breakup"] = {"D": D, "pinch_offs": len(peaks), "L_b_over_D": [v / D for v in peaks], "detached_drops_d_e_over_D": drops,
                                  "L_b_over_D_mean": (sum(peaks) / len(peaks) / D) if peaks else None, "t_star_end": done * pr["inlet_u"][2] / D,
                                  "case": args.case, "Re_We_Fr": inputs.JET_TABLE6[args.case]}
            pre = [r for r in series if r["outlet_phi_max"] < 0.01]
            if len(pre) >= 2:
                rate = (pre[-1]["sum_phi"] - pre[0]["sum_phi"]) / (pre[-1]["t"] - pre[0]["t"])
                out["inflow"] = {"d_sum_phi_dt": rate, "disc_nodes_x_U": disc * pr["inlet_u"][2] * pr["inlet_phi"],
                                 "pi_R2_U": 3.141592653589793 * pr["inlet_r"] ** 2 * pr["inlet_u"][2], "disc_nodes": disc,
                                 "window": [pre[0]["t"], pre[-1]["t"]]}
    print(json.dumps(out))
    sim.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=256)
    ap.add_argument("--precision", type=int, default=32, choices=[32, 64])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--workload", default="sweep", choices=["sweep", "rt", "jet", "jetfs", "d2q9"],
                    help="sweep = BASELINE configs[4] (headline); rt = configs[2] lattice (n/2 x 2n x n/2), walls in y; jet = configs[3] lattice (3n/4 x 3n/4 x 6n)")
    ap.add_argument("--decomp", default=None, choices=["replicas", "slab"],
                    help="slab (default for N > 1): ONE lattice n x n x (n N) cut into N z slabs with a halo exchange per step -- the path's "
                         "own sharding (SURVEY.md 8(e)); replicas: an independent lattice per GPU.  N = 1 default: the undivided lattice")
    ap.add_argument("--no-overlap", action="store_true", help="slab decomposition: plain sequence step; pack; exchange; unpack on one stream")
    ap.add_argument("--plumbing-only", action="store_true",
                    help="no GPU work: start the ranks, rendezvous (gloo), reduce dummy timings and print the line's skeleton (CPU test of --gpus N)")
    ap.add_argument("--nz", type=int, default=0, help="jet workload only: planes along the jet (default 6 n = 1536; shorter for profiling runs)")
    ap.add_argument("--path", type=int, default=0, choices=[0, 1, 2, 3, 4, 5],
                    help="clip_params.path: 0 automatic (default), 1 generic kernels, 2 pair kernels (k_phi2 + k_step2), 3 k_fused wherever admitted")
    ap.add_argument("--case", default="l", help="--long-run jetpaper: row of the paper's Table 6 (a .. l)")
    ap.add_argument("--tile-ty", type=int, default=0, help="clip_params.tile_ty (k_fused rows per tile: 0 automatic, 4, 8, 16)")
    ap.add_argument("--cluster-y", type=int, default=0, choices=[0, 1, 2, 4, 8], help="clip_params.cluster_y (k_fused: y tiles per thread-block cluster; 0 automatic, 1 none)")
    ap.add_argument("--tile-chunks", type=int, default=0, help="clip_params.tile_chunks (k_fused: number of equal z chunks, 0 automatic)")
    ap.add_argument("--long-run", default=None, choices=["rt", "jet", "jetpaper"],
                    help="run BASELINE configs[2] (rt, 20000 steps) or configs[3] (jet, 50000 steps) at full length with diagnostics; one JSON line")
    ap.add_argument("--width", type=float, default=4.0, help="--long-run jetpaper: interface width W (the paper does not state it for the jets)")
    ap.add_argument("--mobility", type=float, default=0.1, help="--long-run jetpaper: Allen-Cahn mobility M (not stated by the paper either)")
    ap.add_argument("--uj", type=float, default=0.05, help="--long-run jetpaper: inlet velocity in lattice units (the paper: 0.05, PAPER.md:849)")
    ap.add_argument("--we", type=float, default=2.2, help="Weber number of the jet (--long-run jet)")
    args = ap.parse_args()
    args.steps_given = any(a == "--steps" or a.startswith("--steps=") for a in sys.argv[1:])
    if args.long_run:
        return run_long(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N` without a launcher: start the N ranks ourselves (one process per GPU), same command line
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
               "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
        raise SystemExit(subprocess.call(cmd))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.plumbing_only:
        return run_plumbing(args)
    if args.impl == "reference":
        run_reference(args)
    elif args.decomp == "slab" or (args.decomp is None and world > 1):
        run_slab(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
