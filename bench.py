#!/usr/bin/env python
"""bench.py -- Jacobi-PCG on synthetic Poisson-Boltzmann grids: iterations/s, time-to-solution, roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 5] [--precision f32]

A "step" is one complete pb_solve (rows a1-a6 of SURVEY.md section 8(a): init, K_spmv/K_vec iterations with
the on-device convergence latch, un-pad) on one right-hand side.  At N=1 the workload is BASELINE.json
configs[4] (385^3, 60 000 atoms, fp32 to relative residual 1e-5), the configuration the north-star metric is
quoted on.  For N>1 every rank solves its own member of config 5's perturbed-charge batch on its own copy of
the operator (replicas, no data-path collective): weak scaling.  One JSON line is printed by rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "pcg_iterations_per_s"
UNIT = "iterations/s"
# Algorithmic words per node per launch ("tighter variant": z never stored, phi update deferred)
WORDS_SPMV = 10     # r, Dinv, p, x, eps_x, eps_y, eps_z read; p, x, Ap written
WORDS_VEC = 4       # r, Ap, Dinv read; r written
WORDS_NORTH_STAR = 16   # the north-star accounting (8 + 8) the >=70 %-of-peak target is stated in
TOL = {"f32": 1e-5, "f64": 1e-10}
GRID = {1: 33, 2: 65, 3: 129, 4: 257, 5: 385}


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config (1-based); 5 = headline")
    ap.add_argument("--precision", default="f32", choices=["f32", "f64"])
    ap.add_argument("--tol", type=float, default=None)
    ap.add_argument("--check-every", type=int, default=32)
    ap.add_argument("--maxiter", type=int, default=20000)
    ap.add_argument("--profile-iters", type=int, default=40)
    ap.add_argument("--cpu-sample-iters", type=int, default=None)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--setup-from-atoms", action="store_true",
                    help="also time pb_create_from_atoms / pb_set_charges (GPU grid setup, NEXT row f1)")
    ap.add_argument("--batch", type=int, default=None,
                    help="solves of config 5's perturbed-charge batch on the same operator (default: 50 at --gpus 1 "
                         "--config 5, else 0)")
    ap.add_argument("--opt", action="append", default=[], metavar="NAME=VALUE",
                    help="per-handle option for the benchmarked solver (pb_set_option names of the binding), repeatable")
    ap.add_argument("--slab", type=int, default=0, metavar="N",
                    help="instead of replicas: ONE solve cut into z-slabs (NEXT row f4).  Under torchrun one slab per "
                         "rank (NCCL halo exchange + all-reduces, strong scaling); at --gpus 1: N slabs emulated on one GPU")
    ap.add_argument("--no-variants", action="store_true",
                    help="skip the other-precision and no-palette legs of the roofline record")
    ap.add_argument("--cpu-per-config", action="store_true",
                    help="also time the oracle on every smaller config (1 thread too for <= 129^3), BASELINE.md section 3")
    ap.add_argument("--refined", action="store_true",
                    help="also time pb_solve_refined (fp32-inner / fp64-outer, NEXT row f3) against the fp64 solve, to 1e-10")
    return ap.parse_args(argv)


def measured_peak():
    """HBM GB/s denominator: MEASURED_PEAKS.json (driver-written) else the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(workload_key):
    """dram bytes per K_spmv launch from the committed ncu --set full summary (profiles/ncu_traffic.csv), or None."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as f:
            for line in f:
                cols = line.strip().split(",")
                if len(cols) >= 2 and cols[0] == workload_key:
                    return int(cols[1])
    except Exception:
        pass
    return None


class ClockSampler:
    """Samples SM clock and throttle reasons during the timed region (pynvml, 100 ms period)."""

    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, index):
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop = threading.Event()
        self._t = None

    def _run(self):
        try:
            import pynvml

            pynvml.nvmlInit()
            h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM)
            while not self._stop.is_set():
                self.samples.append(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM))
                try:
                    r = pynvml.nvmlDeviceGetCurrentClocksEventReasons(h)
                except Exception:
                    r = pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, name in self.REASONS.items():
                    if r & bit:
                        self.reasons.add(name)
                self._stop.wait(0.1)
        except Exception as e:  # no NVML: report that instead of clocks
            self.reasons.add(f"nvml_unavailable:{type(e).__name__}")

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        self._t.join(timeout=2)

    def summary(self):
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def physical_gpu_index(local_rank):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


def aggregate(local_units, local_ms, world, device=None):
    """Whole-job numbers: sum of the units all ranks processed, max over ranks of the device time."""
    if world == 1:
        return float(local_units), float(local_ms)
    import torch
    import torch.distributed as dist

    dev = device if device is not None else "cpu"
    u = torch.tensor([float(local_units)], dtype=torch.float64, device=dev)
    t = torch.tensor([float(local_ms)], dtype=torch.float64, device=dev)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(u.item()), float(t.item())


def workload_name(cfg, prec, tol):
    n = GRID[cfg]
    return f"config{cfg}_{n}^3_{prec}_tol{tol:g}"


def build_inputs(cfg, rank, world, device):
    """Seeded synthetic inputs (workloads/): the operator of config `cfg`; rank r > 0 (or any rank of a
    multi-GPU run) takes member r of the perturbed-charge batch as its right-hand side."""
    from workloads import make_config, perturbed_charges

    inp = make_config(cfg, device=device)
    rhs, bc = inp.rhs, inp.bc
    if world > 1 and "charges" in inp.meta:
        rhs, bc = perturbed_charges(inp, rank, device=device)
    return inp, np.ascontiguousarray(rhs), np.ascontiguousarray(bc)


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle, as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return None
    from oracle import pbref

    prec = args.precision
    tol = args.tol or TOL[prec]
    try:
        import torch

        dev = "cuda" if torch.cuda.is_available() else "cpu"
    except Exception:
        dev = "cpu"
    inp, rhs, bc = build_inputs(args.config, 0, 1, dev)
    n_node = inp.n
    sample = args.cpu_sample_iters or max(2, min(200, int(1.2e9 / n_node)))
    ref = pbref.from_inputs(inp)
    for _ in range(args.warmup):
        ref.solve(tol, min(sample, 2))
    t0 = time.perf_counter()
    iters = 0
    for _ in range(args.steps):
        iters += ref.solve(tol, sample)["iters"]
    dt = time.perf_counter() - t0
    ref.close()
    val = iters / dt
    desc = f"first {sample} PCG iterations of {workload_name(args.config, prec, tol)} per step (fp64 oracle)"
    return {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(1, args.steps),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": workload_name(args.config, prec, tol), "sample": desc},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": pbref.num_threads(), "kind": "oracle",
                             "sample": desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def plan_summary(solver, prec):
    """The launch plan that produced a number (pb_get_plan), as it goes into the JSON line."""
    pl = solver.plan(prec)
    keep = ("txv", "ty", "tz", "ring_slots", "blocks_per_sm", "tiles", "grid", "threads", "smem_bytes", "autotuned",
            "vec_grid", "vec_threads", "persist", "fused", "face_quad", "coef_slots", "face_palette", "diag_palette_vec",
            "diag_palette_spmv",
            "palette_size", "diag_palette_size", "num_sm", "pitch")
    return {k: pl[k] for k in keep}


def timed_solves(solver, torch, stream, prec, tol, args, out, steps, warmup):
    """`steps` complete pb_solve calls on device-resident data, CUDA events on the handle's stream."""
    for _ in range(warmup):
        res = solver.solve(tol, args.maxiter, prec, check_every=args.check_every, out=out)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    iters = 0
    e0.record(stream)
    for _ in range(steps):
        res = solver.solve(tol, args.maxiter, prec, check_every=args.check_every, out=out)
        iters += res["iters"]
    e1.record(stream)
    torch.cuda.synchronize()
    return iters, e0.elapsed_time(e1), res


def kernel_roofline(solver, prec, n_node, profile_iters, peak):
    """CUDA events around every launch of the two kernels (pb_profile), charged with the bytes the handle's storage
    format has to move (pb_bytes_per_node)."""
    solver.solve_begin(prec)
    solver.iterate(prec, 5)
    ms_spmv, ms_vec = solver.profile(prec, profile_iters)
    spmv_node, vec_node = solver.bytes_per_node(prec, 0), solver.bytes_per_node(prec, 1)
    ach_s = spmv_node * n_node / (ms_spmv * 1e-3) / 1e9
    ach_v = vec_node * n_node / (ms_vec * 1e-3) / 1e9 if ms_vec > 0 else None      # fused iteration: no K_vec launch
    return {"spmv_ms": ms_spmv, "vec_ms": ms_vec, "spmv_bytes_per_node": spmv_node, "vec_bytes_per_node": vec_node,
            "spmv_GBs": ach_s, "spmv_frac": ach_s / peak, "vec_GBs": ach_v,
            "vec_frac": (ach_v / peak) if ach_v is not None else None}


def run_ours(args, rank, local_rank, world):
    import torch

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=dev)
    from paper_1704_02745_b200 import build as pb_build

    if rank == 0:
        pb_build.build()
    if world > 1:
        dist.barrier()
    import paper_1704_02745_b200 as pkg

    pkg.load_library()
    prec = args.precision
    tol = args.tol or TOL[prec]
    tdt = torch.float32 if prec == "f32" else torch.float64
    t_gen = time.perf_counter()
    inp, rhs, bc = build_inputs(args.config, rank, world, f"cuda:{local_rank}")
    t_gen = time.perf_counter() - t_gen
    n_node, elt = inp.n, (4 if prec == "f32" else 8)

    stream = torch.cuda.Stream(device=dev)
    t_create = time.perf_counter()
    options = {k: int(v) for k, v in (kv.split("=", 1) for kv in args.opt)}
    solver = pkg.PBSolver(inp.nx, inp.ny, inp.nz, inp.h, inp.eps_x, inp.eps_y, inp.eps_z, inp.kbar2, rhs, bc,
                          stream=stream.cuda_stream, options=options)
    solver.prepare(prec)                     # work arrays of this precision + plan autotune (pb_prepare)
    torch.cuda.synchronize()
    t_create = time.perf_counter() - t_create
    out_d = torch.empty(solver.shape, dtype=tdt, device=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident leg: `value` -------------------------------------------------------------
    for _ in range(args.warmup):
        res = solver.solve(tol, args.maxiter, prec, check_every=args.check_every, out=out_d)
    barrier()
    l0 = solver.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    iters = 0
    with ClockSampler(physical_gpu_index(local_rank)) as clocks:
        e0.record(stream)
        for _ in range(args.steps):
            res = solver.solve(tol, args.maxiter, prec, check_every=args.check_every, out=out_d)
            iters += res["iters"]
        e1.record(stream)
        barrier()
    ms_local = e0.elapsed_time(e1)
    launches = solver.launch_count() - l0
    tot_iters, ms = aggregate(iters, ms_local, world, dev)
    value = tot_iters / (ms * 1e-3)

    # ---- roofline of the two kernels, CUDA events around every launch, taken right after the timed solves (same
    # power / clock state: k_spmv_tma follows the SM clock) ----------------------------------------------------
    peak, peak_src = measured_peak()
    with ClockSampler(physical_gpu_index(local_rank)) as clocks_prof:
        solver.solve(tol, args.maxiter, prec, check_every=args.check_every, out=out_d)
        kr = kernel_roofline(solver, prec, n_node, args.profile_iters, peak)

    # ---- end-to-end leg: host buffers, H2D of rhs/bc and D2H of phi inside the timed region -------
    e2e = None
    if not args.no_e2e:
        rhs_h = torch.from_numpy(rhs).pin_memory()
        bc_h = torch.from_numpy(bc).pin_memory()
        out_h = torch.empty(solver.shape, dtype=tdt).pin_memory()
        for _ in range(min(args.warmup, 2)):
            solver.set_rhs(rhs_h, bc_h)
            solver.solve(tol, args.maxiter, prec, check_every=args.check_every, out=out_h)
        barrier()
        it2 = 0
        t0 = time.perf_counter()
        for _ in range(args.steps):
            solver.set_rhs(rhs_h, bc_h)
            it2 += solver.solve(tol, args.maxiter, prec, check_every=args.check_every, out=out_h)["iters"]
        torch.cuda.synchronize()
        ms2_local = 1e3 * (time.perf_counter() - t0)
        barrier()
        tot2, ms2 = aggregate(it2, ms2_local, world, dev)
        e2e = {"value": tot2 / (ms2 * 1e-3), "unit": UNIT, "ms_per_step": ms2 / args.steps,
               "h2d_bytes_per_step": int(rhs.nbytes + bc.nbytes), "d2h_bytes_per_step": int(n_node * elt + 96)}
        del rhs_h, bc_h, out_h

    # ---- the MD-snapshot batch (same operator, seeded charge perturbations), N = 1 default at config 5 ----
    batch = None
    n_batch = args.batch if args.batch is not None else (50 if (world == 1 and args.config == 5) else 0)
    if n_batch > 0 and "charges" in inp.meta:
        batch = run_batch(args, pkg, inp, prec, tol, n_batch, rank, world, stream, dev, out_d, torch)

    # ---- optional (NEXT row f3): mixed-precision iterative refinement against the plain fp64 solve ----------------
    refined = None
    if args.refined:
        out64 = torch.empty((inp.nz, inp.ny, inp.nx), dtype=torch.float64, device=dev)
        tms = {}
        for name, fn in (("refined", lambda: solver.solve_refined(1e-10, args.maxiter, 1e-5, args.check_every, out=out64)),
                         ("f64", lambda: solver.solve(1e-10, args.maxiter, "f64", check_every=args.check_every, out=out64))):
            fn()                                                # builds the work arrays / warms up
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            r_ = fn()
            torch.cuda.synchronize()
            tms[name] = (1e3 * (time.perf_counter() - t0), r_, solver.residual(out64, "f64"))
        refined = {"tol": 1e-10, "refined_ms": tms["refined"][0], "outer": tms["refined"][1]["outer"],
                   "inner_iterations": tms["refined"][1]["iters"], "true_relres": tms["refined"][2],
                   "f64_ms": tms["f64"][0], "f64_iterations": tms["f64"][1]["iters"], "f64_true_relres": tms["f64"][2],
                   "note": "pb_solve_refined: fp64 potential and true residual, fp32 Jacobi-PCG corrections (inner_tol 1e-5)"}
        del out64

    # ---- optional (NEXT row f1): the same problem built on the GPU from atoms, and a charge update ---------------
    setup = None
    if args.setup_from_atoms and "charges" in inp.meta:
        setup = run_setup_from_atoms(args, pkg, inp, prec, tol, stream, out_d, t_gen, n_batch, torch)

    # ---- roofline of the dominant kernel (K_spmv), CUDA events around every launch ----------------
    wl = workload_name(args.config, prec, tol)
    ms_spmv, ms_vec = kr["spmv_ms"], kr["vec_ms"]
    pal, pald = solver.palette_size(), solver.diag_palette_size()
    # Bytes per launch.  `achieved` counts the bytes k_spmv_tma HAS to move in the storage format the handle uses
    # (pb_bytes_per_node): 10 words per node (tighter variant), or 6 words + 4 index bytes when the face
    # dielectrics and the Jacobi diagonal fit the palettes (lossless byte indices).  The same time charged with SURVEY's
    # uncompressed 10 words is given under `survey_10word` (it exceeds the copy peak because fewer bytes really move).
    spmv_bytes = kr["spmv_bytes_per_node"] * n_node
    vec_bytes = kr["vec_bytes_per_node"] * n_node
    iter_bytes = spmv_bytes + vec_bytes
    ns_bytes = WORDS_NORTH_STAR * elt * n_node
    t_solve = ms_local * 1e-3
    plan = plan_summary(solver, prec)
    fused = bool(plan.get("fused"))
    committed = ncu_traffic(f"{'k_pcg_fused' if fused else 'k_spmv'}:{wl}")
    kvec = (None if fused else
            {"achieved": kr["vec_GBs"], "frac": kr["vec_frac"], "bytes_per_node": kr["vec_bytes_per_node"],
             "diag_palette_size": pald, "ms_per_launch": ms_vec})
    roofline = {"bound": "hbm", "kernel": "k_pcg_fused" if fused else "k_spmv_tma",
                "kernel_note": ("one launch = one whole PCG iteration over all N nodes (K_spmv with K_vec folded in)" if fused
                                else "one launch = K_spmv over all N nodes; K_vec under k_vec"),
                "achieved": kr["spmv_GBs"], "peak": peak, "unit": "GB/s",
                "frac": kr["spmv_frac"], "traffic": committed, "traffic_ncu_committed": committed,
                "traffic_source": "profiles/ncu_traffic.csv: dram__bytes of a committed ncu --set full capture of this "
                                  "kernel and workload; NOT measured in this run",
                "peak_source": peak_src,
                "algorithmic_bytes_per_launch": spmv_bytes, "bytes_per_node": kr["spmv_bytes_per_node"],
                "bytes_accounting": "stored-format bytes (pb_bytes_per_node): what physically has to cross HBM; "
                                    "SURVEY 8(d)'s uncompressed words are in survey_10word / iteration.north_star_*",
                "palette_size": pal, "ms_per_launch": ms_spmv, "clocks_during_profile": clocks_prof.summary(),
                "plan": plan,
                "survey_words": {"words_per_node": WORDS_NORTH_STAR if fused else WORDS_SPMV,
                                 "bytes_per_launch": (WORDS_NORTH_STAR if fused else WORDS_SPMV) * elt * n_node,
                                 "GBs": (WORDS_NORTH_STAR if fused else WORDS_SPMV) * elt * n_node / (ms_spmv * 1e-3) / 1e9,
                                 "note": "the same launch time charged with SURVEY.md 8(d)'s uncompressed words: the whole "
                                         "16-word iteration for the fused kernel, the 10-word K_spmv otherwise"},
                "k_vec": kvec,
                "iteration": {"achieved": iter_bytes * iters / t_solve / 1e9,
                              "frac": iter_bytes * iters / t_solve / 1e9 / peak,
                              "north_star_16word_GBs": ns_bytes * iters / t_solve / 1e9,
                              "north_star_16word_frac_of_measured": ns_bytes * iters / t_solve / 1e9 / peak,
                              "north_star_16word_frac_of_8TBs": ns_bytes * iters / t_solve / 8e12,
                              "note": "achieved/frac: bytes this implementation moves per iteration (k_spmv_tma + k_vec) over "
                                      "the whole timed solves (init, polls, finish included); north_star_*: the same time "
                                      "charged with SURVEY.md 8(d)'s 16 words per node per iteration"}}

    # ---- the other precision and the word (no-palette) format of the same workload, N = 1 only --------------------
    if world == 1 and not args.no_variants:
        other = "f64" if prec == "f32" else "f32"
        try:
            roofline[other] = variant_leg(solver, torch, stream, other, TOL[other], args, inp, peak)
            if fused:
                solver.set_option("fused", 0)      # the same workload through K_spmv + K_vec (two launches per iteration)
                roofline["two_kernel"] = variant_leg(solver, torch, stream, prec, tol, args, inp, peak)
                solver.set_option("fused", 1)
            solver.set_option("palette", 0)        # word format: 40 B (fp32) / 80 B (fp64) per node in k_spmv_tma
            roofline["no_palette"] = variant_leg(solver, torch, stream, prec, tol, args, inp, peak)
            roofline["no_palette"]["note"] = ("PB_OPT_PALETTE = 0: face dielectrics and Dinv as full words, the format an "
                                              "operator with a continuum of face values (e.g. fractional-edge harmonic "
                                              "weights, PAPER.md:182) gets")
            solver.set_option("palette", 1)
        except pkg.PBError as e:                   # e.g. out of memory on a smaller device: report, do not hide
            roofline["variants_error"] = str(e)

    line = None
    if rank == 0:
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            cpu = cpu_baseline(args, inp, tol, wl)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": prec, "data": "synthetic",
                "config": {"workload": wl, "grid": [inp.nx, inp.ny, inp.nz], "unknowns_per_gpu": n_node,
                           "tol": tol, "check_every": args.check_every, "iterations_per_solve": res["iters"],
                           "final_relres": res["relres"], "time_to_solution_ms": ms / args.steps,
                           "parallelism": f"replicas x{world} (one right-hand side per GPU)",
                           "l2": "working set 11 arrays x %.0f MB >> 126 MB L2 (inputs larger than L2)"
                                 % (n_node * elt / 1e6) if n_node * elt * 11 > 4e8 else "working set fits L2",
                           "create_ms": 1e3 * t_create, "input_generation_s": t_gen, "options": options},
                "clocks": clocks.summary(), "e2e": e2e, "gpu_launches": int(launches),
                "roofline": roofline, "cpu_baseline": cpu}
        if batch is not None:
            line["batch"] = batch
        if setup is not None:
            line["setup_from_atoms"] = setup
        if refined is not None:
            line["refined"] = refined
    solver.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return line


def variant_leg(solver, torch, stream, prec, tol, args, inp, peak):
    """One warm-up and two timed solves plus the per-kernel roofline of another precision / storage format of the
    SAME workload and handle (the headline `value` is not touched by this)."""
    tdt = torch.float32 if prec == "f32" else torch.float64
    solver.prepare(prec)
    out = torch.empty(solver.shape, dtype=tdt, device=f"cuda:{torch.cuda.current_device()}")
    iters, ms, res = timed_solves(solver, torch, stream, prec, tol, args, out, steps=2, warmup=1)
    kr = kernel_roofline(solver, prec, inp.n, max(10, args.profile_iters // 2), peak)
    del out
    return {"dtype": prec, "tol": tol, "value": iters / (ms * 1e-3), "unit": UNIT, "iterations_per_solve": res["iters"],
            "final_relres": res["relres"], "ms_per_solve": ms / 2,
            "kernel": "k_pcg_fused" if solver.plan(prec)["fused"] else "k_spmv_tma",
            "achieved": kr["spmv_GBs"], "frac": kr["spmv_frac"], "bytes_per_node": kr["spmv_bytes_per_node"],
            "ms_per_launch": kr["spmv_ms"],
            "k_vec": (None if kr["vec_GBs"] is None else
                      {"achieved": kr["vec_GBs"], "frac": kr["vec_frac"], "bytes_per_node": kr["vec_bytes_per_node"],
                       "ms_per_launch": kr["vec_ms"]}),
            "iteration_frac": (kr["spmv_bytes_per_node"] + kr["vec_bytes_per_node"]) * inp.n * iters / (ms * 1e-3) / 1e9 / peak,
            "plan": plan_summary(solver, prec)}


def run_batch(args, pkg, inp, prec, tol, n_batch, rank, world, stream, dev, out_d, torch):
    """Config 5's perturbed-charge batch (BASELINE.json configs[4]: 50 solves, same operator, charges + N(0, 0.05) e) on
    an atom-built handle -- every member's right-hand side and ghost values are made on the GPU (pb_set_charges /
    pb_solve_batch_charges, NEXT rows f1 + f2):
      sequential: pb_set_charges + pb_solve per member (cold start);  warm_start: the same members solved again from
      the previous member's potential (pb_solve_from);  multi_rhs: pb_solve_batch_charges, 1 / 2 / 4 members per pass."""
    from workloads import perturbed_charge_values

    m = inp.meta
    t0 = time.perf_counter()
    s2 = pkg.PBSolver.from_atoms(inp.nx, inp.ny, inp.nz, inp.h, m["centres"], m["radii"], m["charges"], m["eps_in"],
                                 m["eps_out"], m["kbar2_solvent"], stream=stream.cuda_stream)
    s2.prepare(prec)
    torch.cuda.synchronize()
    t_create = time.perf_counter() - t0
    Q = np.stack([perturbed_charge_values(inp, world * sidx + rank) for sidx in range(n_batch)])
    t_set, t_b, it_b, t_w, it_w = 0.0, 0.0, [], 0.0, []
    out_w = torch.empty_like(out_d)
    for sidx in range(n_batch):
        t0 = time.perf_counter()
        s2.set_charges(Q[sidx])
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        it_b.append(s2.solve(tol, args.maxiter, prec, check_every=args.check_every, out=out_d)["iters"])
        torch.cuda.synchronize()
        t2 = time.perf_counter()
        t_set += t1 - t0
        t_b += t2 - t1
        if sidx == 0:
            out_w.copy_(out_d)
        else:
            t0 = time.perf_counter()
            it_w.append(s2.solve(tol, args.maxiter, prec, check_every=args.check_every, out=out_w, phi0=out_w)["iters"])
            torch.cuda.synchronize()
            t_w += time.perf_counter() - t0
    del out_w
    seq_ms = 1e3 * (t_set + t_b) / n_batch
    multi = {}
    Qd = torch.from_numpy(Q).to(dev)
    tdt = torch.float32 if prec == "f32" else torch.float64
    for width in (1, 2, 4):
        nm = n_batch if width == 2 else min(n_batch, 12)
        nm -= nm % width if nm >= width else 0
        out_m = torch.empty((nm,) + tuple(out_d.shape), dtype=tdt, device=dev)
        s2.set_option("batch_width", width)
        try:
            s2.solve_batch_charges(Qd[:width], tol, args.maxiter, prec, check_every=args.check_every, out=out_m[:width])  # plan + arrays
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            g = s2.solve_batch_charges(Qd[:nm], tol, args.maxiter, prec, check_every=args.check_every, out=out_m)
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            # the members' setup alone (maxiter = 0: charges -> rhs / ghost values -> b, init, un-pad), same call path
            t0 = time.perf_counter()
            s2.solve_batch_charges(Qd[:nm], tol, 0, prec, check_every=args.check_every, out=out_m)
            torch.cuda.synchronize()
            dt_setup = time.perf_counter() - t0
            solve_ms = 1e3 * (dt - dt_setup) / nm
            multi[f"width{width}"] = {"members": nm, "ms_per_member": 1e3 * dt / nm, "solves_per_s": nm / dt,
                                      "setup_ms_per_member": 1e3 * dt_setup / nm,
                                      "solve_ms_per_member": solve_ms, "mean_iters": float(np.mean(g["iters"])),
                                      "ms_per_member_iteration": solve_ms / float(np.mean(g["iters"])),
                                      "all_converged": all(st == 0 for st in g["status"])}
        except pkg.PBError as e:
            multi[f"width{width}"] = {"error": str(e)}
        del out_m
    s2.close()
    seq_solve_ms = 1e3 * t_b / n_batch
    w2 = multi.get("width2", {})
    return {"solves": n_batch, "solves_per_s": n_batch / (t_set + t_b), "ms_per_solve": seq_ms,
            "set_charges_ms": 1e3 * t_set / n_batch, "solve_ms": seq_solve_ms,
            "iterations_per_s": float(np.sum(it_b)) / t_b,
            "mean_iters": float(np.mean(it_b)), "min_iters": int(min(it_b)), "max_iters": int(max(it_b)),
            "warm_start": ({"mean_iters": float(np.mean(it_w)), "solve_ms": 1e3 * t_w / len(it_w)} if it_w else None),
            "multi_rhs": multi,
            "multi_rhs_speedup_width2": (seq_solve_ms / w2["solve_ms_per_member"]) if "solve_ms_per_member" in w2 else None,
            "handle_create_ms": 1e3 * t_create,
            "note": "atom-built handle (pb_create_from_atoms), this rank only, wall clock; set_charges = charge spreading + "
                    "the fp64 Debye-Hueckel boundary sum per member (inside ms_per_solve and ms_per_member; solve_ms_per_member = "
                    "the call minus the same call with maxiter 0); multi_rhs: pb_solve_batch_charges with PB_OPT_BATCH_WIDTH members "
                    "per kernel pass (k_spmv_batch + k_vec_batch)"}


def run_setup_from_atoms(args, pkg, inp, prec, tol, stream, out_d, t_gen, n_batch, torch):
    from workloads import perturbed_charge_values

    m = inp.meta
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    s2 = pkg.PBSolver.from_atoms(inp.nx, inp.ny, inp.nz, inp.h, m["centres"], m["radii"], m["charges"],
                                 m["eps_in"], m["eps_out"], m["kbar2_solvent"], stream=stream.cuda_stream)
    torch.cuda.synchronize()
    t_fa = time.perf_counter() - t0
    t0 = time.perf_counter()
    s2.prepare(prec)
    torch.cuda.synchronize()
    t_prep = time.perf_counter() - t0
    nb = min(n_batch, 10) if n_batch > 0 else 3
    t_sc, t_sv, it_sc = [], [], []
    for sidx in range(nb):
        qs = perturbed_charge_values(inp, sidx)
        t0 = time.perf_counter()
        s2.set_charges(qs)
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        it_sc.append(s2.solve(tol, args.maxiter, prec, check_every=args.check_every, out=out_d)["iters"])
        torch.cuda.synchronize()
        t_sc.append(t1 - t0)
        t_sv.append(time.perf_counter() - t1)
    # the same charge updates with the boundary terms in fp32 (pb_set_setup_precision)
    s2.set_setup_precision("f32")
    t_sc32, it_sc32 = [], []
    for sidx in range(nb):
        qs = perturbed_charge_values(inp, sidx)
        t0 = time.perf_counter()
        s2.set_charges(qs)
        torch.cuda.synchronize()
        t_sc32.append(time.perf_counter() - t0)
        it_sc32.append(s2.solve(tol, args.maxiter, prec, check_every=args.check_every, out=out_d)["iters"])
    s2.close()
    nbc = 2 * (inp.nz * inp.ny + inp.nz * inp.nx + inp.ny * inp.nx)
    terms = float(nbc) * len(m["charges"])
    t_sc, t_sv, t_sc32 = float(np.median(t_sc)), float(np.median(t_sv)), float(np.median(t_sc32))   # per call (host clock)
    return {"create_from_atoms_ms": 1e3 * t_fa, "prepare_ms": 1e3 * t_prep, "set_charges_ms": 1e3 * t_sc,
            "solve_ms": 1e3 * t_sv,
            "mean_iters": float(np.mean(it_sc)), "members": nb, "atoms": int(len(m["charges"])),
            "dh_terms": terms, "dh_gterms_per_s": terms / t_sc / 1e9,
            "set_charges_f32_ms": 1e3 * t_sc32, "dh_f32_gterms_per_s": terms / t_sc32 / 1e9,
            "mean_iters_f32_boundary": float(np.mean(it_sc32)),
            "host_generator_s": t_gen,
            "note": "per-call times are medians over the members (host clock); pb_create_from_atoms = mask + faces + salt + charges + Debye-Hueckel ghosts + pb_create; prepare = "
                    "work arrays + plan autotune; set_charges = charge spreading + the fp64 DH boundary sum (ALU-bound); "
                    "set_charges_f32 = the same with the boundary terms in fp32 (pb_set_setup_precision)"}


def cpu_baseline(args, inp, tol, wl):
    """The fp64 oracle, as it stands, on the host cores: a bounded sample of the benchmarked workload, plus (BASELINE.md
    section 3) every smaller config, with 1 thread as well for grids <= 129^3 (the paper's CPU/CG is single-core,
    PAPER.md:184).  A reported baseline, not the target."""
    from oracle import pbref
    from workloads import make_config

    n_node = inp.n
    sample = args.cpu_sample_iters or max(2, min(400, int(1.2e10 / n_node)))
    ncores = pbref.num_threads()
    ref = pbref.from_inputs(inp)
    t0 = time.perf_counter()
    o = ref.solve(tol, sample)
    dt = time.perf_counter() - t0
    ref.close()
    cpu = {"value": o["iters"] / dt, "unit": UNIT, "cores": ncores, "kind": "oracle", "dtype": "f64",
           "sample": f"first {o['iters']} PCG iterations of {wl} (fp64 C/OpenMP oracle, {dt:.1f} s)"}
    if args.cpu_per_config:
        per = {}
        for cfg in range(1, args.config):
            ci = make_config(cfg, device="cuda")
            for ptol in sorted({TOL["f32"], TOL["f64"]}, reverse=True):
                for threads in ([ncores, 1] if GRID[cfg] <= 129 else [ncores]):
                    budget = int(6e8 / ci.n) + 2 if threads > 1 else int(1.5e8 / ci.n) + 2
                    pbref.set_num_threads(threads)
                    r = pbref.from_inputs(ci)
                    t0 = time.perf_counter()
                    oo = r.solve(ptol, min(5000, budget))
                    d = time.perf_counter() - t0
                    r.close()
                    per[f"config{cfg}_{GRID[cfg]}^3_tol{ptol:g}_{threads}thr"] = {
                        "iterations": oo["iters"], "converged": oo["status"] == 0, "s": d,
                        "iterations_per_s": oo["iters"] / d if d > 0 else None}
            pbref.set_num_threads(ncores)
        cpu["per_config"] = per
    return cpu


def run_slab(args, rank, local_rank, world):
    """One solve of the configured workload cut into z-slabs (paper_1704_02745_b200/slab.py): one slab per rank under
    torchrun (halo planes and the three dot products over NCCL), or args.slab slabs on one GPU.  Strong scaling."""
    import torch

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=dev)
    from paper_1704_02745_b200 import build as pb_build

    if rank == 0:
        pb_build.build()
    if world > 1:
        dist.barrier()
    from paper_1704_02745_b200.slab import SlabComm, SlabRank, partition, slab_inputs, solve_slabs

    prec = args.precision
    tol = args.tol or TOL[prec]
    inp, rhs, bc = build_inputs(args.config, 0, 1, f"cuda:{local_rank}")
    nslabs = world if world > 1 else max(1, args.slab)
    owner = list(range(world)) if world > 1 else [0] * nslabs
    parts = partition(inp.nz, nslabs)
    stream = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(stream):
        comm = SlabComm(owner, rank, dist)
        ranks = {}
        for s in comm.local():
            z0, nzl = parts[s]
            ranks[s] = SlabRank(s, nslabs, inp.nx, inp.ny, nzl, inp.h,
                                *slab_inputs(inp.nx, inp.ny, inp.nz, inp.eps_x, inp.eps_y, inp.eps_z, inp.kbar2, rhs, bc,
                                             z0, nzl), stream=stream.cuda_stream)
        for _ in range(max(1, args.warmup)):
            res = solve_slabs(ranks, comm, tol, args.maxiter, prec, args.check_every, device_result=True)
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        iters = 0
        with ClockSampler(physical_gpu_index(local_rank)) as clocks:
            e0.record(stream)
            for _ in range(args.steps):
                res = solve_slabs(ranks, comm, tol, args.maxiter, prec, args.check_every, device_result=True)
                iters += res[comm.local()[0]]["iters"]
            e1.record(stream)
            torch.cuda.synchronize()
            if world > 1:
                dist.barrier()
        ms_local = e0.elapsed_time(e1)
        for r in ranks.values():
            r.close()
    _, ms = aggregate(0, ms_local, world, dev)
    line = None
    if rank == 0:
        first = res[comm.local()[0]]
        line = {"metric": METRIC, "value": iters / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong",
                "vs_baseline": None, "dtype": prec, "data": "synthetic",
                "config": {"workload": workload_name(args.config, prec, tol), "grid": [inp.nx, inp.ny, inp.nz],
                           "parallelism": f"one solve, {nslabs} z-slabs" + ("" if world > 1 else " emulated on one GPU"),
                           "slabs": parts, "iterations_per_solve": first["iters"], "final_relres": first["relres"],
                           "check_every": args.check_every,
                           "exchange": "per iteration: 2+2 boundary planes per neighbour, all-reduce of 1 and of 2 doubles"},
                "clocks": clocks.summary(), "e2e": None, "gpu_launches": None, "roofline": None, "cpu_baseline": None}
    if world > 1:
        dist.destroy_process_group()
    return line


def self_launch(args, argv):
    """`python bench.py --gpus N` (N > 1) started without a launcher: start the N local ranks ourselves, the way the
    driver does (torch.distributed.run, one rank per GPU, rendezvous on 127.0.0.1)."""
    import socket
    import subprocess

    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *argv]
    return subprocess.call(cmd)


def main(argv=None):
    argv = list(sys.argv[1:] if argv is None else argv)
    args = parse_args(argv)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(self_launch(args, argv))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world != args.gpus and rank == 0:
        print(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}; reporting n_gpus={world}", file=sys.stderr)
    if args.impl == "reference":
        line = run_reference(args, rank, world)
    elif args.slab:
        line = run_slab(args, rank, local_rank, world)
    else:
        line = run_ours(args, rank, local_rank, world)
    if line is not None:
        print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
