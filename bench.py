#!/usr/bin/env python
"""bench.py -- headline measurement of the GMG pressure-Poisson solve on B200.

A "step" is one pass of the whole hot path: one GMG-RBGS Poisson solve (V(2,2) cycles with the
adaptive red-black Gauss-Seidel smoother on anisotropically coarsened levels, to relative
residual 1e-4 from a zero initial guess) on one seeded synthetic workload.  Default workload:
BASELINE.json configs[4], the 1024^3 periodic cube with 64 BDIM-ramped solid spheres -- the
configuration the north_star's HBM-roofline target is stated on (the other configs fit in L2
and are reported under "other_workloads").  Metric: ns per cell per Poisson solve (lower is
better).  Multi-GPU: replicas only (the north_star excludes sharding): every rank solves its
own copy, value = time / (N * cells).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c4|c4_512|c1|...]
    python bench.py --impl reference      # the FP64 CPU oracle on a bounded sample
"""
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

METRIC = "poisson_solve_ns_per_cell_gmg_rbgs_tol1e-4"
UNIT = "ns/cell"


def profiled_traffic(workload, kernel):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of `kernel` from the
    committed `ncu --set full` capture of this workload (profiles/traffic.json), else None."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            return float(json.load(f)[workload][kernel]["dram_bytes_per_launch"])
    except Exception:
        return None


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index = index
        self.samples = []
        self._stop = threading.Event()
        self._t = None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True,
                                     text=True, timeout=5).stdout.strip()
                if out:
                    self.samples.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self._stop.wait(0.2)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for s in self.samples:
            try:
                sm.append(float(s[0]))
                mx.append(float(s[1]))
                for nm, v in zip(names, s[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def _omp_threads(n=None):
    """Thread count of the OpenMP runtime the oracle's library runs on (set when n is given)."""
    import ctypes
    try:
        gomp = ctypes.CDLL("libgomp.so.1")
        if n is not None:
            gomp.omp_set_num_threads(int(n))
        return int(gomp.omp_get_max_threads())
    except OSError:
        return int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))


def oracle_solve_time(wl, threads=None, solver=None):
    """One solve (GMG-RBGS unless told otherwise) of workload wl with the FP64 oracle, as it stands;
    returns seconds, iterations, threads used, status.  threads: None = all the runtime offers."""
    import oracle
    all_threads = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    cores = _omp_threads(threads if threads is not None else all_threads)
    h = oracle.Hierarchy(wl.n, wl.bc, wl.L)
    t0 = time.perf_counter()
    out = h.solve(oracle.GMG_RBGS if solver is None else solver, wl.z, tol=wl.tol, maxiter=wl.maxiter)
    dt = time.perf_counter() - t0
    _omp_threads(all_threads)
    return dt, out["iterations"], cores, out["status"]


def run_reference(args):
    """--impl reference: the oracle (plain FP64 C, OpenMP over k) on the host cores, each step
    one solve of a bounded sample of the workload (same generator, shrunk grid)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2607_07687_b200 import workloads as W
    sample = args.reference_sample
    wl = W.by_name(sample)
    for _ in range(min(args.warmup, 1)):
        oracle_solve_time(wl)
    times, its = [], []
    for _ in range(args.steps):
        dt, it, cores, status = oracle_solve_time(wl)
        times.append(dt)
        its.append(it)
    ms = 1e3 * sum(times) / len(times)
    val = ms * 1e6 / wl.cells
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": ms,
        "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": f"configs[4] recipe shrunk to {sample} ({wl.n[0]}x{wl.n[1]}x{wl.n[2]}), "
                               "GMG-RBGS V(2,2) to tol 1e-4", "iterations": its[-1]},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{sample}: one full solve per step"},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def solver_table(gmg, W, torch, device, names, with_oracle=False):
    """#iterations, final residual, ms and ns/cell of PCG, GMG-PCG, GMG-CGS and GMG-RBGS per workload
    (the columns of the paper's Table 1; device-resident, best of 3).  GMG-PCG =
    V-cycle-preconditioned CG (BASELINE.json's meaning); GMG-CGS = the V-cycle with a Jacobi-PCG
    smoother (the paper's meaning of "GMG-PCG", reading O12)."""
    out = {}
    for name in names:
        wl = W.by_name(name)
        g = gmg.GMG(wl.n, wl.bc, device=str(device))
        L = torch.from_numpy(wl.L).to(device)
        z = torch.from_numpy(wl.z).to(device)
        g.set_coeffs(L)
        p = torch.zeros_like(z)
        row = {}
        for label, solver, cap in (("PCG", gmg.PCG, 5000), ("GMG-PCG", gmg.GMG_PCG, wl.maxiter),
                                   ("GMG-CGS", gmg.GMG_CGS, wl.maxiter),
                                   ("GMG-RBGS", gmg.GMG_RBGS, wl.maxiter)):
            best = None
            for _ in range(3):
                p.zero_()
                g.set_omega(1.0)
                g.solve(p, z, tol=wl.tol, maxiter=cap, solver=solver)
                st = g.stats()
                best = st["gpu_ms"] if best is None else min(best, st["gpu_ms"])
            row[label] = {"iterations": st["iterations"], "resid": st["resid_final_rel"], "ms": best,
                          "ns_per_cell": best * 1e6 / wl.cells}
        g.close()
        if with_oracle:
            # the FP64 oracle beside it (all cores and one thread; a stated
            # baseline, not a target): the same GMG-RBGS solve on the host
            dt, it, cores, status = oracle_solve_time(wl)
            dt1, it1, _, _ = oracle_solve_time(wl, threads=1)
            row["oracle GMG-RBGS (FP64, host)"] = {
                "iterations": it, "status": status, "cores": cores, "ms": dt * 1e3,
                "ns_per_cell": dt * 1e9 / wl.cells, "ms_1thread": dt1 * 1e3,
                "ns_per_cell_1thread": dt1 * 1e9 / wl.cells}
        out[name] = row
    return out


def step_table(gmg, W, torch, device, exps=(5, 6), nsteps=16):
    """Warm-started pressure steps with a moving body (Table 1's shape: average
    iterations per solve, final residual, cost per cell per step): per step gmg_set_coeffs ->
    gmg_divergence -> gmg_solve (p from the step before) -> gmg_project, device-resident, CUDA
    events around the whole step.  The first (cold) step is reported separately."""
    from paper_2607_07687_b200.pressure_step import PressureStepper
    out = {}
    for pe in exps:
        nx = 2 ** (pe + 1)
        n, bc = (nx, nx, nx // 2), W.JELLYFISH_BC
        cells = n[0] * n[1] * n[2]
        seq = [(torch.from_numpy(L).to(device), torch.from_numpy(u).to(device))
               for L, u in W.jellyfish_steps(pe, nsteps)]
        row = {}
        for label, solver, cap in (("PCG", gmg.PCG, 5000), ("GMG-PCG", gmg.GMG_PCG, 50),
                                   ("GMG-CGS", gmg.GMG_CGS, 50), ("GMG-RBGS", gmg.GMG_RBGS, 50)):
            ps = PressureStepper(n, bc, solver=solver, tol=1e-4, maxiter=cap, device=str(device))
            its, res, ms = [], [], []
            Lcur = torch.empty_like(seq[0][0])   # the body update rewrites ONE coefficient array
            for L, u in seq:
                uu = u.clone()
                Lcur.copy_(L)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                rc, st = ps.step(Lcur, uu)
                e1.record()
                torch.cuda.synchronize()
                its.append(st["iterations"]); res.append(st["resid_final_rel"]); ms.append(e0.elapsed_time(e1))
            ps.close()
            warm = slice(1, None)
            row[label] = {"iterations_first": its[0],
                          "iterations_avg": sum(its[warm]) / len(its[warm]),
                          "resid_avg": sum(res[warm]) / len(res[warm]),
                          "ms_per_step": sum(ms[warm]) / len(ms[warm]),
                          "ns_per_cell_per_step": sum(ms[warm]) / len(ms[warm]) * 1e6 / cells}
        out[f"jellyfish_p{pe}_{n[0]}x{n[1]}x{n[2]}_{nsteps}steps"] = row
    return out


def time_kernel_loop(fn, reps, stream):
    import torch
    e0 = torch.cuda.Event(enable_timing=True)
    e1 = torch.cuda.Event(enable_timing=True)
    fn()
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(reps):
        fn()
    e1.record(stream)
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_2607_07687_b200 import gmg, replicas
    from paper_2607_07687_b200 import workloads as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    device = torch.device(f"cuda:{local}")
    if world > 1:
        dist.init_process_group("nccl", device_id=device)

    def barrier():
        replicas.barrier()
        torch.cuda.synchronize()

    t_gen = time.perf_counter()
    wl = W.by_name(args.workload)
    t_gen = time.perf_counter() - t_gen
    N = wl.cells
    g = gmg.GMG(wl.n, wl.bc, device=str(device), **({"use_graph": 0} if args.no_graph else {}))
    L = torch.from_numpy(wl.L).to(device)
    z = torch.from_numpy(wl.z).to(device)
    p = torch.zeros_like(z)
    g.set_coeffs(L)
    stream = torch.cuda.current_stream(device)
    tol, maxiter = wl.tol, wl.maxiter

    # ---- device-resident timing: W warm-up + exactly K timed steps ---------------------------
    for _ in range(args.warmup):
        p.zero_()
        g.set_omega(1.0)
        g.solve(p, z, tol=tol, maxiter=maxiter, solver=gmg.GMG_RBGS)
    launches = 0
    iters = []
    barrier()
    sampler = ClockSampler(local)
    e0 = torch.cuda.Event(enable_timing=True)
    e1 = torch.cuda.Event(enable_timing=True)
    marks = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    with sampler:
        e0.record(stream)
        for i in range(args.steps):
            p.zero_()
            g.set_omega(1.0)
            rc = g.solve(p, z, tol=tol, maxiter=maxiter, solver=gmg.GMG_RBGS)
            st = g.stats()
            launches += st["kernel_launches"] + 1
            iters.append(st["iterations"])
            marks[i].record(stream)
        e1.record(stream)
        barrier()
    ms_total = replicas.max_over_ranks(e0.elapsed_time(e1), device)
    ms_step = ms_total / args.steps
    # burst vs sustained: the first steps run at boost clocks, a long run settles under the power
    # cap -- both are reported, `value` is the mean over ALL timed steps
    n_first = min(5, args.steps)
    ms_first = e0.elapsed_time(marks[n_first - 1]) / n_first
    ms_last = (marks[-n_first - 1].elapsed_time(marks[-1]) / n_first) if args.steps >= 2 * n_first else None
    final = g.stats()
    value = replicas.ns_per_cell(ms_step, N, world)
    ns_per_cell_vcycle = (final["gpu_ms"] * 1e6 / N) / max(final["iterations"], 1)

    # ---- BASELINE.json configs[4]: "fixed 10 GMG-RBGS V-cycles" (reading O9: tol = 0, maxiter = 10;
    # PAPER.md:51 counts V-cycles) -- the per-cycle cost without the loop-entry share of a 3-cycle solve
    fixed = None
    if not args.no_fixed:
        f_ms = []
        for _ in range(3):
            p.zero_()
            g.set_omega(1.0)
            rc10 = g.solve(p, z, tol=0.0, maxiter=10, solver=gmg.GMG_RBGS)
            s10 = g.stats()
            f_ms.append(s10["gpu_ms"])
        f_ms.sort()
        fixed = {"cycles": s10["iterations"], "status": rc10, "ms": f_ms[1], "ms_per_vcycle": f_ms[1] / 10.0,
                 "ns_per_cell_per_vcycle": f_ms[1] * 1e5 / N, "resid_after_10": s10["resid_final_rel"],
                 "algorithmic_bytes_per_cell_per_vcycle": s10["bytes_as_run"] / 10.0 / N,
                 "algorithmic_GBs": s10["bytes_as_run"] / (f_ms[1] * 1e-3) / 1e9,
                 "reference_line_bytes_per_cell_per_vcycle": s10["bytes_algorithmic"] / 10.0 / N,
                 "note": "median of 3; tol = 0, maxiter = 10 (returns NOT_CONVERGED by construction)"}
    p.zero_()
    g.set_omega(1.0)
    g.solve(p, z, tol=tol, maxiter=maxiter, solver=gmg.GMG_RBGS)

    # ---- end to end through the C-ABI with HOST buffers (pinned), copies inside the region -----
    # The workload's initial guess is zero: gmg_solve_host_cold makes it on the device, so per step
    # z goes up (4N bytes) and p comes down (4N bytes).  The general entry point gmg_solve_host
    # uploads a caller-supplied guess as well (8N bytes up); it is timed beside it.
    zh = torch.from_numpy(wl.z).pin_memory()
    ph = torch.zeros(wl.z.shape, dtype=torch.float32).pin_memory()
    e2e_steps = max(1, min(args.steps, 3))

    def time_e2e(call):
        g.set_omega(1.0)
        call()
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            g.set_omega(1.0)
            call()
        barrier()
        return replicas.max_over_ranks(1e3 * (time.perf_counter() - t0) / e2e_steps, device)

    e2e_ms = time_e2e(lambda: g.solve_host_cold(ph, zh, tol=tol, maxiter=maxiter, solver=gmg.GMG_RBGS))
    e2e_val = replicas.ns_per_cell(e2e_ms, N, world)

    def with_guess():
        ph.zero_()      # the caller's guess (zero here), prepared on the host inside the region
        g.solve_host(ph, zh, tol=tol, maxiter=maxiter, solver=gmg.GMG_RBGS)

    e2e_guess_ms = time_e2e(with_guess)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel: the level-0 red+black sweep ------------------------
    peak, peak_src = measured_peak()
    b0 = z
    q = torch.zeros_like(z)
    reps = 4 if N > (1 << 28) else 20
    t_pair = time_kernel_loop(lambda: g.op_smooth(0, q, b0, omega=1.0, nsweeps=2), reps, stream)
    t_sweep = t_pair / 2.0
    # Algorithmic bytes of the sweep AS RUN: 24 B/cell (p read + write, b, three coefficient arrays)
    # where a CTA loads its coefficients, 12 B/cell on the lean path (uniform bricks: the coefficient
    # streams are not moved; SURVEY.md S8(d) "honest only if reported as such").  The 24-B accounting
    # stays beside it as the reference line.
    f_uni = final["uniform_fraction"]
    f_uni_res = final["uniform_fraction_residual"]
    sweep_bytes_cell = 24.0 - 12.0 * f_uni
    sweep_gbs = sweep_bytes_cell * N / (t_sweep * 1e-3) / 1e9
    sweep_gbs_24 = 24.0 * N / (t_sweep * 1e-3) / 1e9
    try:    # the variant of the sweep that also accumulates the stopping-test norm (fused_norm)
        t_sweep_norm = time_kernel_loop(lambda: g.op_sweep_with_norm(0, q, b0, omega=1.0), reps, stream)
    except gmg.GMGError:
        t_sweep_norm = None
    t_rr = time_kernel_loop(lambda: g.op_residual_restrict(0, q, b0), reps, stream)
    _, c0 = g.level_shape(0)
    m = c0[0] * c0[1] * c0[2]
    rr_bytes_cell = 20.0 - 12.0 * f_uni_res + 4.0 / m
    rr_gbs = rr_bytes_cell * N / (t_rr * 1e-3) / 1e9
    # whole solve / cycles, for the bytes as for the time (loop entry and exit included)
    vc_bytes = final["bytes_as_run"] / max(final["iterations"], 1)
    vc_bytes_ref = final["bytes_algorithmic"] / max(final["iterations"], 1)
    vc_ms = (final["gpu_ms"]) / max(final["iterations"], 1)
    vcycle_gbs = vc_bytes / (vc_ms * 1e-3) / 1e9

    # ---- the passes either side of the solve --------------------------
    areps = 3 if N > (1 << 28) else 10
    t_set = time_kernel_loop(lambda: g.set_coeffs(L), areps, stream)
    u = torch.zeros((3,) + tuple(z.shape), dtype=torch.float32, device=device)
    t_div = time_kernel_loop(lambda: g.divergence(u), areps, stream)
    t_prj = time_kernel_loop(lambda: g.project(u, p), areps, stream)
    del u
    set_bytes = 12.0 * (1.0 + 1.0 / m)          # level 0 -> 1; the coarser levels add < 2 %
    around = {
        "set_coeffs": {"ms": t_set, "algorithmic_bytes_per_cell": set_bytes,
                       "algorithmic_GBs": set_bytes * N / (t_set * 1e-3) / 1e9,
                       "note": "validation + every level's coefficients + D2H status, per call"},
        "divergence": {"ms": t_div, "algorithmic_bytes_per_cell": 16.0,
                       "algorithmic_GBs": 16.0 * N / (t_div * 1e-3) / 1e9},
        "project": {"ms": t_prj, "algorithmic_bytes_per_cell": 40.0,
                    "algorithmic_GBs": 40.0 * N / (t_prj * 1e-3) / 1e9},
    }

    # ---- cpu_baseline: the oracle, as it stands, on a bounded sample -------------------------
    cpu = None
    if not args.no_cpu_baseline:
        swl = W.by_name(args.cpu_sample if N > (1 << 27) else args.reference_sample)
        dt, it, cores, status = oracle_solve_time(swl)
        cpu = {"value": dt * 1e9 / swl.cells, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{swl.name} ({swl.n[0]}^3, same recipe as the workload): "
                         f"one full solve, {it} V-cycles, {dt:.1f} s"}

    # ---- the paper's three-way comparison (Table 1's columns) on the small configs ----------
    table = None
    if not args.no_table:
        table = solver_table(gmg, W, torch, device,
                             ["c0", "c1", "c2", "c3p5", "c3p6"] if N > (1 << 22) else [args.workload],
                             with_oracle=not args.no_cpu_baseline)
        # the big workload itself: GMG-RBGS is the timed step above; GMG-PCG beside it
        if N > (1 << 22):
            p.zero_()
            rc = g.solve(p, z, tol=tol, maxiter=maxiter, solver=gmg.GMG_PCG)
            st2 = g.stats()
            p.zero_()
            rc = g.solve(p, z, tol=tol, maxiter=maxiter, solver=gmg.GMG_CGS)
            st3 = g.stats()
            table[args.workload] = {
                "GMG-CGS": {"iterations": st3["iterations"], "resid": st3["resid_final_rel"],
                            "ms": st3["gpu_ms"], "ns_per_cell": st3["gpu_ms"] * 1e6 / N},
                "GMG-RBGS": {"iterations": iters[-1], "resid": final["resid_final_rel"],
                             "ms": final["gpu_ms"], "ns_per_cell": final["gpu_ms"] * 1e6 / N},
                "GMG-PCG": {"iterations": st2["iterations"], "resid": st2["resid_final_rel"],
                            "ms": st2["gpu_ms"], "ns_per_cell": st2["gpu_ms"] * 1e6 / N}}
            if cpu is not None:   # the oracle's row of the big workload = the cpu_baseline sample
                table[args.workload]["oracle GMG-RBGS (FP64, host)"] = dict(cpu, note="on the sample named")

    steps_tab = step_table(gmg, W, torch, device) if (not args.no_table and rank == 0) else None

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step,
        "ms_per_step_first5": ms_first, "ms_per_step_last5": ms_last, "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{wl.name} {wl.n[0]}x{wl.n[1]}x{wl.n[2]} bc={wl.bc} "
                               "GMG-RBGS V(2,2) nu_coarse=32 tol=1e-4 zero initial guess",
                   "cells": N, "levels": final["levels"], "iterations": iters[-1],
                   "resid_final_rel": final["resid_final_rel"],
                   "uniform_fraction_level0": final["uniform_fraction"],
                   "l2_policy": "inputs larger than L2" if 20 * N > 2 * 126e6 else
                                "inputs fit in L2 (no flush; DRAM roofline not meaningful)",
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "input_generation_s": round(t_gen, 1)},
        "ns_per_cell_per_vcycle": ns_per_cell_vcycle,
        "fixed_10_vcycles": fixed,
        "vcycle": {"ms": vc_ms, "algorithmic_GBs": vcycle_gbs, "frac_of_peak": vcycle_gbs / peak,
                   "bytes_per_fine_cell": vc_bytes / N,
                   "reference_line": {"bytes_per_fine_cell": vc_bytes_ref / N,
                                      "GBs": vc_bytes_ref / (vc_ms * 1e-3) / 1e9,
                                      "note": "SURVEY.md S8(d)'s 134 B/cell minimum with every coefficient loaded; "
                                              "the lean path moves fewer bytes, so this figure may exceed the peak"}},
        "roofline": {"bound": "hbm", "kernel": "level-0 red+black Gauss-Seidel sweep",
                     "achieved": sweep_gbs, "peak": peak, "unit": "GB/s", "frac": sweep_gbs / peak,
                     "traffic": profiled_traffic(args.workload, "sweep"), "peak_source": peak_src,
                     "ms_per_launch": t_sweep, "ms_per_launch_with_norm": t_sweep_norm,
                     "algorithmic_bytes_per_cell": sweep_bytes_cell,
                     "uniform_fraction": f_uni,
                     "reference_line_24B": {"GBs": sweep_gbs_24, "frac": sweep_gbs_24 / peak,
                                            "note": "all three coefficient arrays counted although the lean "
                                                    "path did not move them"},
                     "frac_of_nominal_8TBs": sweep_gbs / 8000.0},
        "roofline_residual_restrict": {"achieved": rr_gbs, "peak": peak, "unit": "GB/s",
                                       "frac": rr_gbs / peak, "ms_per_launch": t_rr,
                                       "traffic": profiled_traffic(args.workload, "residual_restrict"),
                                       "algorithmic_bytes_per_cell": rr_bytes_cell,
                                       "uniform_fraction": f_uni_res,
                                       "reference_line_20.5B_GBs": (20.0 + 4.0 / m) * N / (t_rr * 1e-3) / 1e9},
        "cpu_baseline": cpu,
        "e2e": {"value": e2e_val, "unit": UNIT, "ms_per_step": e2e_ms,
                "h2d_bytes_per_step": 4 * N, "d2h_bytes_per_step": 4 * N,
                "api": "gmg_solve_host_cold (zero initial guess made on the device)"},
        "e2e_guess_uploaded": {"value": replicas.ns_per_cell(e2e_guess_ms, N, world), "unit": UNIT,
                               "ms_per_step": e2e_guess_ms, "h2d_bytes_per_step": 8 * N,
                               "d2h_bytes_per_step": 4 * N, "api": "gmg_solve_host"},
        "gpu_launches": int(launches),
        "clocks": sampler.summary(),
        "around_solve": around,
        "solvers": table,
        "pressure_steps": steps_tab,
        "plan": g.describe_plan().strip().split("\n"),
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4")
    ap.add_argument("--reference-sample", default="c4_256",
                    help="grid of the --impl reference arm (one oracle solve per step)")
    ap.add_argument("--cpu-sample", default="c4_512",
                    help="grid of the cpu_baseline leg of the GPU arm (one oracle solve)")
    ap.add_argument("--no-fixed", action="store_true", help="skip the fixed-10-V-cycles run")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-table", action="store_true", help="skip the solver comparison and pressure-step tables")
    ap.add_argument("--no-graph", action="store_true",
                    help="plain kernel launches instead of the CUDA-graph WHILE loop (so that ncu "
                         "lists every kernel of the solve)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
