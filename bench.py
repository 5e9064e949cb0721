#!/usr/bin/env python
"""bench.py -- headline measurement of the FFT-CG hot path (BASELINE.json metric: CG iterations/s and
site-iterations/s at L=2048; achieved HBM GB/s vs peak).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--dtype f64|f32] [--config 2|4] [--impl fcg|reference]

A "step" is one whole solve of the workload (set-up, CG loop to the configured tolerance, finish) through
the C ABI.  Default workload: BASELINE.json configs[2], L=2048, fp64 (the size the metric is quoted on); the
fp32 run of the same config, the L=8192 fp32 point (configs[4]), the stand-alone transforms and the break step are measured in
the same run and reported under "configs"; --full adds the quasi-static loops and the force formulation under "extra".
Prints ONE JSON line (see DESIGN.md section 7 for every key).
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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC, UNIT = "cg_iterations_per_s", "iter/s"
B_ITER_NW = 16.5          # algorithmic bytes per CG iteration in units of N*w
# this implementation's per-kernel algorithmic bytes / (N*w) (DESIGN.md sections 4 and 12).  Default path (spectral search length):
# three launches, the residual update rides in the last pass and q is never stored; --no-spectral-alpha: four launches.
PASS_NW_SL = {"row_fwd": 6.0, "col": 2.5, "row_inv": 5.0}
PASS_NW_4K = {"row_fwd": 6.0, "col": 2.5, "row_inv": 4.0, "update_r": 3.0}
PASS_NW, PASS_NAMES = PASS_NW_SL, list(PASS_NW_SL)
# preconditioned CG: six kernels per iteration, 22 N*w algorithmic bytes
PCG_NAMES = ["row_fwd", "col", "row_inv", "rupd_row_fwd", "col_precond", "row_inv_precond"]
PCG_NW = {"row_fwd": 6.0, "col": 2.5, "row_inv": 4.0, "rupd_row_fwd": 4.0, "col_precond": 2.5, "row_inv_precond": 3.0}


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu: int):
        self.gpu, self.rows, self.proc = gpu, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i].lower().startswith("active")})
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def oracle_sample(w, iters: int):
    """The oracle as it stands, `iters` CG iterations of workload w (tol = 0) on the host cores."""
    from oracle import api as orc
    t0 = time.perf_counter()
    r = orc.cg(w.s, w.k, w.f, w.u0, 0.0, iters)
    dt = time.perf_counter() - t0
    return r["iters"] / dt, dt, orc.num_threads()


def run_reference(args, rank: int):
    """--impl reference: the CPU oracle on this arm's config, metric and unit (tier contract)."""
    if rank != 0:
        return
    from paper_1305_3625_b200 import inputs
    w = workload_of(inputs, args)
    sample = args.ref_iters
    for _ in range(args.warmup):
        oracle_sample(w, 1)
    total_it, total_t, cores = 0, 0.0, 0
    for _ in range(args.steps):
        v, dt, cores = oracle_sample(w, sample)
        total_it += sample; total_t += dt
    value = total_it / total_t
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total_t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{args.config}] L={w.L} {args.dtype}; each step = {sample} CG iterations (tol=0) of the oracle"},
        "site_iterations_per_s": value * w.N,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{sample} CG iterations per step, tol=0, same seeded workload"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def bench_workload(binding, torch, w, steps, warmup, profile_iters=20, e2e_steps=None, loop_mode=0, pcg_steps=0, inputs_mod=None,
                   solver="cg"):
    """Times `steps` solves of workload w on the current device. Returns a dict of measurements."""
    tdt = torch.float64 if w.dtype == np.float64 else torch.float32
    wbytes = w.dtype.itemsize
    h = binding.Fcg(w.L, tdt)
    h.fcg_set_option(binding.FCG_OPT_LOOP_MODE, loop_mode)
    h.fcg_set_option(binding.FCG_OPT_SPECTRAL_ALPHA, 1 if len(PASS_NAMES) == 3 else 0)
    to = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    h.fcg_set_spectrum(to(w.s))
    k, f, u = to(w.k), to(w.f), to(w.u0)
    solve = h.fcg_solve
    if solver == "pcg":                                    # --solver pcg: the whole bench line is about preconditioned CG
        h.fcg_set_preconditioner(to(w.s), inputs_mod.precond_kbar(w.k))
        solve = h.fcg_pcg_solve
    for _ in range(warmup):
        u.zero_()
        it, rr, st = solve(k, f, u, w.tol, w.maxit)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    iters, launches = [], 0
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for s in range(steps):
        ev[s][0].record()
        u.zero_()                                          # u0 = 0 is part of the workload (otherwise a warm start)
        it, rr, st = solve(k, f, u, w.tol, w.maxit)
        ev[s][1].record()
        iters.append(it); launches += h.fcg_last_launch_count()
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    dev_ms = [a.elapsed_time(b) for a, b in ev]
    out = {"iters": iters, "status": st, "relres": rr, "dev_ms": dev_ms, "wall_s": wall, "launches": launches}
    # the library's automatic choices for this size and dtype (include/fcg.h: fcg_get_option)
    out["options"] = {n: h.fcg_get_option(getattr(binding, "FCG_OPT_" + n)) for n in
                      ("LOOP_MODE", "UNROLL", "PDL", "FUSED", "SPECTRAL_ALPHA", "COL_PERSISTENT", "STAGGER_P1", "STAGGER_P2", "STAGGER_P3")}
    # per-kernel times, in loop order, CUDA events on the library's stream
    u.zero_()
    if solver == "pcg":
        out["kernel_ms"] = dict(zip(PCG_NAMES, h.fcg_profile_pcg_iteration(k, f, u, profile_iters)))
        out["e2e_iter_s"] = None; out["h2d"] = 0; out["d2h"] = 0
        h.close()
        return out
    ms = h.fcg_profile_iteration(k, f, u, profile_iters)
    out["kernel_ms"] = dict(zip(PASS_NAMES, ms))          # (with three launches ms[3] is the empty event pair)
    # end to end with HOST buffers through the C ABI
    # (every step copies its k, f, u up from pinned host memory and its u back down, inside the timed region; the initial guesses
    #  -- one zeroed pinned buffer per step -- are prepared before it.)  Two forms of the same public call: blocking
    #  (fcg_solve_host) and pipelined (fcg_solve_host_submit / _wait: the copies of the neighbouring steps run under the current solve).
    e2e_steps = e2e_steps or max(1, min(steps, 6))
    kh, fh = torch.from_numpy(w.k.copy()).pin_memory(), torch.from_numpy(w.f.copy()).pin_memory()
    uhs = [torch.zeros((w.L, w.L), dtype=tdt).pin_memory() for _ in range(e2e_steps)]
    warm = torch.zeros((w.L, w.L), dtype=tdt).pin_memory()
    h.fcg_solve_host(kh, fh, warm, w.tol, w.maxit)                 # warm (allocates the staging buffers)
    warm.zero_(); h.fcg_solve_host_submit(kh, fh, warm, w.tol, w.maxit); h.fcg_solve_host_wait()
    warm.zero_(); h.fcg_solve_host_submit(kh, fh, warm, w.tol, w.maxit); h.fcg_solve_host_wait()      # (both staging sets)
    torch.cuda.synchronize()
    t0 = time.perf_counter(); e_it = 0
    for i in range(e2e_steps):
        h.fcg_solve_host_submit(kh, fh, uhs[i], w.tol, w.maxit)
        if i > 0:
            e_it += h.fcg_solve_host_wait()[0]
    e_it += h.fcg_solve_host_wait()[0]
    out["e2e_iter_s"] = e_it / (time.perf_counter() - t0)
    out["e2e_solution_norm"] = float(uhs[-1].double().norm())
    nb = min(e2e_steps, 2)
    for x in uhs[:nb]:
        x.zero_()
    t0 = time.perf_counter(); b_it = 0
    for i in range(nb):
        b_it += h.fcg_solve_host(kh, fh, uhs[i], w.tol, w.maxit)[0]
    out["e2e_blocking_iter_s"] = b_it / (time.perf_counter() - t0)
    out["e2e_steps"] = e2e_steps
    out["h2d"] = 3 * w.N * wbytes; out["d2h"] = w.N * wbytes
    if pcg_steps:
        # the same workload solved by preconditioned CG (time to the same tolerance; reported beside the headline, not as it)
        kbar = inputs_mod.precond_kbar(w.k)
        h.fcg_set_preconditioner(to(w.s), kbar)
        for _ in range(2):
            u.zero_(); h.fcg_pcg_solve(k, f, u, w.tol, w.maxit)
        pev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(pcg_steps)]
        for s in range(pcg_steps):
            pev[s][0].record(); u.zero_()
            pit, prr, pst = h.fcg_pcg_solve(k, f, u, w.tol, w.maxit)
            pev[s][1].record()
        torch.cuda.synchronize()
        plaunch = h.fcg_last_launch_count()
        pms = [a.elapsed_time(b) for a, b in pev]
        u.zero_()
        pk = h.fcg_profile_pcg_iteration(k, f, u, profile_iters)
        out["pcg"] = {"kbar": kbar, "iterations": pit, "status": pst, "final_rel_residual": prr, "ms_per_solve": statistics.median(pms),
                      "us_per_iteration": 1e3 * statistics.median(pms) / max(pit, 1),
                      "cg_ms_per_solve": statistics.median(dev_ms), "solve_time_ratio_cg_over_pcg": statistics.median(dev_ms) / statistics.median(pms),
                      "kernel_us": {n: 1e3 * x for n, x in zip(PCG_NAMES, pk)},
                      "kernel_gbs": {n: PCG_NW[n] * w.N * wbytes / (x * 1e-3) / 1e9 for n, x in zip(PCG_NAMES, pk)},
                      "bytes_per_iteration": sum(PCG_NW.values()) * w.N * wbytes,
                      "iteration_gbs": sum(PCG_NW.values()) * w.N * wbytes / (statistics.median(pms) * 1e-3 / max(pit, 1)) / 1e9,
                      "launches_per_solve": plaunch}
    h.close()
    return out


def bench_extras(binding, torch, inputs):
    """--full: the quasi-static loop of configs[3] (all 2000 steps, CG and PCG solves, and ensembles; latency-bound: us per CG
    iteration and break steps per second are the figures) and the force formulation (bench_force)."""
    out = {}
    to = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    # quasi-static loop of configs[3], all 2000 steps in one cooperative launch: CG solves, PCG solves, and an ensemble of
    # independent samples (different threshold seeds) on several streams through fcg_fracture_begin / _end
    w3 = inputs.config(3)
    for name, pcg in (("fracture_cfg3", False), ("fracture_cfg3_pcg", True)):
        h = binding.Fcg(w3.L, torch.float64); s3 = to(w3.s); h.fcg_set_spectrum(s3)
        if pcg:
            h.fcg_set_preconditioner(s3, 1.0)
        best = None
        for rep in range(2):
            k, f, u, t = to(w3.k), to(w3.f), to(w3.u0), to(w3.t)
            torch.cuda.synchronize(); t0 = time.perf_counter()
            index, iters, done, st = (h.fcg_pcg_fracture if pcg else h.fcg_fracture)(k, f, u, t, w3.nsteps, w3.tol, w3.maxit)
            dt_s = time.perf_counter() - t0
            best = dt_s if best is None else min(best, dt_s)
        out[name] = {"steps": int(done), "iterations": int(iters.sum()), "wall_s": best, "steps_per_s": int(done) / best,
                     "us_per_iteration": 1e6 * best / max(int(iters.sum()), 1), "status": int(st), "launches": h.fcg_last_launch_count()}
        h.close()
    for nrep in (2, 4, 6):
        reps = []
        for r in range(nrep):
            stream = torch.cuda.Stream()
            with torch.cuda.stream(stream):
                h = binding.Fcg(w3.L, torch.float64, stream=stream); s3 = to(w3.s); h.fcg_set_spectrum(s3); h.fcg_set_preconditioner(s3, 1.0)
                reps.append((h, to(w3.k), to(w3.f), to(w3.u0), to(inputs.thresholds(w3.L, seed=100 + r))))
        torch.cuda.synchronize(); t0 = time.perf_counter()
        for h, k, f, u, t in reps:
            h.fcg_fracture_begin(k, f, u, t, w3.nsteps, w3.tol, w3.maxit, True)
        res = [h.fcg_fracture_end() for h, *_ in reps]
        dt_s = time.perf_counter() - t0
        out[f"fracture_cfg3_pcg_ensemble{nrep}"] = {"samples": nrep, "steps": sum(int(r[2]) for r in res), "wall_s": dt_s,
                                                    "steps_per_s": sum(int(r[2]) for r in res) / dt_s,
                                                    "iterations": sum(int(r[1].sum()) for r in res)}
        for h, *_ in reps:
            h.close()
    out.update(bench_force(binding, torch, inputs))
    return out


def bench_force(binding, torch, inputs):
    """The paper's own formulation in the bond forces: the static chain
    eq. (1c) -> g = Re F G on the device, CG on (I + K G) f = K D at L = 2048 (one bond in 20 broken, tol 1e-12 fp64 / 1e-5 fp32),
    and the quasi-static loop in the forces at L = 256 (threshold gradient 1.0, 500 break steps)."""
    out = {}
    to = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    for L, dt, tdt, name in ((2048, np.float64, torch.float64, "f64"), (2048, np.float32, torch.float32, "f32")):
        h = binding.Fcg(L, tdt)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        G = h.fcg_green_function(inputs.GREEN_NU, inputs.GREEN_E, inputs.GREEN_A); g = h.fcg_kernel_spectrum(G)     # warm
        torch.cuda.synchronize()
        ev[0].record(); h.fcg_green_function(inputs.GREEN_NU, inputs.GREEN_E, inputs.GREEN_A, G)
        ev[1].record(); h.fcg_kernel_spectrum(G, g)
        ev[2].record(); torch.cuda.synchronize()
        h.fcg_set_spectrum(g)
        k = to(inputs.force_k(L, 20).astype(dt)); f = torch.zeros((L, L), dtype=tdt, device="cuda")
        tol = inputs.FORCE_TOL[np.dtype(dt)]
        for _ in range(2):
            f.zero_(); h.fcg_force_solve(k, inputs.FORCE_D, f, tol, 2000)
        reps = 5
        sev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
        for a, b in sev:
            f.zero_(); a.record()
            it, rr, st = h.fcg_force_solve(k, inputs.FORCE_D, f, tol, 2000)
            b.record()
        torch.cuda.synchronize()
        ms = statistics.median(a.elapsed_time(b) for a, b in sev)
        nw = L * L * np.dtype(dt).itemsize
        launches = h.fcg_last_launch_count()
        per_it = round((launches - 4) / max(it, 1))      # the set-up (residual pass) and finish kernels are not per-iteration
        b_nw = 13.5 if per_it == 3 else 15.5             # DESIGN.md sections 4, 12: three launches never store q
        out[f"force_solve_L{L}_{name}"] = {
            "iterations": it, "status": st, "final_rel_residual": rr, "ms_per_solve": ms, "us_per_iteration": 1e3 * ms / max(it, 1),
            "launches_per_solve": launches, "launches_per_iteration": per_it,
            "iteration_gbs": b_nw * nw / (1e-3 * ms / max(it, 1)) / 1e9, "bytes_per_iteration_Nw": b_nw,
            "green_function_us": 1e3 * ev[0].elapsed_time(ev[1]), "kernel_spectrum_us": 1e3 * ev[1].elapsed_time(ev[2])}
        h.close()
    # the same forces through the displacements (reading F7): (K + G^-1) u = K D by fcg_solve / fcg_pcg_solve with s = 1/g, then (1a)
    L = 2048
    h = binding.Fcg(L, torch.float64)
    s = h.fcg_inverse_spectrum(h.fcg_kernel_spectrum(h.fcg_green_function(inputs.GREEN_NU, inputs.GREEN_E, inputs.GREEN_A)))
    h.fcg_set_spectrum(s)
    kh = inputs.force_k(L, 20); k = to(kh)
    h.fcg_set_preconditioner(s, inputs.precond_kbar(kh))
    u = torch.zeros((L, L), dtype=torch.float64, device="cuda"); f = torch.empty_like(u); b = torch.empty_like(u)
    for name, solve in (("cg", h.fcg_solve), ("pcg", h.fcg_pcg_solve)):
        for _ in range(2):
            u.zero_(); h.fcg_force_rhs(k, inputs.FORCE_D, b); solve(k, b, u, 1e-12, 2000); h.fcg_force_from_displacement(k, inputs.FORCE_D, u, f)
        sev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(5)]
        for a, c in sev:
            u.zero_(); a.record()
            h.fcg_force_rhs(k, inputs.FORCE_D, b); it, rr, st = solve(k, b, u, 1e-12, 2000); h.fcg_force_from_displacement(k, inputs.FORCE_D, u, f)
            c.record()
        torch.cuda.synchronize()
        ms = statistics.median(a.elapsed_time(c) for a, c in sev)
        out[f"force_via_displacement_{name}_L2048_f64"] = {
            "iterations": it, "status": st, "final_rel_residual": rr, "ms_per_solve": ms,
            "speedup_over_force_solve": out["force_solve_L2048_f64"]["ms_per_solve"] / ms,
            "note": "b = K D, (K + G^-1) u = b to 1e-12, f = -k (u - D); same forces as force_solve_L2048_f64 to ~1e-10 (tests)"}
    h.close()
    L, nsteps = 256, 500
    h = binding.Fcg(L, torch.float64)
    h.fcg_set_spectrum(h.fcg_kernel_spectrum(h.fcg_green_function(inputs.GREEN_NU, inputs.GREEN_E, inputs.GREEN_A)))
    t = to(inputs.gradient_thresholds(L, 1.0))
    best = None
    for rep in range(2):
        k = to(inputs.force_k(L)); f = torch.zeros((L, L), dtype=torch.float64, device="cuda")
        torch.cuda.synchronize(); t0 = time.perf_counter()
        index, iters, ratio, done, st = h.fcg_force_fracture(k, inputs.FORCE_D, f, t, nsteps, 1e-12, 1000)
        dt_s = time.perf_counter() - t0
        best = dt_s if best is None else min(best, dt_s)
    eq2_wall, eq2_steps = best, int(done)
    out["force_fracture_L256_f64"] = {"steps": int(done), "iterations": int(iters.sum()), "wall_s": best, "steps_per_s": int(done) / best,
                                      "us_per_iteration": 1e6 * best / max(int(iters.sum()), 1), "status": int(st),
                                      "launches": h.fcg_last_launch_count()}
    h.close()
    # the same loop through the displacements (reading F7), CG and PCG solves: same break sequence (tests), a fraction of the iterations
    for name, pcg in (("cg", False), ("pcg", True)):
        h = binding.Fcg(L, torch.float64)
        s = h.fcg_inverse_spectrum(h.fcg_kernel_spectrum(h.fcg_green_function(inputs.GREEN_NU, inputs.GREEN_E, inputs.GREEN_A)))
        h.fcg_set_spectrum(s)
        if pcg:
            h.fcg_set_preconditioner(s, 1.0)
        best = None
        for rep in range(2):
            k = to(inputs.force_k(L)); u = torch.zeros((L, L), dtype=torch.float64, device="cuda")
            torch.cuda.synchronize(); t0 = time.perf_counter()
            index, iters, ratio, done, st = h.fcg_force_fracture_displacement(k, inputs.FORCE_D, u, t, nsteps, 1e-12, 2000, use_pcg=pcg)
            dt_s = time.perf_counter() - t0
            best = dt_s if best is None else min(best, dt_s)
        out[f"force_fracture_via_displacement_{name}_L256_f64"] = {
            "steps": int(done), "iterations": int(iters.sum()), "wall_s": best, "steps_per_s": int(done) / best,
            "us_per_iteration": 1e6 * best / max(int(iters.sum()), 1), "status": int(st), "launches": h.fcg_last_launch_count(),
            "speedup_over_force_fracture": (eq2_wall / max(eq2_steps, 1)) / (best / max(int(done), 1))}
        h.close()
    # ensembles of independent samples (different threshold seeds) of that loop, PCG solves, several streams from one host thread
    for nrep in (2, 4, 6):
        reps = []
        for r in range(nrep):
            stream = torch.cuda.Stream()
            with torch.cuda.stream(stream):
                h = binding.Fcg(L, torch.float64, stream=stream)
                s = h.fcg_inverse_spectrum(h.fcg_kernel_spectrum(h.fcg_green_function(inputs.GREEN_NU, inputs.GREEN_E, inputs.GREEN_A)))
                h.fcg_set_spectrum(s); h.fcg_set_preconditioner(s, 1.0)
                reps.append((h, to(inputs.force_k(L)), torch.zeros((L, L), dtype=torch.float64, device="cuda"),
                             to(inputs.gradient_thresholds(L, 1.0, seed=300 + r))))
        torch.cuda.synchronize(); t0 = time.perf_counter()
        for h, k, u, tt in reps:
            h.fcg_force_fracture_displacement_begin(k, inputs.FORCE_D, u, tt, nsteps, 1e-12, 2000, True)
        res = [h.fcg_force_fracture_displacement_end() for h, *_ in reps]
        dt_s = time.perf_counter() - t0
        out[f"force_fracture_via_displacement_pcg_ensemble{nrep}_L256_f64"] = {
            "samples": nrep, "steps": sum(int(r[3]) for r in res), "wall_s": dt_s, "steps_per_s": sum(int(r[3]) for r in res) / dt_s,
            "iterations": sum(int(r[1].sum()) for r in res)}
        for h, *_ in reps:
            h.close()
    return out


def moved_nw():
    """Bytes one CG iteration of this implementation moves, in units of N*w (DESIGN.md sections 4, 12)."""
    return sum(PASS_NW.values())


def bench_configs(binding, torch, inputs, hbm_peak):
    """Default run, beside the headline: the other numbers north_star asks for, each measured here in a few solves / calls --
    configs[2] in fp32, configs[4] (L = 8192 fp32, the HBM-bound point), the stand-alone transforms (GB/s on 4 N w bytes per
    transform) and the break step (3 N w bytes).  Fractions are of the measured copy peak and of 8 TB/s nominal, on the bytes the
    implementation moves (13.5 N w per iteration); the 16.5 N w survey model is given beside them as an equivalent rate."""
    out = {}
    to = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    for cfg, dt in ((2, np.float32), (4, np.float32)):
        w2 = inputs.config(cfg, dt)
        r2 = bench_workload(binding, torch, w2, 2, 1, profile_iters=10, e2e_steps=1)
        nw2 = w2.N * w2.dtype.itemsize
        t2 = 1e3 * (sum(r2["dev_ms"]) / len(r2["dev_ms"])) / r2["iters"][0]
        gbs = moved_nw() * nw2 / (t2 * 1e-6) / 1e9
        out[f"cfg{cfg}_L{w2.L}_f32"] = {
            "iterations": r2["iters"][0], "status": r2["status"], "final_rel_residual": r2["relres"], "us_per_iteration": t2,
            "iter_per_s": 1e6 / t2, "site_iter_per_s": 1e6 / t2 * w2.N,
            "bytes_moved_per_iteration": moved_nw() * nw2, "iteration_gbs": gbs, "frac_of_measured_peak": gbs / hbm_peak,
            "frac_of_8TBs_nominal": gbs / 8000.0, "equivalent_gbs_16p5_model": B_ITER_NW * nw2 / (t2 * 1e-6) / 1e9,
            "kernel_us": {n: 1e3 * r2["kernel_ms"][n] for n in PASS_NAMES},
            "kernel_gbs": {n: PASS_NW[n] * nw2 / (r2["kernel_ms"][n] * 1e-3) / 1e9 for n in PASS_NAMES},
            "e2e_iter_per_s": r2["e2e_iter_s"]}
        del w2, r2
    for L, dt, tdt in ((2048, np.float64, torch.float64), (8192, np.float32, torch.float32)):
        name = "f64" if dt == np.float64 else "f32"
        nw = L * L * np.dtype(dt).itemsize
        h = binding.Fcg(L, tdt)
        x = to(inputs.fft_field(L).astype(dt))
        X = h.fcg_fft_fwd(x); xb = h.fcg_fft_inv(X)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        torch.cuda.synchronize()
        reps = 10
        ev[0].record()
        for _ in range(reps): h.fcg_fft_fwd(x, X)
        ev[1].record()
        for _ in range(reps): h.fcg_fft_inv(X, xb)
        ev[2].record(); torch.cuda.synchronize()
        tf, ti = ev[0].elapsed_time(ev[1]) / reps, ev[1].elapsed_time(ev[2]) / reps
        out[f"fft_L{L}_{name}"] = {"fwd_us": 1e3 * tf, "inv_us": 1e3 * ti, "fwd_gbs": 4 * nw / (tf * 1e-3) / 1e9, "inv_gbs": 4 * nw / (ti * 1e-3) / 1e9,
                                   "fwd_frac_of_measured_peak": 4 * nw / (tf * 1e-3) / 1e9 / hbm_peak,
                                   "inv_frac_of_measured_peak": 4 * nw / (ti * 1e-3) / 1e9 / hbm_peak,
                                   "round_trip_rel_l2": float((xb - x).norm() / x.norm()), "bytes_per_transform": 4 * nw}
        # break step on the same handle: k, u, t resident; each call = one kernel + a 16-byte read-back and a stream sync
        k = to((0.5 + np.random.default_rng(0).random((L, L))).astype(dt)); t = to(inputs.thresholds(L).astype(dt))
        h.fcg_break_step(k, x, t)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); t0 = time.perf_counter(); e0.record()
        for _ in range(10): h.fcg_break_step(k, x, t)
        e1.record(); torch.cuda.synchronize()
        us = 1e3 * e0.elapsed_time(e1) / 10
        # the same kernel through the allocation-free, asynchronous entry point (no read-back, no host sync): its device time
        res = torch.zeros(3, dtype=torch.int64, device="cuda")
        binding.fcg_break_step_static(k, x, t, res)
        torch.cuda.synchronize(); e0.record()
        for _ in range(10): binding.fcg_break_step_static(k, x, t, res)
        e1.record(); torch.cuda.synchronize()
        dus = 1e3 * e0.elapsed_time(e1) / 10
        out[f"break_step_L{L}_{name}"] = {"us_per_call": us, "device_us": dus, "bytes": 3 * nw, "gbs": 3 * nw / (dus * 1e-6) / 1e9,
                                          "frac_of_measured_peak": 3 * nw / (dus * 1e-6) / 1e9 / hbm_peak,
                                          "note": "us_per_call: 10 blocking fcg_break_step calls (kernel + 16-byte read-back + host sync each); device_us, gbs, "
                                                  "frac: 10 back-to-back fcg_break_step_static calls (4-byte memset + the same kernel, no host sync)"}
        h.close()
        del x, X, xb, k, t
    torch.cuda.empty_cache()
    return out


def iteration_roofline(nw, t_iter_us, hbm_peak, peak_src, dram_iter):
    """Whole iteration against the HBM roofline, on the bytes this implementation MOVES (13.5 N w with three launches, 15.5 with
    four; DESIGN.md sections 4 and 12).  The 16.5 N w of SURVEY.md 8(d) -- the count for a design that stores and re-reads q -- is
    kept beside it as an equivalent rate, labelled; dram_* are the bytes that really reach DRAM per iteration with warm caches
    (single-pass ncu capture under profiles/), which at L = 2048 is well below the bytes moved because L2 serves T2."""
    moved = moved_nw() * nw
    ach = moved / (t_iter_us * 1e-6) / 1e9
    eq = B_ITER_NW * nw / (t_iter_us * 1e-6) / 1e9
    d = {"bound": "hbm", "bytes_per_iteration": moved, "bytes_per_iteration_Nw": moved_nw(), "achieved": ach, "peak": hbm_peak, "unit": "GB/s",
         "frac": ach / hbm_peak, "frac_of_8TBs_nominal": ach / 8000.0, "peak_source": peak_src,
         "floor_us_at_measured_peak": moved / (hbm_peak * 1e9) * 1e6,
         "survey_model_16p5": {"bytes_per_iteration": B_ITER_NW * nw, "equivalent_gbs": eq, "frac": eq / hbm_peak, "frac_of_8TBs_nominal": eq / 8000.0,
                               "note": "SURVEY.md 8(d) counts 16.5 N w for a design that stores q and reads p twice; this one does not, so this is an "
                                       "equivalent rate, not bytes moved"},
         "note": "time = whole solve / iterations (set-up and finish included)"}
    if dram_iter is not None:
        d["dram_bytes_per_iteration_warm"] = dram_iter
        d["dram_gbs"] = dram_iter / (t_iter_us * 1e-6) / 1e9
        d["dram_frac"] = d["dram_gbs"] / hbm_peak
    return d


def workload_of(inputs, args):
    """BASELINE.json configs[args.config] in args.dtype; --L: the same recipe at another lattice size (a parity-test case of the
    suite, e.g. L = 1024, the largest size of the paper -- never the headline: the JSON line's workload string says so)."""
    dt = np.float64 if args.dtype == "f64" else np.float32
    return inputs.config(args.config, dt) if args.L is None else inputs.config(args.config, dt, L=args.L)


def run_slab(args, rank, world, local):
    """--shard slab: ONE solve spread over the ranks by rows instead of one
    replica per rank.  Under torchrun every process is one rank (DistComm: NCCL all-to-all of the half spectrum around the column
    pass, all-reduce of the two scalars); with one process, --slab-ranks G runs G LOGICAL ranks on the one device (LocalComm:
    device copies), which exercises the same kernels and orchestration but measures nothing about scaling."""
    import torch
    import torch.distributed as dist
    from paper_1305_3625_b200 import binding, inputs, slab
    torch.cuda.set_device(local)
    tdt = torch.float64 if args.dtype == "f64" else torch.float32
    w = workload_of(inputs, args)
    to = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        comm, G, mine = slab.DistComm(), world, [rank]
    else:
        comm, G, mine = slab.LocalComm(), args.slab_ranks, list(range(args.slab_ranks))
    sd = to(w.s)
    spectral = args.slab_order == "spectral"
    graph = {"auto": None, "on": True, "off": False}[args.slab_graph]
    ranks = [slab.SlabRank(w.L, tdt, G, g, sd) for g in mine]
    if args.slab_peers:          # the exchange fused into the passes: peer stores instead of all-to-alls
        if world > 1:
            slab.connect_peers_dist(ranks[0], comm)
        else:
            slab.connect_peers_local(ranks)
    k = [to(w.k[r.rows]) for r in ranks]; f = [to(w.f[r.rows]) for r in ranks]
    u = [torch.zeros_like(x) for x in k]
    sampler = ClockSampler(local) if rank == 0 else None
    for _ in range(args.warmup):
        for x in u: x.zero_()
        it, rr, st = slab.slab_solve(ranks, comm, k, f, u, w.tol, w.maxit, spectral=spectral, graph=graph)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    if sampler:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    its, launches = 0, 0
    e0.record()
    for _ in range(args.steps):
        for x in u: x.zero_()
        it, rr, st = slab.slab_solve(ranks, comm, k, f, u, w.tol, w.maxit, spectral=spectral, graph=graph)
        its += it; launches += sum(slab.launch_count(r) for r in ranks)
    e1.record(); torch.cuda.synchronize()
    clocks = sampler.stop() if sampler else None
    ms = e0.elapsed_time(e1)
    if world > 1:                                            # one job: time = max over ranks, work = the iterations of the one solve
        t = torch.tensor([ms], dtype=torch.float64, device="cuda"); dist.all_reduce(t, op=dist.ReduceOp.MAX); ms = float(t.item())
        c = torch.tensor([float(launches)], dtype=torch.float64, device="cuda"); dist.all_reduce(c); launches = int(c.item())
    if rank == 0:
        nw = w.N * w.dtype.itemsize
        t_iter_us = 1e3 * ms / max(its, 1)
        print(json.dumps({
            "metric": METRIC, "value": its / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": args.dtype,
            "data": "synthetic",
            "config": {"workload": f"BASELINE.json configs[{args.config}]: L={w.L} {args.dtype}, ONE solve split by rows over {G} "
                                   f"{'ranks (one per GPU, NCCL)' if world > 1 else 'LOGICAL ranks on one device (device copies)'}, tol={w.tol:g} ({it} iterations)",
                       "parallelism": f"slab x{G}" + (" peer mode" if args.slab_peers else ""), "launches_per_iteration_per_rank": "3 passes + 3 one-block kernels" if spectral else "4 passes + 2 one-block kernels",
                       "collectives_per_iteration": ("2 barriers" if args.slab_peers else "2 all-to-all (N w / G bytes per rank each)") + " + 2 all-reduce (32 B)",
                       "note": ("spectral search length (three passes)" if spectral else "textbook order (four passes)") +
                               ", host poll every eighth iteration" + ("" if graph is False or (graph is None and world > 1) else ", blocks of eight iterations replayed from a CUDA graph") + "; the hardware scaling curve is unmeasured on this one-GPU pool"},
            "site_iterations_per_s": its / (ms * 1e-3) * w.N, "us_per_iteration": t_iter_us,
            "exchange_bytes_per_iteration_per_rank": 2.0 * nw / G * (G - 1) / G,
            "gpu_launches": launches, "clocks": clocks, "final_rel_residual": rr, "status": st}))
    for r in ranks:
        r.close()
    if world > 1:
        dist.destroy_process_group()


def aggregate_over_ranks(dist, torch, step_ms, total_it, launches, e2e_iter_s, device):
    """Replicas only: whole-job time = MAX over ranks of the device time, whole-job work = SUM over ranks.
    `dist` is torch.distributed with an initialised group (nccl on the GPU box, gloo in the CPU test) or None for one rank."""
    if dist is None:
        return float(step_ms), int(total_it), int(launches), float(e2e_iter_s)
    t = torch.tensor([step_ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor([total_it, launches, e2e_iter_s], dtype=torch.float64, device=device)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), int(round(c[0].item())), int(round(c[1].item())), float(c[2].item())


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--dtype", choices=["f64", "f32"], default="f64")
    ap.add_argument("--config", type=int, default=2, choices=[0, 1, 2, 4])
    ap.add_argument("--L", type=int, default=None, choices=[256, 512, 1024, 2048, 4096, 8192],
                    help="the config's recipe at another lattice size (default: the config's own L)")
    ap.add_argument("--impl", choices=["fcg", "reference"], default="fcg")
    ap.add_argument("--ref-iters", type=int, default=8, help="oracle CG iterations per step of --impl reference")
    ap.add_argument("--cpu-baseline-iters", type=int, default=None,
                    help="oracle CG iterations of the cpu_baseline sample (default: sized for ~12 s of host work from a 2-iteration probe)")
    ap.add_argument("--full", action="store_true", help="also time configs[2] fp32 and configs[4] (reported under 'extra')")
    ap.add_argument("--solver", choices=["cg", "pcg", "force"], default="cg",
                    help="pcg: time fcg_pcg_solve instead (metric pcg_iterations_per_s, 22 N w bytes per iteration; no e2e leg) -- "
                         "for profiling the PCG kernels; the headline BASELINE.json names is the default")
    ap.add_argument("--shard", choices=["replicas", "slab"], default="replicas",
                    help="N > 1: replicas (default; one independent solve per GPU, no data-path collective) or slab (ONE solve split by rows "
                         "over the ranks: all-to-all transposes around the column pass, all-reduce of the scalars; DESIGN.md section 18)")
    ap.add_argument("--slab-order", choices=["spectral", "textbook"], default="spectral",
                    help="--shard slab: the iteration with the spectral search length (three passes per iteration, default) or in the textbook order (four)")
    ap.add_argument("--slab-graph", choices=["auto", "on", "off"], default="auto",
                    help="--shard slab: replay blocks of iterations from a CUDA graph (auto: on for logical ranks, off under torchrun)")
    ap.add_argument("--slab-peers", action="store_true",
                    help="--shard slab: peer mode -- the row pass stores straight into the owning rank's exchange buffer and the column pass "
                         "scatters straight into the source ranks' T2 (CUDA IPC mappings over NVLink under torchrun); barriers replace the all-to-alls")
    ap.add_argument("--slab-ranks", type=int, default=4, help="--shard slab with one process: number of LOGICAL ranks on the one device")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="skip the 'configs' block (configs[2] fp32, configs[4], transforms, break step)")
    ap.add_argument("--no-spectral-alpha", action="store_true",
                    help="four launches per iteration: p.Ap as a dot product after the last pass + a residual-update kernel")
    ap.add_argument("--no-pcg", action="store_true", help="skip the preconditioned-CG time-to-solution of the same workload ('pcg' key)")
    ap.add_argument("--loop-mode", type=int, default=0, choices=[0, 1],
                    help="0: whole solve as one CUDA graph with a device-side WHILE node (default); 1: direct launches (for ncu)")
    args = ap.parse_args()

    global PASS_NW, PASS_NAMES
    if args.no_spectral_alpha:
        PASS_NW, PASS_NAMES = PASS_NW_4K, list(PASS_NW_4K)
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.shard == "slab":
        run_slab(args, rank, world, local)
        return

    import torch
    import torch.distributed as dist
    from paper_1305_3625_b200 import binding, inputs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    w = workload_of(inputs, args)
    wbytes = w.dtype.itemsize
    hbm_peak, peak_src = peaks()

    sampler = ClockSampler(local) if rank == 0 else None
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    if sampler:
        sampler.start()
    res = None
    if args.solver != "force":
        res = bench_workload(binding, torch, w, args.steps, args.warmup, loop_mode=args.loop_mode, solver=args.solver, inputs_mod=inputs)
        clocks = sampler.stop() if sampler else None
    if args.solver == "force":
        # profiling mode for the force formulation: CG on (I + K G) f = K D at L = 2048, one bond in 20 broken
        if world > 1:
            raise SystemExit("--solver force is a single-GPU profiling mode")
        tdt = torch.float64 if args.dtype == "f64" else torch.float32
        L = 2048
        h = binding.Fcg(L, tdt)
        h.fcg_set_option(binding.FCG_OPT_LOOP_MODE, args.loop_mode)
        h.fcg_set_spectrum(h.fcg_kernel_spectrum(h.fcg_green_function(inputs.GREEN_NU, inputs.GREEN_E, inputs.GREEN_A)))
        k = torch.from_numpy(inputs.force_k(L, 20).astype(w.dtype)).cuda(); f = torch.zeros((L, L), dtype=tdt, device="cuda")
        tol = inputs.FORCE_TOL[np.dtype(w.dtype)]
        for _ in range(args.warmup):
            f.zero_(); h.fcg_force_solve(k, inputs.FORCE_D, f, tol, 2000)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        its, launches = 0, 0
        for a, b in ev:
            f.zero_(); a.record()
            it, rr, st = h.fcg_force_solve(k, inputs.FORCE_D, f, tol, 2000)
            b.record(); its += it; launches += h.fcg_last_launch_count()
        torch.cuda.synchronize()
        clocks = sampler.stop() if sampler else None
        ms = sum(a.elapsed_time(b) for a, b in ev)
        nw = L * L * wbytes
        per_it = h.fcg_last_launch_count() // max(it, 1)
        b_iter = 13.5 if per_it == 3 else 15.5
        t_iter_us = 1e3 * ms / max(its, 1)
        ach = b_iter * nw / (t_iter_us * 1e-6) / 1e9
        print(json.dumps({
            "metric": "force_cg_iterations_per_s", "value": its / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": args.dtype, "data": "synthetic",
            "config": {"workload": f"force formulation (I + K G) f = K D, L={L} {args.dtype}, 1/20 of the bonds broken, tol={tol:g} ({it} iterations)",
                       "launches_per_iteration": per_it},
            "us_per_iteration": t_iter_us,
            "roofline": {"bound": "hbm", "kernel": "whole iteration", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak,
                         "traffic": None, "algorithmic_bytes_per_launch": b_iter * nw, "peak_source": peak_src},
            "gpu_launches": launches, "clocks": clocks, "final_rel_residual": rr, "status": st}))
        h.close()
        return
    if args.solver == "pcg":
        if world > 1:
            raise SystemExit("--solver pcg is a single-GPU profiling mode")
        names, nws, b_iter = PCG_NAMES, PCG_NW, sum(PCG_NW.values())
        kms = res["kernel_ms"]; nw = w.N * wbytes; it0 = res["iters"][0]
        t_iter_us = 1e3 * (sum(res["dev_ms"]) / len(res["dev_ms"])) / max(it0, 1)
        dom = max(names, key=lambda n: kms[n])
        ach = nws[dom] * nw / (kms[dom] * 1e-3) / 1e9
        print(json.dumps({
            "metric": "pcg_iterations_per_s", "value": sum(res["iters"]) / (sum(res["dev_ms"]) * 1e-3), "unit": UNIT, "n_gpus": 1,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": sum(res["dev_ms"]) / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
            "config": {"workload": f"BASELINE.json configs[{args.config}] L={w.L} {args.dtype} solved by preconditioned CG ({it0} iterations)"},
            "us_per_iteration": t_iter_us, "kernel_us": {n: 1e3 * kms[n] for n in names},
            "kernel_gbs": {n: nws[n] * nw / (kms[n] * 1e-3) / 1e9 for n in names},
            "iteration_roofline": {"bound": "hbm", "bytes_per_iteration": b_iter * nw, "achieved": b_iter * nw / (t_iter_us * 1e-6) / 1e9,
                                   "peak": hbm_peak, "unit": "GB/s", "frac": b_iter * nw / (t_iter_us * 1e-6) / 1e9 / hbm_peak},
            "roofline": {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak, "traffic": None},
            "gpu_launches": res["launches"], "clocks": clocks, "final_rel_residual": res["relres"], "status": res["status"]}))
        return
    if rank == 0 and world == 1 and not args.no_pcg and args.loop_mode == 0:      # outside the timed region of the headline
        res["pcg"] = bench_workload(binding, torch, w, 3, 1, loop_mode=0, pcg_steps=5, inputs_mod=inputs, e2e_steps=1)["pcg"]

    # replicas only: every rank solves its own copy; time = max over ranks, value = sum of work
    step_ms, total_it, launches, res["e2e_iter_s"] = aggregate_over_ranks(
        dist if world > 1 else None, torch, sum(res["dev_ms"]), sum(res["iters"]), res["launches"], res["e2e_iter_s"], "cuda")
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    value = total_it / (step_ms * 1e-3)
    it_per_solve = res["iters"][0]
    t_iter_us = 1e3 * (sum(res["dev_ms"]) / len(res["dev_ms"])) / max(it_per_solve, 1)     # whole solve / iterations (incl. set-up, finish)
    nw = w.N * wbytes
    kms = res["kernel_ms"]
    dom = max(PASS_NAMES, key=lambda n: kms[n])
    achieved = PASS_NW[dom] * nw / (kms[dom] * 1e-3) / 1e9
    traffic = traffic_warm = None
    tj = {}
    tpath = os.path.join(ROOT, "profiles", "traffic.json")          # dram bytes per launch from the committed ncu --set full capture
    if os.path.exists(tpath):
        try:
            tj = json.load(open(tpath))
            traffic = tj.get(f"L{w.L}_{args.dtype}", {}).get(dom)     # cold-cache figure (profiles/r1_notes.md)
            traffic_warm = tj.get(f"warm_L{w.L}_{args.dtype}", {}).get(dom)   # single-pass capture with warm caches (profiles/r1_warm_traffic.md)
        except Exception:
            traffic = traffic_warm = None
    dram_iter = None                                                   # dram bytes per steady-state iteration (warm caches), all kernels
    try:
        tw = tj.get(f"warm_L{w.L}_{args.dtype}", {})
        if all(n in tw for n in PASS_NAMES):
            dram_iter = float(sum(tw[n] for n in PASS_NAMES))
    except Exception:
        dram_iter = None
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": step_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": args.dtype, "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{args.config}]{'' if args.L is None else ' recipe at another size'}: L={w.L} {args.dtype}, tol={w.tol:g}, one step = one full CG solve from u0=0 "
                               f"({it_per_solve} iterations)", "L": w.L, "iterations_per_solve": it_per_solve,
                   "l2_policy": f"inputs larger than L2: working set {7.5 * nw / 2**20:.0f} MiB per solve vs 126 MB L2; no flush",
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "launches_per_iteration": len(PASS_NAMES), "library_options": res.get("options")},
        "site_iterations_per_s": value * w.N,
        "us_per_iteration": t_iter_us,
        "iteration_roofline": iteration_roofline(nw, t_iter_us, hbm_peak, peak_src, dram_iter),
        "kernel_us": {n: 1e3 * kms[n] for n in PASS_NAMES},
        "kernel_gbs": {n: PASS_NW[n] * nw / (kms[n] * 1e-3) / 1e9 for n in PASS_NAMES},
        "roofline": {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": hbm_peak, "unit": "GB/s", "frac": achieved / hbm_peak,
                     "frac_of_8TBs_nominal": achieved / 8000.0,
                     "traffic": traffic, "traffic_warm_caches": traffic_warm, "algorithmic_bytes_per_launch": PASS_NW[dom] * nw, "peak_source": peak_src,
                     # the first and the fused last pass are within a few per cent of each other: all three loop kernels, same definition
                     "all_kernels": {n: {"us": 1e3 * kms[n], "achieved": PASS_NW[n] * nw / (kms[n] * 1e-3) / 1e9,
                                         "frac": PASS_NW[n] * nw / (kms[n] * 1e-3) / 1e9 / hbm_peak} for n in PASS_NAMES}},
        "e2e": {"value": res["e2e_iter_s"], "unit": UNIT, "h2d_bytes_per_step": res["h2d"], "d2h_bytes_per_step": res["d2h"],
                "call": "fcg_solve_host_submit / fcg_solve_host_wait (pinned host buffers, two solves in flight: the copies of step i+1 and "
                        "i-1 run under solve i)", "steps": res.get("e2e_steps"),
                "blocking_call_value": res.get("e2e_blocking_iter_s"), "blocking_call": "fcg_solve_host"},
        "gpu_launches": launches,
        "clocks": clocks,
        "final_rel_residual": res["relres"], "status": res["status"],
    }
    if "pcg" in res:
        line["pcg"] = res["pcg"]
    if world == 1 and not args.no_configs and args.config == 2 and args.dtype == "f64" and args.loop_mode == 0 and args.L is None:
        line["configs"] = bench_configs(binding, torch, inputs, hbm_peak)          # outside the timed region of the headline
    if args.full and world == 1:
        line["extra"] = bench_extras(binding, torch, inputs)
    if not args.no_cpu_baseline and world == 1:
        n_cpu = args.cpu_baseline_iters
        if n_cpu is None:                                  # bounded sample: about 12 s of host work, at least 8 iterations
            v0, _, _ = oracle_sample(w, 2)
            n_cpu = int(min(max(8, round(12.0 * v0)), 4000))
        v, dt, cores = oracle_sample(w, n_cpu)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"{n_cpu} CG iterations (tol=0) of the same workload from u0, {dt:.1f} s"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
