#!/usr/bin/env python
"""bench.py -- density-matrix builds/s of the submatrix hot path on B200 (BASELINE.json metric).

One "step" = one pass of the whole hot path over one synthetic input: sm_density_matrix on
BASELINE config 4 (20736 water molecules, SZV, cutoff 6 A, one submatrix per molecule) with the
library's default options: Gershgorin bracket of K~, a 24-step Lanczos run on K~ (interlacing scale,
bracket, quadrature estimate of mu), then the mu search, every step of which is one sign evaluation
(gather -> Newton-Schulz FP64 DMMA sign of all 20736 submatrices -> electron count), and the final
extract/scatter of D~.  With the default search (readings A11d/A11e) the caller's mu0 = -1
lies outside the Ritz interval taken for the gap and is NOT evaluated: the timed build is ONE sign
evaluation at the quadrature estimate, verified by its converged electron count (plateau acceptance).
`detail.literal_A11` reports the same build with the literal rule (step 0 at mu0, midpoint bisection),
`detail.guarded_tol_1e-8` BASELINE's literal tolerance.  The plan (device BSR container + submatrix
index, built once per sparsity pattern) is created before the timed region, like the paper's
initialisation phase (PAPER.md IV-A); its time is reported in `detail.plan_create_ms`.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]

Prints ONE JSON line (rank 0).  `value` = builds/s with K~ already resident in HBM; `e2e` = the
same through the C-ABI host-buffer call (H2D of K~ and D2H of D~ inside the timed region);
`roofline` = the Newton-Schulz GEMM kernel against the FP64 tensor peak; `cpu_baseline` = the CPU
oracle timed on this box's cores on a bounded sample.  N > 1: the same ONE problem sharded
over the ranks -- contiguous chunks of submatrices balanced by sum n^3, K~ replicated, one
scalar all-reduce per mu step, all-gather of the result columns -- i.e. strong scaling.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "density_matrix_builds_per_s"
UNIT = "builds/s"
EPS = 1e-12
TOL_N = 0.5      # plateau acceptance (reading A11); 1e-8 is unreachable by construction
MU0 = -1.0       # the caller's mu, inside the occupied band (evaluated only by the literal rule, see docstring)
# dram__bytes_read.sum + dram__bytes_write.sum per launch of k_ns_gemm from the committed
# `ncu --set full` capture of the current kernel (profiles/r02_full_captures.md): all-active launch,
# mean of MODE 0 (8.40 + 7.48 GB) and MODE 1 (17.82 + 7.66 GB).
NS_GEMM_DRAM_BYTES_PER_LAUNCH = 20.7e9
NOMINAL_FP64_OVER_BF16 = 45.0 / 2250.0  # guide: B200 FP64 tensor 45 TF/s, bf16 2250 TF/s (nominal)


def fp64_peak_tflops():
    """Roofline denominator for an FP64 contraction: measured bf16 peak x nominal FP64/bf16 ratio."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            pk = json.load(f)
        return pk["bf16_tflops"] * NOMINAL_FP64_OVER_BF16, "measured bf16 burst x 45/2250 (MEASURED_PEAKS.json)"
    return 1590.0 * NOMINAL_FP64_OVER_BF16, "fallback bf16 1.59 PF x 45/2250"


def hbm_peak_gbps():
    """Roofline denominator of the HBM-bound phases: the driver-measured copy bandwidth."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f)["hbm_gbs"], "MEASURED_PEAKS.json hbm_gbs (driver-measured copy bandwidth)"
    return 6544.3, "fallback: the copy bandwidth measured on this pool in round 1"


class ClockSampler:
    """SM clock, power and throttle reasons sampled DURING the timed region (profiling recipe): NVML
    in a background thread of this process (spawning `nvidia-smi -lms` was measured to stall the
    synchronous CUDA calls of the timed region while it attaches and on every query)."""

    def __init__(self, gpu_index, period_s=0.1):
        import threading
        self.samples, self.skip, self.run, self.err = [], 0, True, None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(gpu_index)
        except Exception as e:  # no NVML: the line says so instead of inventing clocks
            self.nv, self.err = None, repr(e)
            return
        self.period = period_s
        self.t = threading.Thread(target=self._loop, daemon=True)
        self.t.start()

    def _loop(self):
        nv = self.nv
        while self.run:
            try:
                sm = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                mx = nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM)
                pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
                rs = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h) if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons") \
                    else nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                self.samples.append((sm, mx, pw, rs))
            except Exception as e:
                self.err = repr(e)
            time.sleep(self.period)

    def mark(self):
        """Samples taken before this call (warm-up) are ignored by stop()."""
        self.skip = len(self.samples)

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.nv is None:
            out["error"] = self.err
            return out
        self.run = False
        self.t.join(timeout=2)
        nv = self.nv
        rows = self.samples[self.skip:] or self.samples[-1:]
        if not rows:
            out["error"] = self.err
            return out
        bits = {"hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
                "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
                "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
                "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4)}
        reasons = sorted(k for k, bit in bits.items() if any(r[3] & bit for r in rows))
        pmax = max(r[2] for r in rows)
        load = [r[0] for r in rows if r[2] >= 0.6 * pmax] or [r[0] for r in rows]
        return {"sm_mhz": statistics.median(load), "sm_max_mhz": max(r[1] for r in rows), "reasons": reasons,
                "power_w_max": pmax, "samples": len(rows)}


def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def max_over_ranks(ms: float, world: int, backend_device) -> float:
    """MAX over ranks of a per-rank time (plumbing only; no data-path collective)."""
    if world == 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=backend_device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def cpu_baseline(m, sample_groups=None, nthreads=0):
    """The oracle as it stands, timed on this box's cores on a bounded sample of the workload:
    Jacobi eigendecomposition + sign + extraction of `sample_groups` submatrices; the whole-job
    time is extrapolated by sum n_i^3 (Eq.(14)).  One decomposition serves the whole mu loop
    (Algorithm 1), so a build costs one pass."""
    from oracle import oracle as O
    cores = nthreads or os.cpu_count() or 1
    idx = O.Index(m)
    if sample_groups is None:
        # bounded sample: ~10-20 s of CPU work (the Jacobi oracle runs ~1.2e9 n^3-units per core in that time)
        mean_n3 = float((idx.sub_dim.astype(np.float64) ** 3).mean())
        k = int(max(min(cores, idx.ngroups), min(idx.ngroups, 1.2e9 * cores / mean_n3)))
        sample_groups = np.unique(np.linspace(0, idx.ngroups - 1, k).astype(np.int32))
    t0 = time.perf_counter()
    _ = O._run_groups(idx, m.values, sample_groups, 0.0, True, True, cores)
    dt = time.perf_counter() - t0
    n3 = idx.sub_dim.astype(np.float64) ** 3
    scale = n3.sum() / n3[sample_groups].sum()
    t_full = dt * scale
    return {"value": 1.0 / t_full, "unit": UNIT, "cores": cores, "kind": "oracle",
            "note": "the test oracle (cyclic Jacobi eigendecomposition), not a tuned CPU implementation",
            "sample": f"{len(sample_groups)} of {idx.ngroups} submatrices (evenly spaced), {dt:.2f} s measured, "
                      f"extrapolated x{scale:.1f} by sum n^3", "seconds_measured": dt}, t_full


def run_reference(args, m, rank):
    """--impl reference: the oracle on the host cores, each step a bounded sample."""
    if rank != 0:
        return
    cores = os.cpu_count() or 1
    times = []
    cb = None
    for it in range(args.warmup + args.steps):
        cb, t_full = cpu_baseline(m)
        if it >= args.warmup:
            times.append(t_full)
    t = sum(times) / len(times)
    line = {"impl": "reference", "metric": METRIC, "value": 1.0 / t, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(args, m), "cpu_baseline": dict(cb, value=1.0 / t),
            "e2e": {"value": 1.0 / t, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def run_phases(args, m, B, torch):
    """--phases: CUDA-event timing of the HBM-bound phases (a3 gather + a4 bound, a6 scatter) and of
    one fixed-mu sign evaluation, each against its roofline.  One JSON line."""
    plan = B.plan_from_matrix(m, B.default_options(mu_guess=args.mu_guess, mu_start=args.mu_start))
    info = B.sm_plan_query(plan)
    ws = B.alloc_workspace(plan)
    vin = torch.from_numpy(m.values).cuda()
    vout = torch.empty_like(vin)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    hbm = 6544.3
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            hbm = json.load(f)["hbm_gbs"]

    def timeit(f, reps=10):
        for _ in range(3):
            f()
        torch.cuda.synchronize()
        ts = []
        for _ in range(reps):
            e0.record(); f(); e1.record(); torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        return min(ts), float(np.median(ts))

    out = {"phases": True, "config": workload_config(args, m), "hbm_peak_GBps": hbm}
    gb = (info.sum_ld2 + info.nnz) * 8 / 1e9
    tmin, tmed = timeit(lambda: B.sm_gather(plan, vin, 0.0, ws))
    out["gather"] = {"ms_min": tmin, "ms_med": tmed, "alg_GB": gb, "GBps": gb / tmed * 1e3, "frac": gb / tmed * 1e3 / hbm}
    _, _, _, sub_dim, _ = B.sm_plan_export_index(plan)
    gw = np.zeros(m.ngroups, np.int64)
    np.add.at(gw, np.repeat(np.arange(m.ngroups), np.diff(m.grp_ptr)), m.blk_size[m.grp_cols])
    sb = ((sub_dim.astype(np.int64) * gw).sum() + info.nnz) * 8 / 1e9
    tmin, tmed = timeit(lambda: B.sm_scatter(plan, 1, vout, ws))
    out["scatter"] = {"ms_min": tmin, "ms_med": tmed, "alg_GB": sb, "GBps": sb / tmed * 1e3, "frac": sb / tmed * 1e3 / hbm}
    st = B.sm_stats_t()
    B.sm_set_timing(plan, True)
    for _ in range(2):
        B.sm_sign_execute(plan, vin, 0.0, EPS, vout, ws, st)
    d = st.as_dict()
    out["sign"] = {"ms_sign": d["ms_sign"], "iter_min": d["iter_min"], "iter_max": d["iter_max"],
                   "gemm_launches": d["gemm_launches"], "alg_TFLOPs": d["tot_sym_flop"] / d["ms_sign"] / 1e9,
                   "ms_gather": d["ms_gather"], "ms_scatter": d["ms_scatter"], "ms_total": d["ms_total"]}
    # opt-in reduced-precision variants (tcgen05): accuracy against the FP64 result, reported separately
    d64 = vout.clone()
    _, tdk64 = B.sm_trace_dk(plan, d64, vin)
    B.sm_plan_destroy(plan)
    del ws
    out["reduced_precision"] = {}
    for prec, name, eps in ((2, "3xTF32 (hi/lo split)", 2e-6), (4, "FP16x2 (hi/lo split)", 2e-6),
                            (3, "BF16x2 (hi/lo split)", 1e-5), (1, "TF32", 1e-5)):
        plan = B.plan_from_matrix(m, B.default_options(precision=prec))
        ws = B.alloc_workspace(plan)
        B.sm_set_timing(plan, True)
        for _ in range(2):
            rc = B.sm_sign_execute(plan, vin, 0.0, eps, vout, ws, st)
        torch.cuda.synchronize()
        d = st.as_dict()
        _, tdk = B.sm_trace_dk(plan, vout, vin)
        out["reduced_precision"][name] = {
            "status": int(rc), "ms_sign": d["ms_sign"], "iter_min": d["iter_min"], "iter_max": d["iter_max"],
            "residual_floor": d["max_residual"], "max_abs_err_vs_fp64": float((vout - d64).abs().max().item()),
            "rel_band_energy_err_vs_fp64": abs(tdk - tdk64) / abs(tdk64), "n_elec": d["n_elec"]}
        B.sm_plan_destroy(plan)
        del ws
    print(json.dumps(out), flush=True)


def run_extras(args, m, B, torch, plan, info, ws, d_in, d_out, mu, hbm_peak):
    """Everything else north_star names, measured in the same run after the timed regions (rank 0):
    phase rooflines of gather / scatter (CUDA events, best and median of 10), the literal A11 search, the
    guarded tol_n = 1e-8 run, and the opt-in reduced-precision variant on the same input."""
    out = {}
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def timeit(f, reps=10):
        for _ in range(3):
            f()
        torch.cuda.synchronize()
        ts = []
        for _ in range(reps):
            e0.record(); f(); e1.record(); torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        return min(ts), float(np.median(ts))

    tmp_out = torch.empty_like(d_out)
    gb = (info.sum_ld2 + info.nnz) * 8 / 1e9
    tmin, tmed = timeit(lambda: B.sm_gather(plan, d_in, mu, ws))
    out["gather"] = {"ms_min": tmin, "ms_med": tmed, "alg_GB": gb, "GBps": gb / tmed * 1e3, "frac": gb / tmed * 1e3 / hbm_peak}
    _, _, _, sub_dim, _ = B.sm_plan_export_index(plan)
    gw = np.zeros(m.ngroups, np.int64)
    np.add.at(gw, np.repeat(np.arange(m.ngroups), np.diff(m.grp_ptr)), m.blk_size[m.grp_cols])
    sb = ((sub_dim.astype(np.int64) * gw).sum() + info.nnz) * 8 / 1e9
    tmin, tmed = timeit(lambda: B.sm_scatter(plan, 1, tmp_out, ws))
    out["scatter"] = {"ms_min": tmin, "ms_med": tmed, "alg_GB": sb, "GBps": sb / tmed * 1e3, "frac": sb / tmed * 1e3 / hbm_peak}
    st = B.sm_stats_t()
    n_target = float(m.n_occ)

    # the literal tolerance of BASELINE config 4, guarded by mu_tol / max_mu_steps
    e0.record()
    rc, mu_g = B.sm_density_matrix(plan, d_in, n_target, 1e-8, EPS, MU0, tmp_out, ws, st)
    e1.record(); torch.cuda.synchronize()
    out["guarded_tol_1e-8"] = {"status": int(rc), "status_text": B.sm_strerror(int(rc)), "mu_steps": st.mu_steps,
                               "sign_evaluations": st.tot_evaluations, "abs_g": abs(st.n_elec - n_target),
                               "mu": mu_g, "ms": e0.elapsed_time(e1)}

    # reading A11 as written: step 0 at the caller's mu0, midpoint bisection (no quadrature estimate)
    plan2 = B.plan_from_matrix(m, B.default_options(mu_guess=0, mu_start=0))
    B.sm_density_matrix(plan2, d_in, n_target, TOL_N, EPS, MU0, tmp_out, ws, st)
    torch.cuda.synchronize()
    k = 3
    e0.record()
    for _ in range(k):
        rc, mu_l = B.sm_density_matrix(plan2, d_in, n_target, TOL_N, EPS, MU0, tmp_out, ws, st)
    e1.record(); torch.cuda.synchronize()
    d = st.as_dict()
    out["literal_A11"] = {"builds_per_s": k / (e0.elapsed_time(e1) * 1e-3), "ms_per_build": e0.elapsed_time(e1) / k,
                          "status": int(rc), "mu": mu_l, "mu_steps": d["mu_steps"], "sign_evaluations": d["tot_evaluations"],
                          "iter_trace": d["iter_trace"], "mu_trace": d["mu_trace"]}
    B.sm_plan_destroy(plan2)

    # Algorithm 1 as written (one eigendecomposition per build, mu loop on (lambda, w))
    plan4 = B.plan_from_matrix(m, B.default_options(method=1))
    B.sm_set_timing(plan4, True)
    B.sm_density_matrix(plan4, d_in, n_target, TOL_N, EPS, MU0, tmp_out, ws, st)
    torch.cuda.synchronize()
    k = 2
    e0.record()
    for _ in range(k):
        rc, mu_e = B.sm_density_matrix(plan4, d_in, n_target, TOL_N, EPS, MU0, tmp_out, ws, st)
    e1.record(); torch.cuda.synchronize()
    d = st.as_dict()
    out["algorithm1_eig"] = {"builds_per_s": k / (e0.elapsed_time(e1) * 1e-3), "ms_per_build": e0.elapsed_time(e1) / k,
                             "status": int(rc), "mu": mu_e, "mu_steps": d["mu_steps"], "decompositions": d["tot_evaluations"],
                             "jacobi_sweeps": [d["iter_min"], d["iter_max"]], "ms_decompose": d["ms_sign"],
                             "max_abs_diff_vs_newton_schulz": None}
    rc, mu_e2 = B.sm_density_matrix(plan4, d_in, n_target, TOL_N, EPS, mu, tmp_out, ws, st)  # same mu as the timed NS build
    torch.cuda.synchronize()
    if mu_e2 == mu:
        out["algorithm1_eig"]["max_abs_diff_vs_newton_schulz"] = float((tmp_out - d_out).abs().max().item())
    e0.record()
    rc, mu_g = B.sm_density_matrix(plan4, d_in, n_target, 1e-8, EPS, MU0, tmp_out, ws, st)
    e1.record(); torch.cuda.synchronize()
    out["algorithm1_eig"]["guarded_tol_1e-8"] = {"status": int(rc), "mu_steps": st.mu_steps, "decompositions": st.tot_evaluations,
                                                 "abs_g": abs(st.n_elec - n_target), "mu": mu_g, "ms": e0.elapsed_time(e1)}
    B.sm_plan_destroy(plan4)

    # opt-in reduced precision (tcgen05: 3xTF32 and the 16-bit split rungs FP16x2 / BF16x2) on the same input at the accepted mu, against
    # the FP64 result
    _, tdk64 = B.sm_trace_dk(plan, d_out, d_in)
    for prec, key, eps_r in ((2, "reduced_precision_3xTF32", 2e-6), (4, "reduced_precision_FP16x2", 2e-6),
                             (3, "reduced_precision_BF16x2", 1e-5)):
        plan3 = B.plan_from_matrix(m, B.default_options(precision=prec))
        need = B.sm_plan_query(plan3).workspace_bytes
        ws3 = ws if need <= ws.numel() * 8 else B.alloc_workspace(plan3)
        B.sm_set_timing(plan3, True)
        for _ in range(2):
            rc = B.sm_sign_execute(plan3, d_in, mu, eps_r, tmp_out, ws3, st)
        torch.cuda.synchronize()
        d = st.as_dict()
        _, tdk = B.sm_trace_dk(plan3, tmp_out, d_in)
        out[key] = {
            "status": int(rc), "ms_sign": d["ms_sign"], "ms_total": d["ms_total"], "iter_min": d["iter_min"],
            "iter_max": d["iter_max"], "residual_floor": d["max_residual"],
            "max_abs_err_vs_fp64": float((tmp_out - d_out).abs().max().item()),
            "rel_band_energy_err_vs_fp64": abs(tdk - tdk64) / abs(tdk64), "n_elec": d["n_elec"]}
        B.sm_plan_destroy(plan3)
        del ws3
    # the FP64 evaluation at the same mu, for the comparison above
    B.sm_sign_execute(plan, d_in, mu, EPS, tmp_out, ws, st)
    torch.cuda.synchronize()
    out["fp64_sign_evaluation"] = {"ms_sign": st.ms_sign, "ms_gather": st.ms_gather, "ms_scatter": st.ms_scatter,
                                   "ms_total": st.ms_total, "iter_min": st.iter_min, "iter_max": st.iter_max,
                                   "exits_predicted": st.exits_predicted, "exits_two_step": st.exits_two_step}
    # the same evaluation with the exits of readings A9b / A9c switched off (predict = 1: predicted exit only; 0: every
    # convergence confirmed by a computed residual), and how far the results are from the default's
    d_def = tmp_out.clone()
    out["exit_modes"] = {"predict=2 (default)": {"ms_sign": st.ms_sign, "max_residual": st.max_residual}}
    for pr in (1, 0):
        planp = B.plan_from_matrix(m, B.default_options(predict=pr))
        need = B.sm_plan_query(planp).workspace_bytes
        wsp = ws if need <= ws.numel() * 8 else B.alloc_workspace(planp)
        B.sm_set_timing(planp, True)
        for _ in range(2):
            rc = B.sm_sign_execute(planp, d_in, mu, EPS, tmp_out, wsp, st)
        torch.cuda.synchronize()
        out["exit_modes"][f"predict={pr}"] = {
            "status": int(rc), "ms_sign": st.ms_sign, "max_residual": st.max_residual, "iter_max": st.iter_max,
            "exits_predicted": st.exits_predicted, "exits_two_step": st.exits_two_step,
            "max_abs_diff_vs_default": float((tmp_out - d_def).abs().max().item())}
        B.sm_plan_destroy(planp)
        del wsp
    return out


def workload_config(args, m):
    from paper_2004_10811_b200 import workloads as W
    c = W.CONFIGS[args.config]
    return {"workload": f"BASELINE config {args.config}: " + (
                f"{c['n_mol']} H2O {c['basis']} cutoff {c['cutoff']} A, one submatrix per molecule"
                if c["kind"] == "water" else f"{c['batch']} dense n={c['n']} (block-diagonal plan)"),
            "n_basis": int(m.n_basis), "nnzb": int(m.nnzb), "ngroups": int(m.ngroups),
            "n_target": int(m.n_occ), "tol_n": TOL_N, "mu0": MU0, "eps": EPS,
            "mu_search": ("bisection started at the Lanczos quadrature estimate (A11d, A11e: mu0 lies outside the "
                          "Ritz interval taken for the gap)" if getattr(args, "mu_start", 1) else
                          "bisection from mu0, first interior step from the Lanczos quadrature (A11d)")
                         if getattr(args, "mu_guess", 1) else "midpoint bisection from mu0 (A11)",
            "cache": "inputs larger than L2 (dense workspace >> 126 MB)" if args.config in (3, 4, 5)
                     else "L2 flushed between steps", "seed": args.seed}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true",
                    help="skip the extra measurements of `detail` (phase rooflines, literal A11 search, guarded "
                         "1e-8 run, reduced-precision run)")
    ap.add_argument("--mu-guess", type=int, default=1, choices=[0, 1],
                    help="1 (library default): first interior step of the mu search from the Lanczos quadrature "
                         "(DESIGN.md reading A11d); 0: pure midpoint bisection (reading A11)")
    ap.add_argument("--mu-start", type=int, default=1, dest="mu_start",
                    help="1 (library default): step 0 of the mu search evaluates the quadrature estimate when mu0 lies "
                         "outside the Ritz interval taken for the gap (reading A11e); 0: step 0 always evaluates mu0")
    ap.add_argument("--phases", action="store_true",
                    help="time gather / scatter / one sign evaluation separately (phase rooflines) and exit")
    args = ap.parse_args()
    rank, local_rank, world = dist_env()
    from paper_2004_10811_b200 import workloads as W

    if args.impl == "reference":
        if rank == 0:
            run_reference(args, W.make_config(args.config, args.seed), rank)
        return

    import torch
    import torch.distributed as dist
    from paper_2004_10811_b200 import binding as B
    B.lib()  # fail loudly if the CUDA library is missing
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local_rank % torch.cuda.device_count())
    local_rank = local_rank % torch.cuda.device_count()
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        backend = os.environ.get("SM_DIST_BACKEND", "nccl")  # "gloo": functional check of the N > 1 path without N GPUs
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        else:
            dist.init_process_group(backend)

    # N > 1: ONE problem, every rank holds the whole K~ and owns a contiguous chunk of the
    # submatrices balanced by sum n^3; strong scaling
    m = W.make_config(args.config, args.seed)
    if args.phases:
        if rank == 0:
            run_phases(args, m, B, torch)
        return
    # roofline denominators measured in THIS run, with the clocks they were measured at
    peaks = None
    if rank == 0:
        smp = ClockSampler(local_rank, period_s=0.01) if not os.environ.get('SM_NO_SAMPLER') else None
        time.sleep(0.05)
        pk = B.sm_measure_peaks()
        peaks = {"dmma_issue_tflops": pk.dmma_tflops, "hbm_copy_GBps": pk.hbm_copy_gbs, "ms_dmma": pk.ms_dmma,
                 "ms_copy": pk.ms_copy, "num_sms": pk.num_sms, "clocks": smp.stop() if smp else None,
                 "how": "sm_measure_peaks: mma.sync.m8n8k4.f64 from registers, 16 warps/SM x 16 accumulators; "
                        "16-byte grid-stride copy of 1 GiB (read + write bytes); best of 5 each"}
    plan = B.plan_from_matrix(m, B.default_options(mu_guess=args.mu_guess, mu_start=args.mu_start,
                                                   shard_rank=rank, shard_world=world))
    if world > 1:  # one scalar all-reduce per mu step (the electron count), D~ columns by all-gather
        B.sm_plan_set_allreduce(plan, B.make_allreduce(device=torch.device("cuda", local_rank)))
    info = B.sm_plan_query(plan)
    ws = B.alloc_workspace(plan)
    d_in = torch.from_numpy(m.values).cuda()
    d_out = torch.empty_like(d_in)
    h_in = torch.from_numpy(m.values).pin_memory()
    h_out = torch.empty_like(h_in).pin_memory()
    flush = torch.empty(256 * 1024 * 1024 // 8, dtype=torch.float64, device="cuda") if args.config not in (3, 4, 5) else None
    stats = B.sm_stats_t()
    B.sm_set_timing(plan, True)
    n_target = float(m.n_occ)
    stream = torch.cuda.current_stream()

    def step_device():
        if flush is not None:
            flush.zero_()
        r = B.sm_density_matrix(plan, d_in, n_target, TOL_N, EPS, MU0, d_out, ws, stats)
        if world > 1:
            B.allgather_result(d_out, info)
        return r

    def step_host():
        if flush is not None:
            flush.zero_()
        if world == 1:
            return B.sm_density_matrix_host(plan, h_in, n_target, TOL_N, EPS, MU0, h_out, ws, stats)
        d_in.copy_(h_in, non_blocking=True)  # every rank receives the whole K~ and returns the whole D~
        r = B.sm_density_matrix(plan, d_in, n_target, TOL_N, EPS, MU0, d_out, ws, stats)
        B.allgather_result(d_out, info)
        h_out.copy_(d_out, non_blocking=True)
        torch.cuda.current_stream().synchronize()
        return r

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # the clock sampler attaches BEFORE the warm-up (nvidia-smi's start-up stalls synchronous CUDA calls
    # for a while); only the samples taken during the timed region are kept
    sampler = ClockSampler(local_rank) if (rank == 0 and not os.environ.get('SM_NO_SAMPLER')) else None
    for _ in range(args.warmup):
        st, mu = step_device()
    barrier()
    if sampler is not None:
        sampler.mark()
    launches0 = B.sm_launch_count(plan)
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    gemm_ms = gemm_launches = sym_flop = n3 = evals = gemm_only_ms = 0.0
    gather_ms = 0.0
    evs[0].record(stream)
    for i in range(args.steps):
        st, mu = step_device()
        evs[i + 1].record(stream)
        gemm_ms += stats.tot_ms_sign; gemm_launches += stats.tot_gemm_launches; gemm_only_ms += stats.tot_ms_gemm
        sym_flop += stats.tot_sym_flop; n3 += stats.tot_sum_iter_n3; evals += stats.tot_evaluations
        gather_ms += stats.tot_ms_gather
    barrier()
    launches = B.sm_launch_count(plan) - launches0
    ms = max_over_ranks(evs[0].elapsed_time(evs[-1]), world, torch.device("cuda", local_rank))
    per_step = [evs[i].elapsed_time(evs[i + 1]) for i in range(args.steps)]
    clocks = sampler.stop() if sampler else None
    last = stats.as_dict()

    # end to end through the host-buffer C-ABI call: same number of steps as the device-resident figure
    for _ in range(min(args.warmup, 2)):
        step_host()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    k_e2e = args.steps
    e0.record(stream)
    for _ in range(k_e2e):
        step_host()
    e1.record(stream)
    barrier()
    ms_e2e = max_over_ranks(e0.elapsed_time(e1), world, torch.device("cuda", local_rank))

    if rank == 0:
        peak, peak_src = fp64_peak_tflops()
        hbm_peak, hbm_src = hbm_peak_gbps()
        # dominant kernel: k_ns_gemm<0|1>.  Algorithmic flops of one symmetric n x n product:
        # n(n+1)/2 outputs x 2n flop = n^2 (n+1); per launch = sum over the active submatrices.
        # gemm_only_ms = CUDA-event time of the k_ns_gemm launches alone: the library records an event before and
        # after every product launch on its stream (sm_stats_t.tot_ms_gemm).  gemm_ms = the whole Newton-Schulz
        # phase (products + decision / bound / control kernels + the thin last updates, which are HBM-bound and
        # carry almost no flop): reported as sign_phase_tflops.
        ach = sym_flop / (gemm_only_ms * 1e-3) / 1e12 if gemm_only_ms > 0 else 0.0
        ach_phase = sym_flop / (gemm_ms * 1e-3) / 1e12 if gemm_ms > 0 else 0.0
        dmma = peaks["dmma_issue_tflops"]
        roofline = {"bound": "tensor", "kernel": "k_ns_gemm (FP64 DMMA Newton-Schulz, both modes)",
                    "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                    "traffic": NS_GEMM_DRAM_BYTES_PER_LAUNCH, "peak_source": peak_src,
                    "peak_dmma_issue_measured": dmma, "frac_of_dmma_issue": ach / dmma if dmma else None,
                    "launches_timed": int(gemm_launches), "avg_launch_ms": gemm_only_ms / max(gemm_launches, 1),
                    "sign_phase_tflops": ach_phase, "gemm_share_of_step": gemm_only_ms / ms if ms > 0 else None,
                    "alg_flop_per_launch": sym_flop / max(gemm_launches, 1),
                    "full_gemm_equiv_tflops": 2.0 * n3 / (gemm_ms * 1e-3) / 1e12 if gemm_ms > 0 else 0.0,
                    "sign_share_of_step": gemm_ms / ms if ms > 0 else None}
        gather_bytes = (info.sum_ld2 + info.nnz) * 8.0
        detail = {"status": int(st), "mu": mu, "mu_steps": last["mu_steps"], "n_elec": last["n_elec"],
                  "what_is_timed": "per build: Gershgorin bracket + 24-step Lanczos run + sign evaluations of the mu "
                                   "search (see sign_evaluations_per_step) + scatter",
                  "sign_evaluations_per_step": evals / args.steps,
                  "ms_per_step_best": min(per_step), "ms_per_step_median": statistics.median(per_step),
                  "ns_iterations_last_eval": last["iterations"], "iter_min": last["iter_min"],
                  "iter_max": last["iter_max"], "max_residual": last["max_residual"],
                  "dim_min": info.dim_min, "dim_mean": info.dim_mean, "dim_max": info.dim_max,
                  "workspace_GB": info.workspace_bytes / 1e9, "n_tiles": info.n_tiles,
                  "gather_GBps_in_build": gather_bytes * evals / (gather_ms * 1e-3) / 1e9 if gather_ms > 0 else None,
                  "ms_scatter_last": last["ms_scatter"], "mu_trace": last["mu_trace"],
                  "ne_trace": last["ne_trace"], "ne_err_trace": last["ne_err_trace"],
                  "iter_trace": last["iter_trace"], "spec_lo": last["spec_lo"], "spec_hi": last["spec_hi"],
                  "bracket": [last["bracket_lo"], last["bracket_hi"]],
                  "mu_guess": last["mu_guess"] if last["mu_guess"] == last["mu_guess"] else None,
                  "plan_create_ms": info.ms_plan_create,
                  "index_build": {"ms": info.ms_index_kernels, "alg_GB": info.index_alg_bytes / 1e9,
                                  "GBps": info.index_alg_bytes / 1e6 / info.ms_index_kernels if info.ms_index_kernels > 0 else None,
                                  "frac": info.index_alg_bytes / 1e6 / info.ms_index_kernels / hbm_peak if info.ms_index_kernels > 0 else None},
                  "hbm_peak_GBps": hbm_peak, "hbm_peak_source": hbm_src, "peaks_measured_this_run": peaks}
        if world > 1:
            detail["sharding"] = {"rule": "contiguous chunks balanced by sum n^3, PAPER.md L235 (sm_partition_groups)",
                                  "rank0_groups": [info.shard_group_begin, info.shard_group_end],
                                  "collectives_per_build": "1 all-reduce of 2 doubles per sign evaluation + all-gather of D~ "
                                                           "(one broadcast per rank of its value range)",
                                  "note": "GEMM / launch figures of this line are rank 0's"}
        if not args.no_extras and world == 1:
            detail.update(run_extras(args, m, B, torch, plan, info, ws, d_in, d_out, mu, hbm_peak))
        line = {"metric": METRIC, "value": args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
                "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
                "data": "synthetic", "config": workload_config(args, m), "clocks": clocks,
                "e2e": {"value": k_e2e / (ms_e2e * 1e-3), "unit": UNIT, "steps": k_e2e,
                        "h2d_bytes_per_step": int(info.nnz * 8), "d2h_bytes_per_step": int(info.nnz * 8)},
                "gpu_launches": int(launches), "roofline": roofline, "detail": detail}
        if not args.no_cpu_baseline:
            cb, _ = cpu_baseline(m)
            line["cpu_baseline"] = cb
        print(json.dumps(line), flush=True)
    B.sm_plan_destroy(plan)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
