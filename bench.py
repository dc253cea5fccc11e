#!/usr/bin/env python
"""bench.py - throughput of the FP64 ship-wave residual F(u) on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config cfg5_721x241]

One "step" = one pass of the whole hot path over one batch of synthetic input at the
configuration the metric is quoted on (cfg5, 721x241): sws_residual(u) followed by
sws_jv_batch(u, V[16]) = 18 residual evaluations (1 + (16 + 1)), 5.43e11 pair interactions.
`value` = residual evaluations per second with u and V resident in HBM; `e2e` = the same
through the host-buffer C-ABI calls (pinned host memory, H2D + D2H inside the timed region).

The path does not shard ("replicas only"): with --gpus N (launched by torchrun,
one rank per GPU) every rank runs the same step on its own GPU, no data-path collective;
`value` = N * evaluations / max-over-ranks time, scaling "weak".

--impl reference times the CPU oracle (oracle/, the paper's algorithm as plain C, as it
stands) on the host cores, on a bounded row sample of the same workload.
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

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

import workloads as W  # noqa: E402

METRIC = "fp64_residual_evals_per_s"
UNIT = "evals/s"
# Work of the all-pairs kernel per pair interaction, from its SASS inner loops:
#   near columns (S2 summed pair by pair): 43 FP64-pipe instructions = 24 DFMA (2 flops) + 19 DMUL/DADD;
#   far columns (S2 column sum from its Euler-Maclaurin form): 27 = 16 DFMA + 11 DMUL/DADD
#   (round 2, last session: the cube's third factor and the K2 sum ride the accumulating FMAs; 44 / 28 before).
# The 216 FP64 instructions (SASS count, sws_farfield.cuh) of the expansion per (target, far column) - 0.9 per
# pair at M = 241 - are NOT counted as achieved work.
FP64_INSTR_NEAR, FLOPS_NEAR = 43, 67
FP64_INSTR_FAR, FLOPS_FAR = 27, 43
FP64_LANES_PER_SM = 64  # FP64 FMA lanes per SM per clock on B200
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel at cfg5 from the ncu --set full
# capture summarised in NCU_PROFILE (a static figure: this run does not measure it).  The constant-bank kernel is
# launched once per slab of 8 source columns (91 launches per state); the staged kernel once per call.
NCU_DRAM_BYTES_PER_LAUNCH = {"k_allpairs_const": {"cfg5_721x241": 13.61e6}, "k_allpairs": {"cfg5_721x241": 160.42e6}}
NCU_PROFILE = {"k_allpairs_const": "profiles/r2b_allpairs_const_ncu.md", "k_allpairs": "profiles/r2a_allpairs_ncu.md"}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for nm, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def measured_peaks() -> dict:
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return json.loads(p.read_text())
        except Exception:
            return {}
    return {}


def oracle_sample(cfg, seconds: float, rows_fixed: int | None = None):
    """Time the f64 oracle (as it stands) on a seeded sample of integral-equation rows of cfg;
    returns (evals_per_s, rows, elapsed_s, threads).  rows/T of one evaluation's pairs are
    computed; the O(NM) part is computed in full each call."""
    import oracle
    orc = oracle.Oracle("f64")
    p, u = cfg.params(), W.state(cfg)
    T = cfg.targets
    threads = int(os.environ.get("OMP_NUM_THREADS", "0")) or (os.cpu_count() or 1)
    rng = np.random.default_rng(99)
    if rows_fixed is None:
        probe = np.sort(rng.choice(T, size=min(T, 512), replace=False)).astype(np.int32)
        t0 = time.perf_counter()
        orc.residual(p, u, rows=probe)
        dt = max(time.perf_counter() - t0, 1e-3)
        rows_fixed = int(min(T, max(512, probe.size * seconds / dt)))
    rows = np.sort(rng.choice(T, size=rows_fixed, replace=False)).astype(np.int32)
    t0 = time.perf_counter()
    orc.residual(p, u, rows=rows)
    dt = time.perf_counter() - t0
    return (rows.size / T) / dt, int(rows.size), dt, threads


def run_reference(args) -> None:
    """The oracle arm: rank 0 only; every step is one bounded row sample of cfg."""
    rank, world, _ = dist_env()
    if rank != 0:
        return
    cfg = W.BY_NAME[args.config]
    rows = args.ref_rows
    for _ in range(args.warmup):
        oracle_sample(cfg, 0.0, rows_fixed=rows)
    vals, threads, tot = [], 1, 0.0
    for _ in range(args.steps):
        v, nrows, dt, threads = oracle_sample(cfg, 0.0, rows_fixed=rows)
        vals.append(v)
        tot += dt
    value = args.steps * (rows / cfg.targets) / tot
    sample = (f"{rows} seeded integral-equation rows of {cfg.targets} per step (+ all O(NM) rows), "
              f"{rows * cfg.sources:.3e} pair interactions per step, scaled by rows/T")
    line = {
        "impl": "reference", "metric": f"{METRIC}_{cfg.N}x{cfg.M}", "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": cfg.name, "N": cfg.N, "M": cfg.M, "sample": sample},
        "pairs_per_s": value * cfg.pairs,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def fp32_variant_report(sws, device: int, names=("cfg4_361x121",), steps: int = 3) -> dict:
    """BASELINE.json config 4: "an FP32-accumulate variant, reported separately with its measured
    error".  sws_params.precision = 1 (FP32 pair arithmetic, Q12) timed on the same step
    (sws_residual + sws_jv_batch) with CUDA events; the error is the max-norm distance of its F(u)
    from the FP64 CUDA path on the same input (which the gpu tests hold to 1e-10 of the oracle;
    tests/test_gpu_parity.py measures the variant against the oracle itself)."""
    import torch
    out = {}
    for name in names:
        cfg = W.BY_NAME[name]
        b = cfg.b if cfg.b > 0 else 1
        u = torch.from_numpy(W.state(cfg)).cuda(device)
        V = torch.from_numpy(W.directions(cfg, b)).cuda(device)
        with sws.Context(cfg.params(), device=device) as c64:
            F64 = c64.residual(u).clone()
        with sws.Context(cfg.params(), max_batch=b, device=device, precision=1) as c32:
            F32 = c32.residual(u)
            c32.jv_batch(u, V)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(steps):
                c32.residual(u, out=F32)
                c32.jv_batch(u, V)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / steps
            ap_ms = c32.time_allpairs(b + 1, 2)
            err = float((F32 - F64).abs().max() / F64.abs().max())
        evals = 1 + (b + 1)
        out[name] = {"evals_per_s": evals / (ms * 1e-3), "pairs_per_s": evals * cfg.pairs / (ms * 1e-3),
                     "ms_per_step": ms, "jv_batch": b, "evals_per_step": evals,
                     "allpairs_pairs_per_s": (b + 1) * cfg.pairs / (ap_ms * 1e-3),
                     "max_rel_err_vs_fp64_path": err}
    out["note"] = ("precision=1: FP32 pair arithmetic (packed f32x2, MUFU.RSQ), FP32 accumulation per source "
                   "column, FP64 across columns, for the far-field S2 column sums and everywhere outside the "
                   "all-pairs kernel; reported, not part of `value`")
    return out


# FP64 instructions per pair of k_allpairs_lin<BT> (SASS inner loop): 71 shared by the
# BT directions (31 DFMA + 40 DMUL/DADD) + 4 DFMA per direction
LIN_INSTR_SHARED, LIN_FLOPS_SHARED = 71, 102


def jv_exact_report(ctx, cfg, u, V, steps: int, flush, peak_tf: float) -> dict:
    """sws_jv_exact_batch on the bench workload: b analytic Jacobian-vector
    products per call, timed like the main step (CUDA events, L2 flush between iterations)."""
    import torch
    b = int(V.shape[0])
    JV = torch.empty((b, cfg.n), dtype=torch.float64, device=u.device)
    for _ in range(2):
        ctx.jv_exact_batch(u, V, out=JV)
    torch.cuda.synchronize()
    ctx.set_profiling(True)
    ctx.profile_read(reset=True)
    ms = 0.0
    for _ in range(steps):
        flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ctx.jv_exact_batch(u, V, out=JV)
        e1.record()
        torch.cuda.synchronize()
        ms += e0.elapsed_time(e1)
    ap_ms, ap_n = ctx.profile_read(reset=True)
    ctx.set_profiling(False)
    ms /= steps
    info = ctx.lin_plan_info(b)
    bt = info["dirs_per_tile"]
    groups = -(-b // bt)
    flops_pair = LIN_FLOPS_SHARED + 8 * bt
    ach = flops_pair * cfg.pairs * groups / (ap_ms / max(ap_n, 1) * 1e-3) / 1e12
    return {"jv_per_s": b / (ms * 1e-3), "ms_per_batch": ms, "b": b, "launches_per_batch": ctx.last_launch_count,
            "allpairs_lin_ms": ap_ms / max(ap_n, 1), "share_of_batch": ap_ms / max(ap_n, 1) / ms,
            "pair_direction_products_per_s": b * cfg.pairs / (ms * 1e-3),
            "fp64_instr_per_pair": LIN_INSTR_SHARED + 4 * bt, "flops_per_pair": flops_pair,
            "achieved_tflops": ach, "frac_of_fp64_peak": ach / peak_tf, "plan": info,
            "note": "analytic J(u)v (no finite difference); parity 1e-10 of |JV|_inf against the complex-step "
                    "oracle in tests/test_gpu_parity.py"}


def jv_apply_report(ctx, cfg, u, V, steps: int, flush) -> dict:
    """sws_linearize once + sws_jv_apply (the Newton-Krylov shape): b = 1 (one GMRES product) and the
    full batch, CUDA events, L2 flush between iterations."""
    import torch
    out = {}
    ctx.linearize(u)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    flush.zero_()
    e0.record(); ctx.linearize(u); e1.record()
    torch.cuda.synchronize()
    out["linearize_ms"] = e0.elapsed_time(e1)
    for b in (1, int(V.shape[0])):
        Vb = V[:b].contiguous()
        JV = torch.empty((b, cfg.n), dtype=torch.float64, device=u.device)
        ctx.jv_apply(Vb, out=JV)
        torch.cuda.synchronize()
        ms = 0.0
        for _ in range(steps):
            flush.zero_()
            e0.record(); ctx.jv_apply(Vb, out=JV); e1.record()
            torch.cuda.synchronize()
            ms += e0.elapsed_time(e1)
        ms /= steps
        out[f"b{b}"] = {"ms_per_call": ms, "jv_per_s": b / (ms * 1e-3), "fp64_instr_per_pair": 41 + 4 * b,
                        "pair_direction_products_per_s": b * cfg.pairs / (ms * 1e-3)}
    return out


def solve_report(sws, device: int, names=("paper_361x121", "paper_721x241"), bandwidth: int = 31) -> dict:
    """The whole preconditioned JFNK solve on the paper's own meshes, from the flat
    initial guess, eps = 1, F = 0.7: wall time of the Newton driver with u resident on the
    device, plus the one-off preconditioner assembly + factorisation.  Context (other hardware): the paper
    reports 3.5 min (361x121) and 1.5 h (721x241) on a Tesla M2090 workstation, 75 min (361x121) on a desktop."""
    import torch

    import paper_1403_5044_b200.jfnk as jf
    out = {}
    for name in names:
        cfg = W.PAPER_BY_NAME[name]
        p = cfg.params()
        with sws.Context(p, max_batch=1, device=device) as ctx, \
                jf.Preconditioner(p, bandwidth=bandwidth, device=device, f32_panels=True) as pc, \
                jf.Solver(ctx, pc, 60) as s:
            u0 = torch.from_numpy(W.flat_state(cfg)).cuda(device)
            kw = dict(ftol=1e-9, eta=1e-3, restart=60, gmres_maxit=120)
            s.newton(u0, max_newton=1, **kw)                # warm-up (one Newton step)
            torch.cuda.synchronize()
            # the paper's own scheme: eq. (25) difference quotients, one residual evaluation per product
            t0 = time.perf_counter()
            u_fd, log_fd, st_fd = s.newton(u0, jv_mode=2, **kw)
            torch.cuda.synchronize()
            dt_fd = time.perf_counter() - t0
            # the same with inner tolerances that follow the nonlinear progress (sws_newton_opts.forcing = 1)
            t0 = time.perf_counter()
            u_ew, log_ew, st_ew = s.newton(u0, jv_mode=2, forcing=1, eta_max=0.5, **kw)
            torch.cuda.synchronize()
            dt_ew = time.perf_counter() - t0
            t0 = time.perf_counter()
            u, log, st = s.newton(u0, **kw)
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            out[name] = {"solve_s": dt, "precond_panels": "fp32",
                         "fd_jv": {"solve_s": dt_fd, "newton_steps": st_fd["steps"], "converged": st_fd["converged"],
                                   "jv_products": st_fd["jv_products"], "residual_evals": st_fd["residual_evals"],
                                   "final_residual_inf": log_fd[-1]["finf"], "ms_jv": st_fd["ms_jv"],
                                   "max_abs_diff_to_analytic_root": float((u_fd - u).abs().max())},
                         "fd_jv_forcing": {"solve_s": dt_ew, "newton_steps": st_ew["steps"],
                                           "converged": st_ew["converged"], "jv_products": st_ew["jv_products"],
                                           "residual_evals": st_ew["residual_evals"],
                                           "final_residual_inf": log_ew[-1]["finf"],
                                           "gmres_its_per_step": [e["gmres_its"] for e in log_ew[:-1]],
                                           "max_abs_diff_to_analytic_root": float((u_ew - u).abs().max())}, "precond_setup_s": pc.setup_ms * 1e-3, "precond_GB": pc.bytes / 1e9,
                         "block_bandwidth": pc.bandwidth, "newton_steps": st["steps"], "converged": st["converged"],
                         "jv_products": st["jv_products"], "residual_evals": st["residual_evals"],
                         "precond_applies": st["precond_applies"], "final_residual_inf": log[-1]["finf"],
                         "ms_jv": st["ms_jv"], "ms_precond": st["ms_precond"], "ms_residual": st["ms_residual"],
                         "gmres_its_per_step": [e["gmres_its"] for e in log[:-1]]}
    # Fig. 7 of the paper (L336): F = 1.4, 721 x 241, dx = dy = 0.3, x_0 = -56; the fastest configuration only
    cfg = W.PAPER_BY_NAME["paper_fig7_721x241"]
    p = cfg.params()
    with sws.Context(p, max_batch=1, device=device) as ctx, \
            jf.Preconditioner(p, bandwidth=bandwidth, device=device, f32_panels=True) as pc, \
            jf.Solver(ctx, pc, 60) as s:
        u0 = torch.from_numpy(W.flat_state(cfg)).cuda(device)
        kw = dict(ftol=1e-9, eta=1e-3, restart=60, gmres_maxit=120, jv_mode=2, forcing=1, eta_max=0.5)
        s.newton(u0, max_newton=1, **kw)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        u, log, st = s.newton(u0, **kw)
        torch.cuda.synchronize()
        out["paper_fig7_721x241_F1.4"] = {
            "fd_jv_forcing": {"solve_s": time.perf_counter() - t0, "newton_steps": st["steps"], "converged": st["converged"],
                              "jv_products": st["jv_products"], "residual_evals": st["residual_evals"],
                              "final_residual_inf": log[-1]["finf"],
                              "gmres_its_per_step": [e["gmres_its"] for e in log[:-1]]},
            "precond_setup_s": pc.setup_ms * 1e-3, "block_bandwidth": pc.bandwidth, "precond_panels": "fp32"}
    out["block_krylov_721x241"] = block_krylov_report(sws, jf, device, bandwidth)
    out["note"] = ("flat initial guess, eps=1, F=0.7, ||E||_inf <= 1e-9, inexact Newton eta=1e-3, analytic Jv "
                   "(sws_linearize + sws_jv_apply; `fd_jv`: eq. (25) quotients, jv_mode 2, one sws_residual per "
                   "product; `fd_jv_forcing`: the same with Eisenstat-Walker forcing terms, eta_max 0.5), block-banded linear-Jacobian preconditioner "
                   "with its factor panels stored in FP32 (`precond_panels`; since round 2: solve and apply times are not "
                   "comparable with round 1's FP64 panels); paper (other "
                   "hardware, KINSOL + FD Jv): 361x121 in ~3.5 min and 721x241 in 1.5 h on a Tesla M2090 workstation")
    return out


def block_krylov_report(sws, jf, device: int, bandwidth: int) -> dict:
    """SURVEY.md 8(f)2 "block/s-step Krylov that actually uses b > 1": the whole solve of the paper's 721x241 mesh
    with enlarged GMRES (sws_gmres_opts.block = t pieces of the right-hand side by groups of y-lines, ONE
    sws_jv_apply(V[t]) and ONE t-vector preconditioner sweep per block iteration) for t = 1 (plain GMRES), 4, 16;
    analytic Jv, eta = 1e-3.  pair_instructions = FP64 instructions of the all-pairs kernels to convergence:
    71 per pair per sws_linearize, 41 + 4 t per pair per sws_jv_apply(t), 27.4 per pair per sws_residual
    (SASS counts)."""
    import torch
    cfg = W.PAPER_BY_NAME["paper_721x241"]
    p = cfg.params()
    out = {}
    with sws.Context(p, max_batch=16, device=device) as ctx, \
            jf.Preconditioner(p, bandwidth=bandwidth, device=device, f32_panels=True) as pc, jf.Solver(ctx, pc, 176) as s:
        u0 = torch.from_numpy(W.flat_state(cfg)).cuda(device)
        kw = dict(ftol=1e-9, eta=1e-3, restart=160, gmres_maxit=640)
        s.newton(u0, max_newton=1, **kw)
        V = torch.randn(16, cfg.n, dtype=torch.float64, device=u0.device)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for t in (1, 4, 16):
            Vt = V[:t].contiguous()
            pc.apply_multi(Vt)
            torch.cuda.synchronize()
            e0.record(); pc.apply_multi(Vt); e1.record()
            torch.cuda.synchronize()
            pc_ms = e0.elapsed_time(e1)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            u, log, st = s.newton(u0, block=t if t > 1 else 0, **kw)
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            calls = st["jv_products"] // t
            instr = cfg.pairs * (st["steps"] * 71 + calls * (41 + 4 * t) + st["residual_evals"] * 27.4)
            out[f"t{t}"] = {"solve_s": dt, "converged": st["converged"], "newton_steps": st["steps"],
                            "jv_products": st["jv_products"], "block_iterations_per_step":
                            [e["gmres_its"] // t for e in log[:-1]], "pair_instructions": instr,
                            "precond_apply_ms": pc_ms, "precond_apply_ms_per_vector": pc_ms / t,
                            "ms_jv": st["ms_jv"], "ms_precond": st["ms_precond"]}
    out["note"] = ("enlarging the Krylov space by y-line groups does not reduce the number of (block) iterations on this "
                   "problem - the preconditioned spectrum is already clustered - so t > 1 costs t x the products: plain "
                   "GMRES (t = 1) stays the solver's default; the row is closed with this table (DESIGN.md section 5)")
    return out


def table1_report(sws, device: int, steps: int = 5) -> dict:
    """PAPER.md Table 1 (L281-290): seconds per function evaluation on the paper's five meshes (eps = 1,
    F = 0.7), here one sws_residual on a seeded synthetic state of that shape (CUDA events, L2 flushed by the
    256 MB fill between repetitions, median of `steps`).  The paper's columns (other hardware) ride along as
    context: multicore MATLAB on 2x Xeon E5-2670 and MATLAB + CUDA on a Tesla M2090."""
    import torch
    paper = {"91x31": (0.87, 0.02), "181x61": (4.38, 0.18), "271x91": (20.40, 0.83), "361x121": (64.35, 2.52),
             "451x151": (153.91, 6.04)}
    shapes = [(91, 31, 0.3, -9.0), (181, 61, 0.3, -14.0), (271, 91, 0.2, -14.0), (361, 121, 0.15, -14.0),
              (451, 151, 0.12, -14.0)]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=f"cuda:{device}")
    out = {}
    for N, M, h, x1 in shapes:
        cfg = W.custom(N, M, h, x1, eps=1.0, amp=0.05, seed=40 + N)
        u = torch.from_numpy(W.state(cfg)).cuda(device)
        with sws.Context(cfg.params(), device=device) as ctx:
            F = ctx.residual(u)
            for _ in range(3):
                ctx.residual(u, out=F)
            torch.cuda.synchronize()
            ts = []
            for _ in range(steps):
                flush.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(); ctx.residual(u, out=F); e1.record()
                torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1))
            loop_ms = ctx.time_residual(u, F, 50)       # 50 evaluations back to back, issued inside the library
        sec = float(np.median(ts)) * 1e-3
        cpu, gpu = paper[f"{N}x{M}"]
        out[f"{N}x{M}"] = {"seconds_per_evaluation": sec, "pairs_per_s": cfg.pairs / sec,
                           "seconds_per_evaluation_back_to_back": loop_ms * 1e-3,
                           "paper_workstation_matlab_s": cpu, "paper_m2090_s": gpu, "ratio_to_paper_m2090": gpu / sec}
    out["note"] = ("one sws_residual (whole u -> F path: up to 181x61 2 kernel launches - a cooperative launch for the "
                   "O(NM) stages, then the staged all-pairs kernel, which also assembles E2; from 271x91 the constant-bank "
                   "all-pairs path: one launch per slab of 16 source columns on two streams + a finishing launch) per "
                   "evaluation, synthetic state; "
                   "`seconds_per_evaluation` = an isolated call between synchronisations after an L2 flush, "
                   "`..._back_to_back` = sws_time_residual (a solver's view); the "
                   "paper's numbers are other hardware (2x Xeon E5-2670 / Tesla M2090, L265) and its own converged "
                   "states: context, not a target")
    return out


def configs_report(sws, device: int, peak_tf: float, names, steps: int = 20) -> dict:
    """BASELINE.json configs 1-4 in FP64 on their own step (single F(u) + the config's b-batch; cfg1: the single
    evaluation only): evaluations/s, pair interactions/s, share and executed-flop fraction of the all-pairs kernel.
    CUDA events per step on the launching stream, the 256 MB L2 flush between steps (not timed); `warm` = the same
    steps back to back without the flush (the working set of these meshes is far below the 126 MB L2)."""
    import torch
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=f"cuda:{device}")
    out = {}
    for name in names:
        cfg = W.BY_NAME[name]
        b = cfg.b
        u = torch.from_numpy(W.state(cfg)).cuda(device)
        V = torch.from_numpy(W.directions(cfg, b)).cuda(device) if b else None
        evals = 1 + ((b + 1) if b else 0)
        with sws.Context(cfg.params(), max_batch=b, device=device) as ctx:
            F = ctx.residual(u)

            def step():
                ctx.residual(u, out=F)
                n1 = ctx.last_launch_count
                if b:
                    ctx.jv_batch(u, V)
                    return n1 + ctx.last_launch_count
                return n1
            for _ in range(3):
                launches = step()
            torch.cuda.synchronize()
            ctx.set_profiling(True)
            ctx.profile_read(reset=True)
            ms = 0.0
            for _ in range(steps):
                flush.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(); step(); e1.record()
                torch.cuda.synchronize()
                ms += e0.elapsed_time(e1)
            ap_ms, ap_n = ctx.profile_read(reset=True)
            ctx.set_profiling(False)
            ms /= steps
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(steps):
                step()
            e1.record()
            torch.cuda.synchronize()
            ms_warm = e0.elapsed_time(e1) / steps
            near = ctx.farfield_stats((b + 1) if b else 1)
            flops_pair = near * FLOPS_NEAR + (1.0 - near) * FLOPS_FAR
            ach = flops_pair * evals * cfg.pairs * steps / (ap_ms * 1e-3) / 1e12
            out[name] = {"N": cfg.N, "M": cfg.M, "jv_batch": b, "evals_per_step": evals, "ms_per_step": ms,
                         "evals_per_s": evals / (ms * 1e-3), "pairs_per_s": evals * cfg.pairs / (ms * 1e-3),
                         "ms_per_step_warm": ms_warm, "evals_per_s_warm": evals / (ms_warm * 1e-3),
                         "launches_per_step": launches, "allpairs_share_of_step": ap_ms / steps / ms,
                         "near_column_fraction": near, "flops_per_pair": flops_pair,
                         "allpairs_achieved_tflops": ach, "allpairs_frac_of_fp64_peak": ach / peak_tf,
                         "allpairs_path": "k_allpairs_const" if ctx.const_plan_info()["active"] else "k_allpairs",
                         "plan": ctx.const_plan_info() if ctx.const_plan_info()["active"] else ctx.plan_info(1)}
    out["note"] = ("FP64, step = sws_residual(u) + sws_jv_batch(u, V[b]) as BASELINE.json states each config (cfg1: one "
                   "F(u)); parity of every one of these steps: tests/test_gpu_parity.py")
    return out


def run_ours(args) -> None:
    import torch

    import paper_1403_5044_b200 as sws
    from paper_1403_5044_b200 import replicas

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback for the product path)")
    torch.cuda.set_device(local)
    replicas.init("nccl", device=local)
    cfg = W.BY_NAME[args.config]
    b = cfg.b if cfg.b > 0 else 1
    p = cfg.params()
    u_h, V_h = W.state(cfg), W.directions(cfg, b)
    evals_per_step = 1 + (b + 1)          # sws_residual + the (b + 1) states of sws_jv_batch
    pairs_per_step = evals_per_step * cfg.pairs

    ctx = sws.Context(p, max_batch=b, device=local)
    u = torch.from_numpy(u_h).cuda(local)
    V = torch.from_numpy(V_h).cuda(local)
    F = torch.empty(cfg.n, dtype=torch.float64, device=u.device)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=u.device)  # > 126 MB L2
    launches_per_step = 0

    def step(mid=None):
        nonlocal launches_per_step
        ctx.residual(u, out=F)
        n1 = ctx.last_launch_count
        if mid is not None:
            mid.record()
        JV = ctx.jv_batch(u, V)
        launches_per_step = n1 + ctx.last_launch_count
        return JV

    for _ in range(max(args.warmup, 0)):
        step()
    torch.cuda.synchronize()

    # ---- timed region: device-resident inputs -------------------------------------------
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    ctx.set_profiling(True)
    ctx.profile_read(reset=True)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True),
           torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    replicas.barrier()
    torch.cuda.synchronize()
    for e0, em, e1 in ev:
        flush.zero_()                      # L2 flush between timed iterations (not timed)
        e0.record()
        step(em)
        e1.record()
    torch.cuda.synchronize()
    replicas.barrier()
    ms_total = sum(e0.elapsed_time(e1) for e0, _, e1 in ev)
    ms_batch = sum(em.elapsed_time(e1) for _, em, e1 in ev)   # the sws_jv_batch part of the steps
    ap_ms, ap_launches = ctx.profile_read(reset=True)
    ctx.set_profiling(False)
    near = ctx.farfield_stats(b + 1)       # of the b + 1 states of the last sws_jv_batch
    clocks = sampler.stop() if rank == 0 else None
    ms_total = replicas.max_over_ranks(ms_total)
    value = world * args.steps * evals_per_step / (ms_total * 1e-3)

    # ---- end to end: host buffers through the C-ABI host calls ----------------------------
    u_pin = torch.from_numpy(u_h).pin_memory()
    V_pin = torch.from_numpy(V_h).pin_memory()
    F_pin = torch.empty(cfg.n, dtype=torch.float64).pin_memory()
    JV_pin = torch.empty((b, cfg.n), dtype=torch.float64).pin_memory()
    Fp_pin = torch.empty((b, cfg.n), dtype=torch.float64).pin_memory()
    F0_pin = torch.empty(cfg.n, dtype=torch.float64).pin_memory()

    def step_host():
        ctx.residual_host(u_pin.numpy(), out=F_pin.numpy())
        ctx.jv_batch_host(u_pin.numpy(), V_pin.numpy(), out=JV_pin.numpy(), fpert=Fp_pin.numpy(),
                          f0=F0_pin.numpy())
        return float(JV_pin[0, 0])         # device -> host read of the step's result

    step_host()
    e2e_steps = args.steps
    replicas.barrier()
    torch.cuda.synchronize()
    ms_e2e = 0.0
    for _ in range(e2e_steps):
        flush.zero_()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        step_host()                        # ends with a stream synchronise inside the library
        ms_e2e += (time.perf_counter() - t0) * 1e3
    replicas.barrier()
    ms_e2e = replicas.max_over_ranks(ms_e2e)
    e2e_value = world * e2e_steps * evals_per_step / (ms_e2e * 1e-3)
    nb = cfg.n * 8
    h2d = nb + (nb + b * nb)                # u; then u and V
    d2h = nb + (b * nb + b * nb + nb)       # F; then JV, Fpert, F0

    if rank != 0:
        ctx.close()
        replicas.finalize()
        return

    # ---- roofline of the dominant kernel (all-pairs), bound: FP64 ALU pipe ---------------
    peaks = measured_peaks()
    from paper_1403_5044_b200 import debug as sws_debug
    probe = sws_debug.probe_fp64_peak(local)
    sm_count = probe["sm_count"]
    sm_max = (clocks or {}).get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0
    peak_tf = sm_count * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    mix = sws_debug.probe_fp64_mix(0, 32, local)      # measured issue rate of two-register DFMAs
    peak_measured_tf = mix["fp64_instr_per_sm_clk"] * 2 * sm_count * sm_max * 1e6 / 1e12
    pairs_timed = args.steps * pairs_per_step
    ap_s = ap_ms * 1e-3
    flops_pair = near * FLOPS_NEAR + (1.0 - near) * FLOPS_FAR
    instr_pair = near * FP64_INSTR_NEAR + (1.0 - near) * FP64_INSTR_FAR
    achieved_tf = flops_pair * pairs_timed / ap_s / 1e12
    sm_mhz = (clocks or {}).get("sm_mhz") or sm_max
    pipe_frac = instr_pair * pairs_timed / (sm_count * FP64_LANES_PER_SM * sm_mhz * 1e6 * ap_s)
    cinfo = ctx.const_plan_info()
    kernel = "k_allpairs_const" if cinfo["active"] else "k_allpairs"
    # kernel launches inside the timed all-pairs phases: one per (state, slab) on the constant-bank path
    kernels_timed = args.steps * evals_per_step * cinfo["slabs"] if cinfo["active"] else ap_launches
    if cinfo["active"]:   # per launch: the tile's target records once, the slab, the accumulators read + written
        alg_bytes = cfg.targets * 64 + cinfo["cols_per_slab"] * cfg.M * 32 + 2 * cfg.targets * 8
        alg_note = ("algorithmic bytes per launch = T*64 (target records) + 8 columns x M x 32 (the slab, through the "
                    "constant bank) + T*8 read + T*8 written (accumulators); the slab's group sums (one 8 B value per "
                    "target per group of columns) are written and read back inside the launch")
    else:
        alg_bytes = cfg.sources * 32 + cfg.targets * 64 + ctx.plan_info(1)["chunks"] * cfg.targets * 8
        alg_note = ("algorithmic bytes per state = S*32 + T*64 bytes read once + one 8 B partial sum per target per "
                    "column group written")
    roofline = {
        "bound": "alu", "kernel": kernel, "achieved": achieved_tf, "peak": peak_tf, "unit": "TFLOP/s",
        "frac": achieved_tf / peak_tf, "traffic": NCU_DRAM_BYTES_PER_LAUNCH[kernel].get(cfg.name),
        "traffic_source": f"{NCU_PROFILE[kernel]} (static: one ncu --set full capture of one launch of this kernel, "
                          "not measured by this run)",
        "peak_measured": peak_measured_tf,
        "peak_measured_source": f"sws_probe_fp64_mix kind 0 (register-only two-register DFMA loop, libsws_debug): "
                                f"{mix['fp64_instr_per_sm_clk']:.2f} of {FP64_LANES_PER_SM} FP64 thread-instructions/SM/clk "
                                f"x 2 flops x {sm_count} SMs x {sm_max:.0f} MHz",
        "frac_of_peak_measured": achieved_tf / peak_measured_tf if peak_measured_tf else None,
        "traffic_note": "DRAM bytes (read + written) of one launch; " + alg_note,
        "algorithmic_bytes_per_launch": alg_bytes,
        # per STATE the picture differs on the constant-bank path: every one of the slab launches re-reads the target
        # records and the accumulators, so one state moves (launches x per-launch traffic) through DRAM / L2 where the
        # algorithm needs the fields once: S*32 + T*64 + 2*T*8 bytes.  The re-read costs ~25 GB/s (0.4 % of HBM
        # bandwidth) at cfg5 - the kernel is bound by the FP64 pipe - but it is stated here, not hidden.
        "traffic_per_state": (NCU_DRAM_BYTES_PER_LAUNCH[kernel].get(cfg.name) or 0) * (cinfo["slabs"] if cinfo["active"] else 1) or None,
        "algorithmic_bytes_per_state": cfg.sources * 32 + cfg.targets * 64 + 2 * cfg.targets * 8,
        "traffic_per_state_over_algorithmic": ((NCU_DRAM_BYTES_PER_LAUNCH[kernel].get(cfg.name) or 0)
                                                * (cinfo["slabs"] if cinfo["active"] else 1)
                                                / (cfg.sources * 32 + cfg.targets * 64 + 2 * cfg.targets * 8)) or None,
        "peak_source": f"derived: {sm_count} SMs x {FP64_LANES_PER_SM} FP64 FMA lanes x 2 x {sm_max:.0f} MHz "
                       "(FP64 is not in MEASURED_PEAKS.json; DESIGN.md 'Peak')",
        "flops_per_pair": flops_pair, "fp64_instr_per_pair": instr_pair,
        "near_column_fraction": near,
        "work_note": f"executed pair-loop work: {FLOPS_NEAR} flops/pair on the near columns (direct S2), "
                     f"{FLOPS_FAR} on the far ones (S2 column sum in closed form + Euler-Maclaurin, sws_set_farfield); "
                     "with the plain 67 flops/pair definition the same time reads "
                     f"{FLOPS_NEAR * pairs_timed / ap_s / 1e12:.1f} TFLOP/s-equivalent",
        "launches_timed": kernels_timed, "avg_launch_ms": ap_ms / max(kernels_timed, 1),
        "phases_timed": ap_launches,
        "timing_note": "achieved = flops of all pairs of the timed steps / summed live CUDA-event time of the all-pairs "
                       "phases on the caller's stream (sws_set_profiling); on the constant-bank path a phase is the "
                       "slab launches of its states on the library's two streams (fork / join on the caller's stream, "
                       "slab copies included) and avg_launch_ms = that time / kernel launches",
        "share_of_step": ap_ms / ms_total if world == 1 else None,
        "dfma_probe_tflops": probe["tflops"], "dfma_probe_sm_mhz": probe["sm_mhz"],
        "frac_of_dfma_probe": achieved_tf / probe["tflops"] if probe["tflops"] else None,
        "fp64_pipe_issue_frac_at_sampled_clock": pipe_frac,
    }

    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        v, nrows, dt, threads = oracle_sample(cfg, args.cpu_seconds)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle",
                        "sample": f"{nrows} seeded integral-equation rows of {cfg.targets} (+ all O(NM) rows) of "
                                  f"one F(u) at {cfg.name}, {nrows * cfg.sources:.3e} pair interactions in "
                                  f"{dt:.1f} s, scaled by rows/T",
                        "pairs_per_s": v * cfg.pairs}

    jvx = None
    if world == 1 and not args.no_jv_exact:
        jvx = jv_exact_report(ctx, cfg, u, V, max(2, args.steps), flush, peak_tf)
        # the finite-difference batch of the main step computes the same b products from b + 1 evaluations
        jvx["speedup_vs_fd_batch"] = (jvx["jv_per_s"] /
                                      (b / ((ms_total / args.steps) * 1e-3 * (b + 1) / evals_per_step)))

    if jvx is not None:
        jvx["linearize_apply"] = jv_apply_report(ctx, cfg, u, V, max(2, args.steps), flush)

    solve = None
    if world == 1 and not args.no_solve:
        solve = solve_report(sws, local)

    table1 = None
    if world == 1 and not args.no_table1:
        table1 = table1_report(sws, local)

    configs = None
    if world == 1 and not args.no_configs:
        configs = configs_report(sws, local, peak_tf, [c.name for c in W.CONFIGS[:4]])

    fp32 = None
    if world == 1 and not args.no_fp32:
        fp32 = fp32_variant_report(sws, local, names=tuple(dict.fromkeys(["cfg4_361x121", cfg.name])))

    line = {
        "metric": f"{METRIC}_{cfg.N}x{cfg.M}", "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "N": cfg.N, "M": cfg.M, "h": cfg.h, "eps": cfg.eps,
                   "froude": cfg.froude, "jv_batch": b, "evals_per_step": evals_per_step,
                   "pairs_per_eval": cfg.pairs, "step": "sws_residual(u) + sws_jv_batch(u, V[b])",
                   "l2": "256 MB buffer written between timed iterations (L2 flush)",
                   "parallelism": "replicas only" if world > 1 else "1 gpu",
                   "plan": {"allpairs_path": kernel, "const": cinfo,
                            "staged_single": ctx.plan_info(1), "staged_batch": ctx.plan_info(b + 1)}},
        "pairs_per_s": value * cfg.pairs,
        # the step evaluates E(u) twice (sws_residual and state 0 of the batch, as BASELINE.json words the config):
        # a JFNK consumer that takes F0 from the batch needs the b + 1 DISTINCT states of sws_jv_batch alone
        "jv_batch_alone": {"ms": ms_batch / args.steps, "distinct_states": b + 1,
                           "distinct_state_evals_per_s": world * args.steps * (b + 1) / (ms_batch * 1e-3)}
        if world == 1 else None,
        "roofline": roofline, "cpu_baseline": cpu_baseline,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": ms_e2e / e2e_steps},
        "gpu_launches": launches_per_step * args.steps,
        "clocks": clocks,
        "workspace_bytes": ctx.workspace_bytes,
        "configs": configs,
        "jv_exact": jvx,
        "fp32_variant": fp32,
        "solve": solve,
        "table1": table1,
    }
    print(json.dumps(line), flush=True)
    ctx.close()
    replicas.finalize()


def run_microbench(args) -> None:
    """--microbench: the FP64 instruction-mix probes behind the cycle model of DESIGN.md section 6, one JSON
    line (not a bench value: no workload is run)."""
    import torch

    import paper_1403_5044_b200 as sws
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --microbench: no CUDA device")
    from paper_1403_5044_b200 import debug as sws_debug
    rows = [sws_debug.probe_fp64_mix(k, w) for k in range(len(sws_debug.FP64_MIX_KINDS)) for w in (16, 32, 64)]
    print(json.dumps({"microbench": "fp64_instruction_mix", "unit": "FP64 thread-instructions / SM / clk (64 = issue limit)",
                      "rows": rows, "dfma_probe": sws_debug.probe_fp64_peak(0)}), flush=True)


def run_experiments(args) -> None:
    """--experiments: the measurements behind profiles/r2_experiments.md and profiles/r2_small_meshes.md, one JSON
    line (not a bench value).  batch_sharing: the all-pairs kernel alone for a single state and for the b + 1 states
    of each config's batch with one and with two states per CTA (sws_set_states_per_cta).  small_meshes:
    sws_time_residual (evaluations back to back, issued inside the library) with the fused cooperative fields launch
    and with the three separate launches, and the all-pairs kernel alone."""
    import torch

    import paper_1403_5044_b200 as sws
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --experiments: no CUDA device")
    out = {"experiments": "round 2", "allpairs_paths": {}, "batch_sharing": {}, "small_meshes": {}}
    # the all-pairs phase of ONE state alone (sws_time_allpairs) on the constant-bank path and on the staged kernel,
    # and whole evaluations back to back (sws_time_residual), on the BASELINE meshes and the sizes in between
    for (N, M, h) in ((181, 61, 0.3), (226, 76, 0.24), (271, 91, 0.2), (316, 106, 0.17), (361, 121, 0.15),
                      (721, 241, 0.075)):
        cfg = W.custom(N, M, h, -16.0, eps=1.0, amp=0.1, seed=5)
        with sws.Context(cfg.params()) as ctx:
            u = torch.from_numpy(W.state(cfg)).cuda()
            F = torch.empty_like(u)
            row = {"targets": cfg.targets, "default_path": "const" if ctx.const_plan_info()["active"] else "staged"}
            for mode, key in ((1, "const"), (0, "staged")):
                ctx.set_const_path(mode)
                ctx.residual(u, out=F)
                torch.cuda.synchronize()
                reps = 5 if N > 400 else 30
                row[f"{key}_allpairs_ms"] = min(ctx.time_allpairs(1, reps) for _ in range(3))
                row[f"{key}_residual_ms"] = min(ctx.time_residual(u, F, reps) for _ in range(3))
            row["const_plan"] = ctx.const_plan_info()
            out["allpairs_paths"][f"{N}x{M}"] = row
    for name in ("cfg5_721x241", "cfg4_361x121", "cfg3_181x61"):
        cfg = W.BY_NAME[name]
        b = cfg.b
        with sws.Context(cfg.params(), max_batch=b) as ctx:
            ctx.set_const_path(0)      # this section is about the staged kernel's batched mode
            u = torch.from_numpy(W.state(cfg)).cuda()
            V = torch.from_numpy(W.directions(cfg, b)).cuda()
            ctx.jv_batch(u, V)
            torch.cuda.synchronize()
            one = ctx.time_allpairs(1, 5)
            row = {"b": b, "single_ms": one}
            for ns in (1, 2):
                ctx.set_states_per_cta(ns)
                ms = ctx.time_allpairs(b + 1, 3)
                row[f"ns{ns}_ms"] = ms
                row[f"ns{ns}_over_states_x_single"] = ms / ((b + 1) * one)
            out["batch_sharing"][name] = row
    for (N, M, h, x1) in [(31, 11, 0.8, -8.0), (61, 21, 0.4, -8.0), (91, 31, 0.3, -9.0), (181, 61, 0.3, -14.0),
                          (361, 121, 0.15, -14.0)]:
        cfg = W.custom(N, M, h, x1, eps=1.0, amp=0.05, seed=40 + N)
        with sws.Context(cfg.params()) as ctx:
            u = torch.from_numpy(W.state(cfg)).cuda()
            F = ctx.residual(u)
            torch.cuda.synchronize()
            row = {"allpairs_alone_us": ctx.time_allpairs(1, 50) * 1e3}
            for fused in (1, 0):
                ctx.set_fused_fields(bool(fused))
                row["fused_us" if fused else "separate_us"] = ctx.time_residual(u, F, 100) * 1e3
                row["launches_fused" if fused else "launches_separate"] = ctx.last_launch_count
            out["small_meshes"][f"{N}x{M}"] = row
    print(json.dumps(out), flush=True)


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", default="cfg5_721x241", choices=sorted(W.BY_NAME))
    ap.add_argument("--cpu-seconds", type=float, default=30.0, help="CPU work of the cpu_baseline leg")
    ap.add_argument("--ref-rows", type=int, default=2048, help="rows per step of --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-fp32", action="store_true", help="skip the reported FP32-variant section")
    ap.add_argument("--no-jv-exact", action="store_true", help="skip the analytic-Jv section")
    ap.add_argument("--no-solve", action="store_true", help="skip the full JFNK solve section")
    ap.add_argument("--no-table1", action="store_true", help="skip the paper's Table 1 meshes")
    ap.add_argument("--no-configs", action="store_true", help="skip the FP64 section on BASELINE configs 1-4")
    ap.add_argument("--microbench", action="store_true", help="only run the FP64 instruction-mix probes")
    ap.add_argument("--experiments", action="store_true",
                    help="only run the round-2 experiments (states per CTA, small-mesh launch paths)")
    args = ap.parse_args()
    if args.microbench:
        run_microbench(args)
        return
    if args.experiments:
        run_experiments(args)
        return
    if args.warmup < 3 and args.impl == "ours":
        print("bench.py: warning: fewer than 3 warm-up steps", file=sys.stderr)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
