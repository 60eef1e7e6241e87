#!/usr/bin/env python
"""bench.py -- the hot path of the TSM loop estimator on B200, one JSON line on stdout.

A "step" is one pass of the whole hot path over one batch of noise sources of the
32^3 x 64 workload (BASELINE.json configs[4], the one `metric` is quoted on): generate
12 Z4 sources on the device, source preparation, 100 fixed iterations of fp32 even-odd CG
on Mhat^dag Mhat (4 stencil launches, 2 one-block reductions and 1 fused BLAS launch each), reconstruction, local
and one-derivative loop contractions, accumulation into the Eq. 2.4 sums.

  value     = LP CG solves/s with the gauge field resident in HBM (device-timed, CUDA events)
  e2e       = the same through the public API with HOST buffers: every step uploads the gauge
              configuration from pinned host memory (tsm_set_gauge), solves, contracts, and
              reads the loops back to the host
  roofline  = the stencil kernels inside the timed steps: algorithmic bytes / CUDA-event time
  cpu_baseline = the oracle timed on this box's host cores on a bounded sample
  workloads = the same figures, compact, for BASELINE.json configs 1-4 (north_star: "for each workload")

python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload 1..5]

With --gpus N > 1 and no WORLD_SIZE in the environment the script starts its N ranks itself
(torch.distributed.run on 127.0.0.1); N replicas, no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1211_0126_b200 import replicas  # noqa: E402
from paper_1211_0126_b200 import workloads as W  # noqa: E402

METRIC = "lp_cg_solves_per_s"
UNIT = "solves/s"
PRECS = {"f64": 0, "f32": 1, "bf16": 2}


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ----------------------------------------------------------------------------- algorithmic bytes
def stencil_bytes_per_site(prec: str, recon: int, nrhs: int, kind: int) -> float:
    """SURVEY.md 8(d) / DESIGN.md: compulsory bytes per output site per source of one stencil
    launch: 8 neighbour spinors are each read once per field (24 reals in, 24 out = 48 w_s),
    8 links of n_g reals shared by the nrhs sources of a batch, +24 w_s for the x term (kinds 1, 2, 3;
    kind 2 also leaves |out|^2 per tile, which moves no extra field; kind 3 does not store its
    result but reads and writes the CG residual r, fp32 when the spinors are bf16)."""
    w_s = {"f64": 8, "f32": 4, "bf16": 2}[prec]
    w_r = 4 if prec == "bf16" else w_s
    w_g, n_g = (8, 18) if prec == "f64" else (4, recon)
    links = 8.0 * n_g * w_g / nrhs
    if kind == 3:
        return 48 * w_s + 48 * w_r + links
    return (48 + (24 if kind else 0)) * w_s + links


def ncu_traffic(workload: str, prec: str, nrhs: int):
    """DRAM traffic per stencil launch (dram__bytes_read.sum + dram__bytes_write.sum, mean of the four stencil
    launches of one CG iteration) from the committed ncu summary profiles/r02_traffic.json, written by
    `python -m paper_1211_0126_b200.ncu_summary` from an `ncu --set full` capture; the entry names the commit
    of the kernels it was captured at.  None when there is no capture for this case."""
    path = os.path.join(ROOT, "profiles", "r02_traffic.json")
    if not os.path.exists(path):
        return None
    try:
        return json.load(open(path)).get(f"{workload}/{prec}/nrhs{nrhs}")
    except (OSError, ValueError):
        return None


def workload_config(wl, nrhs: int, world: int) -> dict:
    """The `config` object of the JSON line: a pure function of the workload, so both arms print the same one."""
    Vh = wl.V // 2
    w_s = {"f64": 8, "f32": 4, "bf16": 2}[wl.lp_prec]
    link_mb = 2 * Vh * 8 * (18 * 8 if wl.lp_prec == "f64" else wl.reconstruct * 4) / 1e6
    vec_mb = Vh * 24 * w_s * nrhs / 1e6
    l2 = (f"inputs larger than L2 (links {link_mb:.0f} MB + {nrhs} x {vec_mb / nrhs:.0f} MB per vector); no flush needed"
          if link_mb + 5 * vec_mb > 126 else
          f"L2-RESIDENT working set (links {link_mb:.1f} MB + 5 vectors x {vec_mb:.1f} MB < 126 MB): the method re-reads the same "
          "fields every iteration, so no flush is applied; GB/s figures of this workload are not HBM figures")
    return {"workload": wl.name, "lattice": list(wl.dims), "kappa": wl.kappa, "mu": wl.mu, "links_eps": wl.eps,
            "nrhs_per_batch": nrhs, "lp_prec": wl.lp_prec, "lp_iters": wl.lp_iters, "lp_tol": wl.lp_tol, "reconstruct": wl.reconstruct,
            "derivative_loops": wl.derivative, "parallelism": f"replicas x{world}", "l2": l2}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, device: int):
        self.device = device
        self.rows = []
        self.proc = None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.device), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([t.strip() for t in line.split(",")])

    def __exit__(self, *exc):
        if self.proc is not None:
            time.sleep(0.15)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
                for k, n in enumerate(names):
                    if r[3 + k].lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                "samples": len(sm)}


# ----------------------------------------------------------------------------- the oracle legs
# An LP solve the oracle finishes within about a minute on the box's cores is run IN FULL (configs 1-4);
# config 5's 100-iteration solve (~275 s) is extrapolated linearly from 1- and 3-iteration solves.
def oracle_runs_in_full(wl) -> bool:
    return not (wl.lp_tol == 0 and wl.lp_iters * wl.V > 5e7)


def oracle_warm(wl, U):
    """One untimed call: thread pool start-up, page faults and the library load stay out of the timings."""
    import oracle
    oracle.hop(wl.dims, wl.t_boundary, U, oracle.noise(wl.dims, wl.noise_seed, 0), 0)


def oracle_lp_step(wl, U, sid: int, k_short: int | None = None):
    """One bounded sample of a step on the host cores, the oracle as it stands: one source; either the whole LP
    solve at the workload's truncation (source preparation, CG, reconstruction, fp64 residual), or -- config 5 --
    the same solve cut at k_short iterations.  Returns (seconds, iterations done, solution)."""
    import oracle
    eta = oracle.noise(wl.dims, wl.noise_seed, sid)
    t0 = time.perf_counter()
    if k_short is None:
        s, info = oracle.solve(wl.dims, wl.t_boundary, wl.kappa, wl.mu, U, eta, wl.lp_tol, wl.lp_iters)
    else:
        s, info = oracle.solve(wl.dims, wl.t_boundary, wl.kappa, wl.mu, U, eta, 0.0, k_short)
    return time.perf_counter() - t0, info["iters"], (eta, s)


def oracle_contract_time(wl, U, eta, s) -> float:
    import oracle
    t0 = time.perf_counter()
    oracle.all_loops(wl.dims, wl.t_boundary, U, eta, s, wl.derivative)
    return time.perf_counter() - t0


def oracle_baseline(wl, U, with_one_thread: bool):
    """cpu_baseline of our arm: the oracle on a bounded sample of the step (one source).  Returns the dict."""
    import oracle
    oracle_warm(wl, U)
    detail = {}
    if oracle_runs_in_full(wl):
        t_solve, iters, (eta, s) = oracle_lp_step(wl, U, 0)
        t_contract = oracle_contract_time(wl, U, eta, s)
        detail.update(t_lp_solve_s=t_solve, lp_iterations=iters, t_contract_s=t_contract, extrapolated=False)
        sample = (f"1 source in full: source preparation, the {iters}-iteration LP solve at the workload's truncation, "
                  "reconstruction, fp64 residual and one contraction pass")
    else:
        t1, _, _ = oracle_lp_step(wl, U, 0, 1)
        t3, _, (eta, s) = oracle_lp_step(wl, U, 0, 3)
        t_iter = (t3 - t1) / 2.0
        assert t_iter > 0, "oracle timing sample is inconsistent (3 iterations faster than 1)"
        t_contract = oracle_contract_time(wl, U, eta, s)
        t_solve = t1 + (wl.lp_iters - 1) * t_iter
        detail.update(t_1iter_solve_s=t1, t_3iter_solve_s=t3, t_per_cg_iteration_s=t_iter, t_contract_s=t_contract,
                      lp_iterations=wl.lp_iters, t_lp_solve_s=t_solve, extrapolated=True)
        sample = ("1 source: source preparation, 1- and 3-iteration CG solves, reconstruction, fp64 residual and one "
                  f"contraction pass run in full; the {wl.lp_iters}-iteration solve extrapolated linearly in the iteration count")
    # one full-lattice application of the hopping term (the oracle's Dslash), median of 5
    psi = oracle.noise(wl.dims, wl.noise_seed, 1)
    ts = []
    for _ in range(5):
        t0 = time.perf_counter()
        oracle.hop(wl.dims, wl.t_boundary, U, psi, -1)
        ts.append(time.perf_counter() - t0)
    detail["t_full_lattice_dslash_s_median_of_5"] = float(np.median(ts))
    if wl.V <= 131072:   # configs 1-3: one HP solve of the oracle in full as well
        eta_hp = oracle.noise(wl.dims, wl.noise_seed, 0)
        t0 = time.perf_counter()
        _, info_hp = oracle.solve(wl.dims, wl.t_boundary, wl.kappa, wl.mu, U, eta_hp, wl.hp_tol, 5000)
        detail["t_hp_solve_s"] = time.perf_counter() - t0
        detail["hp_iterations"] = info_hp["iters"]
    if with_one_thread and wl.V <= 131072:   # configs 1-3: the same on ONE host thread as well
        try:
            import ctypes
            gomp = ctypes.CDLL("libgomp.so.1")
            gomp.omp_set_num_threads(1)
            t1s, it1, _ = oracle_lp_step(wl, U, 0)
            t0 = time.perf_counter()
            oracle.hop(wl.dims, wl.t_boundary, U, psi, -1)
            td = time.perf_counter() - t0
            gomp.omp_set_num_threads(oracle.n_threads())
            detail["one_thread"] = {"t_lp_solve_s": t1s, "lp_iterations": it1, "t_full_lattice_dslash_s": td}
        except OSError:
            pass
    return {"value": 1.0 / (detail["t_lp_solve_s"] + detail["t_contract_s"]), "unit": UNIT, "cores": oracle.n_threads(),
            "kind": "oracle", "sample": sample, "extrapolated": detail["extrapolated"], "detail": detail}


def run_reference(args, wl):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only).  A step is a bounded sample
    of the workload's step: the whole LP solve + contraction where the oracle finishes it within about a minute,
    else (config 5) alternately a 1- and a 3-iteration solve, from which the full solve is extrapolated.
    `ms_per_step` is the time actually spent per timed step; `value` the (extrapolated) rate of full steps."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    oracle.build()
    U = wl.links()
    oracle_warm(wl, U)
    full = oracle_runs_in_full(wl)
    spent, by_k, t_contract, iters_seen = [], {1: [], 3: []}, None, None
    for k in range(args.warmup + args.steps):
        timed = k >= args.warmup
        t0 = time.perf_counter()
        if full:
            t_s, iters_seen, (eta, s) = oracle_lp_step(wl, U, k)
            t_c = oracle_contract_time(wl, U, eta, s)
            if timed:
                by_k[1].append(t_s + t_c)
        else:
            kk = 1 if k % 2 == 0 else 3
            t_s, _, (eta, s) = oracle_lp_step(wl, U, k, kk)
            if timed or not by_k[kk]:
                by_k[kk].append(t_s)
            if t_contract is None:          # one contraction pass, in the first (warm-up) step
                t_contract = oracle_contract_time(wl, U, eta, s)
        if timed:
            spent.append(time.perf_counter() - t0)
    cores = oracle.n_threads()
    if full:
        t_step = float(np.mean(by_k[1]))
        detail = {"lp_iterations": iters_seen, "extrapolated": False}
        sample = (f"per step: 1 source of the workload in full: source preparation, the LP solve at the workload's truncation "
                  f"({iters_seen} iterations), reconstruction, fp64 residual, one contraction pass")
    else:
        t1, t3 = float(np.mean(by_k[1])), float(np.mean(by_k[3]))
        t_iter = (t3 - t1) / 2.0
        assert t_iter > 0, "oracle timing sample is inconsistent"
        t_step = t1 + (wl.lp_iters - 1) * t_iter + t_contract
        detail = {"t_1iter_solve_s": t1, "t_3iter_solve_s": t3, "t_per_cg_iteration_s": t_iter, "t_contract_s": t_contract,
                  "lp_iterations": wl.lp_iters, "extrapolated": True, "s_per_full_step_extrapolated": t_step}
        sample = ("per step: 1 source of the workload; source preparation, a 1- or a 3-iteration CG solve (alternating), "
                  f"reconstruction and fp64 residual run in full; one contraction pass in the first warm-up step; the "
                  f"{wl.lp_iters}-iteration solve is extrapolated linearly in the iteration count, so `value` is an "
                  "extrapolated rate while `ms_per_step` is the time actually spent per step")
    value = 1.0 / t_step
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": float(np.mean(spent)) * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(wl, args.nrhs if args.nrhs > 0 else wl.nrhs, max(1, args.gpus)),
            "extrapolated": not full,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "detail": detail},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------- our arm
def finite_max(torch, buf, pname):
    v = buf.view({"f32": torch.float32, "f64": torch.float64, "bf16": torch.bfloat16}[pname]).float().abs().max().item()
    return v


def stencil_table(t, tsm, torch, wl, cases, peak, reps=50):
    """Single-launch stencil timings on FIXED inputs: D_eo a -> b and D_oe a -> c, the output never fed back
    (repeated applications multiply the norm by 4-6.5 and overflow fp32 within ~50 launches)."""
    table = {}
    stream = torch.cuda.current_stream()
    for pname, n in cases:
        p = PRECS[pname]
        a, b, c = t.alloc_field(p, n), t.alloc_field(p, n), t.alloc_field(p, n)
        if pname == "bf16":
            a.view(torch.bfloat16).copy_(torch.randn(a.numel() // 2, device=a.device, dtype=torch.float32))
        else:
            (a.view(torch.float32) if pname == "f32" else a.view(torch.float64)).normal_()
        for _ in range(5):
            t.dslash(tsm.OP_D_EO, p, n, a, b)
            t.dslash(tsm.OP_D_OE, p, n, a, c)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(reps):
            t.dslash(tsm.OP_D_EO, p, n, a, b)
            t.dslash(tsm.OP_D_OE, p, n, a, c)
        e1.record(stream)
        torch.cuda.synchronize()
        us = e0.elapsed_time(e1) * 1e3 / (2 * reps)
        by = stencil_bytes_per_site(pname, wl.reconstruct, n, 0) * (wl.V // 2) * n
        mx = max(finite_max(torch, b, pname), finite_max(torch, c, pname))
        table[f"{pname}_nrhs{n}"] = {"us": us, "algorithmic_GBs": by / us / 1e3, "frac_of_measured_peak": by / us / 1e3 / peak,
                                     "frac_of_8000": by / us / 1e3 / 8000.0, "gflops": 1320.0 * (wl.V // 2) * n / us / 1e3,
                                     "max_abs_out": mx, "finite": bool(np.isfinite(mx))}
        del a, b, c
    return table


def workload_summary(cfg: int, tsm, torch, peak, with_oracle: bool):
    """Compact figures for one of the small workloads (configs 1-4): single-launch stencil, LP solves/s in the
    workload's own launch configuration, the whole Eq. 2.4 set, iteration counts, and the oracle beside them."""
    wl = W.WORKLOADS[cfg]
    U = wl.links()
    stream = torch.cuda.current_stream()
    t = tsm.Tsm(wl.dims, t_boundary=wl.t_boundary, device=torch.cuda.current_device(), max_nrhs=wl.nrhs, stream=stream)
    t.set_params(wl.kappa, wl.mu)
    t.set_gauge(U, wl.reconstruct)
    if wl.lp_prec == "f64":
        t.set_hp_precision(tsm.F64)     # config 1 is "fp64 throughout"
    prec = PRECS[wl.lp_prec]
    out = {"lattice": list(wl.dims), "lp": f"{wl.lp_prec}, " + (f"tol {wl.lp_tol:g}" if wl.lp_tol > 0 else f"{wl.lp_iters} iterations"),
           "nrhs_per_batch": wl.nrhs, "reconstruct": wl.reconstruct}
    cases = [("f32", 1), ("f64", 1)] + ([(wl.lp_prec, wl.nrhs)] if (wl.lp_prec, wl.nrhs) not in (("f32", 1), ("f64", 1)) else [])
    out["dslash"] = {k: {"us": v["us"], "algorithmic_GBs": v["algorithmic_GBs"], "frac_of_measured_peak": v["frac_of_measured_peak"],
                         "gflops": v["gflops"], "finite": v["finite"]}
                     for k, v in stencil_table(t, tsm, torch, wl, cases, peak, reps=100).items()}
    out["l2_resident"] = wl.V <= 131072
    t.loops_reset(wl.derivative)
    steps, nb = 20, 0
    for k in range(3):
        t.solve(wl.noise_seed, list(range(k * wl.nrhs, (k + 1) * wl.nrhs)), prec, wl.lp_tol, wl.lp_iters, slot=1)
        t.loops_add_lp(1)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for k in range(steps):
        rc, info = t.solve(wl.noise_seed, list(range(1000 + k * wl.nrhs, 1000 + (k + 1) * wl.nrhs)), prec, wl.lp_tol, wl.lp_iters, slot=1)
        t.loops_add_lp(1)
        nb += wl.nrhs
    e1.record(stream)
    torch.cuda.synchronize()
    out["lp_solves_per_s"] = nb / (e0.elapsed_time(e1) * 1e-3)
    out["lp_iters"] = sorted(set(i["iters"] for i in info))
    # the same steps only ENQUEUED (tsm_solve_async; what tsm_run_loop_set does for its LP-only batches): the host runs
    # ahead of the device, one wait at the end
    e0.record(stream)
    for k in range(steps):
        t.solve_async(wl.noise_seed, list(range(2000 + k * wl.nrhs, 2000 + (k + 1) * wl.nrhs)), prec, wl.lp_tol, wl.lp_iters, slot=1)
        t.loops_add_lp(1)
    e1.record(stream)
    rc, info = t.solve_wait(1)
    torch.cuda.synchronize()
    out["lp_solves_per_s_enqueued"] = nb / (e0.elapsed_time(e1) * 1e-3)
    loops, secs, rc = t.run_loop_set(wl.noise_seed, wl.n_hp, wl.n_lp, prec, wl.lp_tol, wl.lp_iters, hp_tol=wl.hp_tol,
                                     hp_max_iter=5000, nrhs=wl.nrhs, with_derivative=wl.derivative)
    out["tsm_loop_set"] = {"seconds": secs, "n_hp": wl.n_hp, "n_lp": wl.n_lp, "rc": rc, "hp_solver": t.hp_precision_name(),
                           "finite": bool(np.isfinite(loops.view(np.float64)).all())}
    rc, info = t.solve(wl.noise_seed, list(range(min(wl.nrhs, wl.n_hp))), tsm.F64, wl.hp_tol, 5000, slot=0, want_true_resid=True)
    out["hp_solve"] = {"iters": sorted(set(i["iters"] for i in info)), "secs_batch": info[0]["secs"],
                       "true_resid_max": max(i["rel_resid_true"] for i in info)}
    t.close()
    if with_oracle:
        ob = oracle_baseline(wl, U, with_one_thread=True)
        out["oracle"] = {"lp_solves_per_s": ob["value"], "cores": ob["cores"], "extrapolated": ob["extrapolated"], **ob["detail"]}
    return out


def run_ours(args, wl):
    import torch
    import torch.distributed as dist
    from paper_1211_0126_b200 import tsm

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (there is no CPU fallback for the product path)")
    if world != args.gpus:
        raise RuntimeError(f"--gpus {args.gpus} but {world} rank(s) were started")
    if local >= torch.cuda.device_count():
        raise RuntimeError(f"rank {rank}: local rank {local} has no GPU ({torch.cuda.device_count()} visible)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    peak, peak_src = measured_peaks()
    prec_name = wl.lp_prec
    prec = PRECS[prec_name]
    nrhs = args.nrhs if args.nrhs > 0 else wl.nrhs
    tol, iters = wl.lp_tol, wl.lp_iters

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    t0 = time.perf_counter()
    U = replicas.node_shared_links(wl, local, world, barrier if world > 1 else None)   # generated once per node
    log(f"[bench] rank {rank}: links {wl.name} ready in {time.perf_counter() - t0:.1f} s")
    links_host = torch.from_numpy(np.ascontiguousarray(U).view(np.float64).reshape(-1)).pin_memory()
    stream = torch.cuda.current_stream()
    t = tsm.Tsm(wl.dims, t_boundary=wl.t_boundary, device=local, max_nrhs=nrhs, stream=stream)
    t.set_params(wl.kappa, wl.mu)
    if args.stencil_kernel:
        t.set_stencil_kernel(args.stencil_kernel)
    if args.graphs >= 0:
        t.set_graphs(args.graphs)
    dev = t.set_gauge(links_host, wl.reconstruct)
    log(f"[bench] unitarity deviation {dev:.2e}; workspace {t.workspace.numel() / 2**30:.1f} GiB")
    t.loops_reset(wl.derivative)
    # replicas only: every rank works on its own, disjoint source ids
    next_step = [0]

    def step():
        ids = replicas.replica_source_ids(rank, next_step[0], nrhs)
        next_step[0] += 1
        rc, info = t.solve(wl.noise_seed, ids, prec, tol, iters, slot=1)
        t.loops_add_lp(1)
        return info

    for _ in range(args.warmup):
        info = step()
    # ---- timed region: resident inputs.  On the large lattices every stencil / BLAS launch inside it is
    # bracketed by CUDA events on the library's stream (roofline).  On the small, launch-bound lattices
    # (configs 1-3) the timed steps run their CG iterations as CUDA graphs, which per-launch events would
    # break up, so the per-launch events are taken in an immediate repeat of the same steps.
    events_in_timed = wl.V >= (1 << 20)
    t.profile(events_in_timed)
    barrier()
    l0 = t.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clk:
        e0.record(stream)
        for _ in range(args.steps):
            info = step()
        e1.record(stream)
        barrier()
    ms = e0.elapsed_time(e1)
    launches = t.launch_count() - l0
    if not events_in_timed:
        t.profile(True)
        for _ in range(args.steps):
            step()
        torch.cuda.synchronize()
    t.profile(False)
    prof = {k: t.profile_read(prec, k, nrhs) for k in range(5)}
    ms = replicas.max_over_ranks(ms, device=f"cuda:{local}")
    value = replicas.whole_job_throughput(nrhs, args.steps, ms, world)

    # ---- roofline of the stencil kernels inside the timed steps
    Vh = wl.V // 2
    alg_bytes = sum(stencil_bytes_per_site(prec_name, wl.reconstruct, nrhs, k) * Vh * nrhs * prof[k][1] for k in range(4))
    st_ms = sum(prof[k][0] for k in range(4))
    st_n = sum(prof[k][1] for k in range(4))
    achieved = alg_bytes / (st_ms * 1e-3) / 1e9 if st_ms > 0 else 0.0
    traffic = ncu_traffic(wl.name, prec_name, nrhs)
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic["bytes_per_launch"] if traffic else None,
                "traffic_source": ({k: traffic[k] for k in ("commit", "summary", "kernels") if k in traffic} if traffic else None),
                "traffic_unit": "bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum, profiles/r02_traffic.json)",
                "peak_source": peak_src, "kernel": f"{t.stencil_kernel_name(prec, nrhs)}<{prec_name}, recon {wl.reconstruct}> x {nrhs} sources (the 4 stencil launches of a CG iteration)",
                "launches_timed": st_n, "avg_launch_us": st_ms * 1e3 / max(st_n, 1),
                "algorithmic_bytes_per_launch": alg_bytes / max(st_n, 1),
                "share_of_step": {"stencil": st_ms / ms, "cg_update_xp": prof[4][0] / ms} if events_in_timed else None,
                "per_kind_us": {str(k): (prof[k][0] * 1e3 / prof[k][1] if prof[k][1] else None) for k in range(5)},
                "per_kind_frac": {str(k): (stencil_bytes_per_site(prec_name, wl.reconstruct, nrhs, k) * Vh * nrhs * prof[k][1] / (prof[k][0] * 1e-3) / 1e9 / peak
                                           if prof[k][1] else None) for k in range(4)},
                "gflops_at_1320_per_site": 1320.0 * Vh * nrhs * st_n / (st_ms * 1e-3) / 1e9 if st_ms > 0 else 0.0,
                "events": "inside the timed steps" if events_in_timed else "in a repeat of the timed steps (the timed steps run CG as CUDA graphs)"}

    # second kernel class of the step: the CG x/p update (reads x, p, r; writes x, p)
    w_p = {"f64": 8, "f32": 4, "bf16": 2}[prec_name]
    w_x = 4 if prec_name == "bf16" else w_p
    xp_bytes = (48 * w_x + 24 * w_x + 48 * w_p) * Vh * nrhs
    xp_ms, xp_n = prof[4]
    roofline_xp = None
    if xp_n:
        xp_gbs = xp_bytes * xp_n / (xp_ms * 1e-3) / 1e9
        roofline_xp = {"bound": "hbm", "achieved": xp_gbs, "peak": peak, "unit": "GB/s", "frac": xp_gbs / peak,
                       "kernel": "k_cg_update_xp", "avg_launch_us": xp_ms * 1e3 / xp_n, "algorithmic_bytes_per_launch": xp_bytes}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": prec_name, "data": "synthetic", "config": workload_config(wl, nrhs, world),
            "gpu_launches": int(launches), "clocks": clk.summary(), "roofline": roofline, "roofline_cg_update": roofline_xp,
            "lp_iters_done": [i["iters"] for i in info]}

    # ---- e2e on every rank: host gauge field in (pinned memory -> tsm_set_gauge), host loops out, every step;
    # wall clock between device synchronisations, MAX over ranks, whole-job throughput
    if not args.skip_extras:
        n_e2e = max(1, min(args.steps, 3))
        barrier()
        w0 = time.perf_counter()
        for k in range(n_e2e):
            t.set_gauge(links_host, wl.reconstruct)          # H2D of the configuration + reorder kernels
            t.loops_reset(wl.derivative)
            step()
            loops_e2e = t.loops_finalize()                   # D2H of the [n_ops][T] loops
        torch.cuda.synchronize()
        secs_e2e = replicas.max_over_ranks(time.perf_counter() - w0, device=f"cuda:{local}")
        t.loops_reset(wl.derivative)
        line["e2e"] = {"value": world * nrhs * n_e2e / secs_e2e, "unit": UNIT, "h2d_bytes_per_step": int(links_host.numel() * 8),
                       "d2h_bytes_per_step": int(loops_e2e.nbytes), "steps": n_e2e,
                       "note": "per rank and step: the gauge configuration re-uploaded from pinned host memory, one batch solved and "
                               "contracted, the loops read back; in production one upload serves N_HP+N_LP solves"}

    if rank == 0 and not args.skip_extras:
        line.update(extras(args, wl, t, tsm, torch, prec, prec_name, peak, U, world))
    t.close()
    if rank == 0 and not args.skip_extras and not args.no_workloads and world == 1 and args.workload == 5:
        # north_star: "report, for each workload": configs 1-4, compact, in the same driver-run line
        line["workloads"] = {W.WORKLOADS[c].name: workload_summary(c, tsm, torch, peak, not args.no_cpu_baseline) for c in (1, 2, 3, 4)}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()   # rank 0 runs the single-rank extras; the others wait here instead of tearing NCCL down under it
        dist.destroy_process_group()


def extras(args, wl, t, tsm, torch, prec, prec_name, peak, U, world):
    """Single-launch stencil table, contraction kernels, full loop set, HP solves, oracle baseline."""
    out = {}
    nrhs = args.nrhs if args.nrhs > 0 else wl.nrhs
    # ---- single-launch stencil table (north_star: >= 70 % of HBM peak on single-RHS fp32 / fp64)
    out["dslash"] = stencil_table(t, tsm, torch, wl, (("f32", 1), ("f64", 1), ("f32", nrhs), ("bf16", 1)), peak)

    # ---- the same step with bf16-storage spinors (reading A15: fp32 is the headline, bf16 storage is reported beside it)
    if prec_name == "f32":
        ids = list(range(900000, 900000 + nrhs))
        t.solve(wl.noise_seed, ids, tsm.BF16, wl.lp_tol, wl.lp_iters, slot=1)
        rc_b, info_b = t.solve(wl.noise_seed, ids, tsm.BF16, wl.lp_tol, wl.lp_iters, slot=1, want_true_resid=True)
        out["lp_bf16_storage"] = {"solves_per_s": nrhs / info_b[0]["secs"], "secs_batch": info_b[0]["secs"], "iters": info_b[0]["iters"],
                                  "true_resid_max": max(i["rel_resid_true"] for i in info_b),
                                  "note": "solve only (no contraction); p, t, w in bf16, x, r and all sums fp32/fp64"}
        t.solve(wl.noise_seed, ids, prec, wl.lp_tol, wl.lp_iters, slot=1)   # leave an fp32 solution of this batch in the slot

    # ---- contraction kernels (H8, H9, the one-end loops of Eq. 2.5 (N1) and of Eq. 2.6 (N2; its two D_W stencil
    # launches are counted with the stencils, not here) on the slot the timed steps left
    bench_momenta = [(1, 0, 0), (0, 1, 0), (0, 0, 1), (-1, 0, 0), (0, -1, 0), (0, 0, -1)]
    t.loops_reset(wl.derivative, one_end=True, gen_one_end=True, momenta=bench_momenta)
    t.profile(True)
    for _ in range(3):
        t.loops_add_lp(1)
    t.profile(False)
    sp = PRECS["f32" if prec_name == "bf16" else prec_name]
    w_sol = 8 if prec_name == "f64" else 4
    names = {5: "local_16_gamma", 6: "derivative_4_directions", 7: "one_end_eq_2_5", 8: "gen_one_end_eq_2_6_contraction_only",
             9: "momentum_projected_6_momenta"}
    # algorithmic bytes per site of the full lattice and source (SURVEY.md 8(d) convention): s once (eta is regenerated,
    # never read); derivative: s once + the 8 links of the site ONCE PER BATCH
    n_g = 18 if prec_name == "f64" else wl.reconstruct
    by_site = {5: 24 * w_sol, 6: 24 * w_sol + 8 * n_g * (8 if prec_name == "f64" else 4) / nrhs, 7: 24 * w_sol, 8: 48 * w_sol, 9: 24 * w_sol}
    ct = {}
    for k in (5, 6, 7, 8, 9):
        ms_k, n_k = t.profile_read(sp, k, nrhs)
        if n_k:
            us = ms_k * 1e3 / n_k
            gb = by_site[k] * wl.V * nrhs / us / 1e3
            ct[names[k]] = {"us": us, "algorithmic_GBs": gb, "frac_of_measured_peak": gb / peak}
    out["contraction"] = ct
    t.loops_reset(wl.derivative)

    # ---- the whole of Eq. 2.4 for this configuration (reading A23)
    if not args.no_full_set:
        loops, secs, rc = t.run_loop_set(wl.noise_seed, wl.n_hp, wl.n_lp, prec, wl.lp_tol, wl.lp_iters, hp_tol=wl.hp_tol,
                                         hp_max_iter=5000, nrhs=nrhs, with_derivative=wl.derivative)
        out["tsm_loop_set"] = {"seconds": secs, "n_hp": wl.n_hp, "n_lp": wl.n_lp, "rc": rc, "hp_solver": t.hp_precision_name(),
                               "finite": bool(np.isfinite(loops.view(np.float64)).all())}
        rc, info = t.solve(wl.noise_seed, list(range(min(nrhs, wl.n_hp))), tsm.F64, wl.hp_tol, 5000, slot=0, want_true_resid=True)
        out["hp_solve_fp64"] = {"iters": [i["iters"] for i in info], "secs_batch": info[0]["secs"],
                                "true_resid_max": max(i["rel_resid_true"] for i in info)}
        # N4: the same HP solves as fp64 defect correction around the fp32 CG
        rc, info = t.solve(wl.noise_seed, list(range(min(nrhs, wl.n_hp))), tsm.MIXED, wl.hp_tol, 5000, slot=0, want_true_resid=True)
        out["hp_solve_mixed"] = {"iters_fp32_total": [i["iters"] for i in info], "secs_batch": info[0]["secs"],
                                 "true_resid_max": max(i["rel_resid_true"] for i in info)}
        other = tsm.F64 if t.hp_precision == tsm.MIXED else tsm.MIXED
        mine = t.hp_precision
        t.set_hp_precision(other)
        loops_o, secs_o, rc_o = t.run_loop_set(wl.noise_seed, wl.n_hp, wl.n_lp, prec, wl.lp_tol, wl.lp_iters, hp_tol=wl.hp_tol,
                                               hp_max_iter=5000, nrhs=nrhs, with_derivative=wl.derivative)
        t.set_hp_precision(mine)
        out["tsm_loop_set_other_hp_solver"] = {"seconds": secs_o, "rc": rc_o, "hp_solver": "fp64" if other == tsm.F64 else "mixed",
                                               "max_rel_diff_of_the_loops": float(np.abs(loops_o - loops).max() / np.abs(loops).max())}

    # ---- the oracle on this box's host cores, bounded sample (rank 0, N = 1 only)
    if not args.no_cpu_baseline and world == 1:
        import oracle
        oracle.build()
        out["cpu_baseline"] = oracle_baseline(wl, U, with_one_thread=True)
    return out


def run_probe_mma(args):
    """--probe-mma: the tensor-core clause of north_star measured once (csrc/mma_probe.cu):
    the per-(site, hop) SU(3) x (3 x 24) product, L2-resident operands, in five formulations.  One JSON line."""
    import torch
    from paper_1211_0126_b200 import tsm
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (there is no CPU fallback for the product path)")
    t = tsm.Tsm((4, 4, 4, 8), max_nrhs=1, stream=torch.cuda.current_stream())
    nsites, inner, reps = 1 << 16, 64, args.probe_reps
    names = {0: "fp32 packed FMA (FFMA2), thread per (site, source)", 1: "mma.sync m16n8k8 TF32", 2: "mma.sync m16n8k8 3xTF32 (split operands)",
             3: "fp64 FMA (DFMA), thread per (site, source)", 4: "mma.sync m8n8k4 fp64 (DMMA)"}
    out = {}
    for v in range(5):
        us, err = t.probe_su3_tensor(v, nsites, inner, reps)
        flops = nsites * inner * 24 * 3 * 8 * 3      # 3 complex rows x 3 complex MACs (8 real flops) per column
        out[names[v]] = {"us_per_launch": us, "site_hops_per_us": nsites * inner / us, "useful_gflops": flops / us / 1e3, "max_rel_err": err}
    # what one batched stencil launch of config 5 needs: V_h x 8 hops products of this shape
    wl = W.WORKLOADS[5]
    need = (wl.V // 2) * 8
    line = {"probe": "su3_x_3x24_per_site_hop", "nsites": nsites, "inner": inner, "reps": reps, "site_hops_per_stencil_launch_cfg5_nrhs12": need,
            "us_for_one_stencil_launch_worth": {k: need / v["site_hops_per_us"] for k, v in out.items()}, "variants": out}
    t.close()
    print(json.dumps(line), flush=True)


def spawn_ranks(args) -> int:
    """`python bench.py --gpus N` without a launcher: start the N ranks ourselves (one process per GPU)."""
    if args.impl == "ours":
        import torch
        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if have < args.gpus:
            log(f"[bench] --gpus {args.gpus} needs {args.gpus} CUDA devices, {have} visible: refusing to run fewer ranks than asked")
            return 2
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", type=int, default=5)
    ap.add_argument("--nrhs", type=int, default=0, help="sources per batch (default: the workload's; other values are profiling aids, not the headline)")
    ap.add_argument("--stencil-kernel", type=int, default=0, help="force a stencil kernel (tsm_set_stencil_kernel; profiling aid, not the headline)")
    ap.add_argument("--graphs", type=int, default=-1, help="tsm_set_graphs mode 0..3 (profiling aid; default: the library's)")
    ap.add_argument("--skip-extras", action="store_true", help="only the timed steps (no e2e/table/full set/oracle/workloads)")
    ap.add_argument("--no-full-set", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-workloads", action="store_true", help="skip the compact block for configs 1-4")
    ap.add_argument("--probe-mma", action="store_true", help="only the tensor-core probe of csrc/mma_probe.cu (DESIGN.md section 6)")
    ap.add_argument("--probe-reps", type=int, default=200, help="timed launches per variant of --probe-mma (1 under ncu)")
    args = ap.parse_args()
    if args.gpus < 1:
        ap.error("--gpus must be >= 1")
    if args.probe_mma:
        run_probe_mma(args)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(spawn_ranks(args))
    wl = W.WORKLOADS[args.workload]
    if args.impl == "reference":
        run_reference(args, wl)
    else:
        run_ours(args, wl)


if __name__ == "__main__":
    main()
