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

python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload 1..5]
"""
from __future__ import annotations

import argparse
import json
import os
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


# DRAM traffic per stencil launch from ncu (dram__bytes_read.sum + dram__bytes_write.sum, mean of the four
# stencil launches of one CG iteration), keyed by (workload, precision, sources per batch); the capture and
# its command are in profiles/r01_dslash_r12_tile.md and profiles/r01_dslash_r1.md.  None when not captured.
NCU_TRAFFIC_BYTES = {
    ("cfg5_32x32x32x64", "f32", 12): (4.628e9 + 3.420e9 + 5.987e9 + 3.391e9) / 4,
    ("cfg5_32x32x32x64", "f32", 1): (0.906e9 + 0.789e9 + 0.905e9 + 0.789e9) / 4,
}


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
def oracle_sample(wl, U, sid: int = 0):
    """Bounded sample of one step on the host cores, with the oracle as it stands: one source,
    source preparation + 1 and 3 CG iterations + reconstruction (+ residual check), and one
    pass of the loop contractions; the full lp_iters-iteration solve is extrapolated linearly
    in the iteration count.  Returns (seconds per solve incl. contraction, detail dict)."""
    import oracle
    eta = oracle.noise(wl.dims, wl.noise_seed, sid)
    t0 = time.perf_counter()
    s1, _ = oracle.solve(wl.dims, wl.t_boundary, wl.kappa, wl.mu, U, eta, 0.0, 1)
    t1 = time.perf_counter()
    s3, _ = oracle.solve(wl.dims, wl.t_boundary, wl.kappa, wl.mu, U, eta, 0.0, 3)
    t3 = time.perf_counter()
    oracle.all_loops(wl.dims, wl.t_boundary, U, eta, s3, wl.derivative)
    tl = time.perf_counter()
    t_iter = ((t3 - t1) - (t1 - t0)) / 2.0
    iters = wl.lp_iters if wl.lp_tol == 0 else 10
    t_solve = (t1 - t0) + (iters - 1) * t_iter + (tl - t3)
    detail = {"t_1iter_solve_s": t1 - t0, "t_per_cg_iteration_s": t_iter, "t_contract_s": tl - t3,
              "iterations_extrapolated_to": iters}
    return t_solve, detail


def run_reference(args, wl):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    oracle.build()
    U = wl.links()
    times = []
    detail = {}
    for k in range(args.warmup + args.steps):
        t, detail = oracle_sample(wl, U, sid=k)
        if k >= args.warmup:
            times.append(t)
    t = float(np.mean(times))
    value = 1.0 / t
    cores = oracle.n_threads()
    sample = ("per step: 1 source of the workload; source preparation, 1- and 3-iteration CG solves, "
              "reconstruction, fp64 residual and one contraction pass run in full, the "
              f"{detail['iterations_extrapolated_to']}-iteration solve extrapolated linearly")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl.name, "lattice": list(wl.dims), "lp_iters": wl.lp_iters, "lp_tol": wl.lp_tol,
                       "derivative_loops": wl.derivative},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                             "detail": detail},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------- our arm
def run_ours(args, wl):
    import torch
    import torch.distributed as dist
    from paper_1211_0126_b200 import tsm

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (there is no CPU fallback for the product path)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    peak, peak_src = measured_peaks()
    prec_name = wl.lp_prec
    prec = PRECS[prec_name]
    nrhs = args.nrhs if args.nrhs > 0 else wl.nrhs
    tol, iters = wl.lp_tol, wl.lp_iters

    t0 = time.perf_counter()
    U = wl.links()
    log(f"[bench] rank {rank}: links {wl.name} generated in {time.perf_counter() - t0:.1f} s")
    links_host = torch.from_numpy(U.view(np.float64).reshape(-1)).pin_memory()
    stream = torch.cuda.current_stream()
    t = tsm.Tsm(wl.dims, t_boundary=wl.t_boundary, device=local, max_nrhs=nrhs, stream=stream)
    t.set_params(wl.kappa, wl.mu)
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

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

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
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": NCU_TRAFFIC_BYTES.get((wl.name, prec_name, nrhs)), "traffic_unit": "bytes per launch (ncu, profiles/)",
                "peak_source": peak_src, "kernel": f"{'k_dslash_tile' if nrhs > 1 and prec_name != 'f64' else 'k_dslash'}<{prec_name}, recon {wl.reconstruct}> x {nrhs} sources (the 4 stencil launches of a CG iteration)",
                "launches_timed": st_n, "avg_launch_us": st_ms * 1e3 / max(st_n, 1),
                "algorithmic_bytes_per_launch": alg_bytes / max(st_n, 1),
                "share_of_step": {"stencil": st_ms / ms, "cg_update_xp": prof[4][0] / ms} if events_in_timed else None,
                "per_kind_us": {str(k): (prof[k][0] * 1e3 / prof[k][1] if prof[k][1] else None) for k in range(5)},
                "gflops_at_1320_per_site": 1320.0 * Vh * nrhs * st_n / (st_ms * 1e-3) / 1e9 if st_ms > 0 else 0.0}

    w_s = {"f64": 8, "f32": 4, "bf16": 2}[prec_name]
    link_mb = 2 * Vh * 8 * (18 * 8 if prec_name == "f64" else wl.reconstruct * 4) / 1e6
    vec_mb = Vh * 24 * w_s * nrhs / 1e6
    l2_note = (f"inputs larger than L2 (links {link_mb:.0f} MB + {nrhs} x {vec_mb / nrhs:.0f} MB per vector)" if link_mb + 5 * vec_mb > 126
               else f"L2-RESIDENT working set (links {link_mb:.1f} MB + 5 vectors x {vec_mb:.1f} MB < 126 MB): the method re-reads the same "
                    "fields every iteration, so no flush is applied; GB/s figures of this workload are not HBM figures")
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
            "dtype": prec_name, "data": "synthetic",
            "config": {"workload": wl.name, "lattice": list(wl.dims), "kappa": wl.kappa, "mu": wl.mu, "links_eps": wl.eps,
                       "nrhs_per_batch": nrhs, "lp_iters": iters, "lp_tol": tol, "reconstruct": wl.reconstruct,
                       "derivative_loops": wl.derivative, "parallelism": f"replicas x{world}",
                       "roofline_events": "inside the timed steps" if events_in_timed else "in a repeat of the timed steps (the timed steps run CG as CUDA graphs)",
                       "l2": l2_note},
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
        line.update(extras(args, wl, t, tsm, torch, links_host, prec, prec_name, step, peak, U))
    if rank == 0:
        print(json.dumps(line), flush=True)
    t.close()
    if world > 1:
        dist.barrier()   # rank 0 runs the single-rank extras; the others wait here instead of tearing NCCL down under it
        dist.destroy_process_group()


def extras(args, wl, t, tsm, torch, links_host, prec, prec_name, step, peak, U):
    """e2e through the host-buffer API, single-launch stencil table, full loop set, oracle baseline."""
    out = {}
    nrhs = args.nrhs if args.nrhs > 0 else wl.nrhs
    stream = torch.cuda.current_stream()
    # ---- single-launch stencil table (north_star: >= 70 % of HBM peak on single-RHS fp32 / fp64)
    table = {}
    for pname, n in (("f32", 1), ("f64", 1), ("f32", nrhs), ("bf16", 1)):
        p = PRECS[pname]
        a = t.alloc_field(p, n)
        b = t.alloc_field(p, n)
        a.view(torch.int16)[:] = 0x3C00 if pname == "bf16" else 0
        if pname != "bf16":
            (a.view(torch.float32) if pname == "f32" else a.view(torch.float64)).normal_()
        reps = 50
        for _ in range(5):
            t.dslash(tsm.OP_D_EO, p, n, a, b)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(reps):
            t.dslash(tsm.OP_D_EO, p, n, a, b)
            t.dslash(tsm.OP_D_OE, p, n, b, a)
        e1.record(stream)
        torch.cuda.synchronize()
        us = e0.elapsed_time(e1) * 1e3 / (2 * reps)
        by = stencil_bytes_per_site(pname, wl.reconstruct, n, 0) * (wl.V // 2) * n
        table[f"{pname}_nrhs{n}"] = {"us": us, "algorithmic_GBs": by / us / 1e3, "frac_of_measured_peak": by / us / 1e3 / peak,
                                     "frac_of_8000": by / us / 1e3 / 8000.0, "gflops": 1320.0 * (wl.V // 2) * n / us / 1e3}
        del a, b
    out["dslash"] = table

    # ---- the same step with bf16-storage spinors (reading A15: fp32 is the headline, bf16 storage is reported beside it)
    if prec_name == "f32":
        ids = list(range(900000, 900000 + nrhs))
        t.solve(wl.noise_seed, ids, tsm.BF16, wl.lp_tol, wl.lp_iters, slot=1)
        rc_b, info_b = t.solve(wl.noise_seed, ids, tsm.BF16, wl.lp_tol, wl.lp_iters, slot=1, want_true_resid=True)
        out["lp_bf16_storage"] = {"solves_per_s": nrhs / info_b[0]["secs"], "secs_batch": info_b[0]["secs"], "iters": info_b[0]["iters"],
                                  "true_resid_max": max(i["rel_resid_true"] for i in info_b),
                                  "note": "solve only (no contraction); p, t, w in bf16, x, r and all sums fp32/fp64"}

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
    # algorithmic bytes per site of the full lattice and source: s once (eta is regenerated, never read);
    # derivative: s once + the 8 links of the site
    n_g = 18 if prec_name == "f64" else wl.reconstruct
    by_site = {5: 24 * w_sol, 6: 24 * w_sol + 8 * n_g * (8 if prec_name == "f64" else 4), 7: 24 * w_sol, 8: 48 * w_sol, 9: 24 * w_sol}
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
        out["tsm_loop_set"] = {"seconds": secs, "n_hp": wl.n_hp, "n_lp": wl.n_lp, "rc": rc,
                               "finite": bool(np.isfinite(loops.view(np.float64)).all())}
        rc, info = t.solve(wl.noise_seed, list(range(min(nrhs, wl.n_hp))), tsm.F64, wl.hp_tol, 5000, slot=0, want_true_resid=True)
        out["hp_solve"] = {"iters": [i["iters"] for i in info], "secs_batch": info[0]["secs"],
                           "true_resid_max": max(i["rel_resid_true"] for i in info)}
        # N4: the same HP solves as fp64 defect correction around the fp32 CG, and Eq. 2.4 with them
        rc, info = t.solve(wl.noise_seed, list(range(min(nrhs, wl.n_hp))), tsm.MIXED, wl.hp_tol, 5000, slot=0, want_true_resid=True)
        out["hp_solve_mixed"] = {"iters_fp32_total": [i["iters"] for i in info], "secs_batch": info[0]["secs"],
                                 "true_resid_max": max(i["rel_resid_true"] for i in info)}
        t.set_hp_precision(tsm.MIXED)
        loops_m, secs_m, rc_m = t.run_loop_set(wl.noise_seed, wl.n_hp, wl.n_lp, prec, wl.lp_tol, wl.lp_iters, hp_tol=wl.hp_tol,
                                               hp_max_iter=5000, nrhs=nrhs, with_derivative=wl.derivative)
        t.set_hp_precision(tsm.F64)
        out["tsm_loop_set_mixed_hp"] = {"seconds": secs_m, "rc": rc_m,
                                        "max_rel_diff_to_fp64_hp": float(np.abs(loops_m - loops).max() / np.abs(loops).max())}

    # ---- the oracle on this box's host cores, bounded sample
    if not args.no_cpu_baseline:
        import oracle
        oracle.build()
        tcpu, detail = oracle_sample(wl, U)
        t0 = time.perf_counter()
        oracle.loops_one_end(wl.dims, wl.kappa, wl.mu, oracle.noise(wl.dims, wl.noise_seed, 0))
        detail["t_one_end_contract_s"] = time.perf_counter() - t0
        if wl.V <= 131072:   # configs 1-3: the same sample on ONE host thread as well
            try:
                import ctypes
                gomp = ctypes.CDLL("libgomp.so.1")
                gomp.omp_set_num_threads(1)
                t1, d1 = oracle_sample(wl, U)
                gomp.omp_set_num_threads(oracle.n_threads())
                detail["one_thread"] = {"solves_per_s": 1.0 / t1, "t_per_cg_iteration_s": d1["t_per_cg_iteration_s"]}
            except OSError:
                pass
        t0 = time.perf_counter()
        oracle.loops_gen_one_end(wl.dims, wl.t_boundary, wl.kappa, U, oracle.noise(wl.dims, wl.noise_seed, 0))
        detail["t_gen_one_end_contract_s"] = time.perf_counter() - t0
        out["cpu_baseline"] = {"value": 1.0 / tcpu, "unit": UNIT, "cores": oracle.n_threads(), "kind": "oracle",
                               "sample": ("1 source: source preparation, 1- and 3-iteration CG solves, reconstruction, residual and one "
                                          f"contraction pass run in full; the {detail['iterations_extrapolated_to']}-iteration solve "
                                          "extrapolated linearly in the iteration count"),
                               "detail": detail}
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", type=int, default=5)
    ap.add_argument("--nrhs", type=int, default=0, help="sources per batch (default: the workload's; other values are profiling aids, not the headline)")
    ap.add_argument("--skip-extras", action="store_true", help="only the timed steps (no e2e/table/full set/oracle)")
    ap.add_argument("--no-full-set", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    wl = W.WORKLOADS[args.workload]
    if args.impl == "reference":
        run_reference(args, wl)
    else:
        run_ours(args, wl)


if __name__ == "__main__":
    main()
