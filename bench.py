#!/usr/bin/env python
"""bench.py -- the headline benchmark of this repository (contract: task prompt / DESIGN.md "Measurement").

Metric (BASELINE.json): OCI fp64 cell-solves/s, seconds per converged time step and iterations, OCI vs the GPU SI
sweep, across a dt sweep, on one B200.

Workload: BASELINE.json configs[4] ("config 5"): single group, S16 (n = 64), 65536 cells, per-cell sigma_t
log-uniform in [0.01, 100]/cm, c ~ U[0.5, 0.999], dt sweep {1, 1e-1, 1e-2, 1e-3, 1e-4} -- the config the metric's
"OCI vs GPU SI ... across a dt sweep" is spelled out on, and the largest one (2.1 GB of per-cell inverses, 17x the
L2, so no L2 flush is needed between iterations). Synthetic, seeded (workloads.config5, seed 1005).

A "step" is one converged time step = the whole hot path: a1+a2 assemble + eliminate every cell
(the time step size changes every step, cycling through the sweep, so the matrices really do change), a3 constant
RHS, a4-a7 fused OCI iterations until max|dphi| < 1e-8 (residual read on the host once every 8 iterations), a8
advance. value = J x (iterations performed) / device time, summed over the K timed steps.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

N > 1 (launched under torchrun, one rank per GPU): independent replicas of the same problem (DESIGN.md "Multi-GPU:
replicas only"), barrier + max-over-ranks time, value = all ranks' cell-solves / that time, "scaling": "weak".
--impl reference times the CPU oracle (oracle/, unmodified) on the host cores on bounded samples of the same
workload.
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
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

import workloads as W  # noqa: E402

SWEEP = [1.0, 1e-1, 1e-2, 1e-3, 1e-4]
TOL = 1e-8
CHECK_EVERY = 8
MAX_ITERS = 4000
METRIC = "oci_cell_solves_per_s"
UNIT = "cell-solves/s"
# `traffic` (dram__bytes_read.sum + dram__bytes_write.sum per launch, from `ncu --set full`) is read from
# profiles/r03_kernel_traffic.csv, which records for every capture the hash of the kernel's source files; a value is
# printed only if that hash equals the hash of the sources this run was built from (ncu_traffic() below).
TRAFFIC_FILE = "profiles/r03_kernel_traffic.csv"
KERNEL_SOURCES = {   # kernel -> the files (under paper_2503_00264_b200/csrc/) its code lives in
    "oci_iterate_wpc_kernel": ["iterate.cu", "common.cuh"],
    "factor_wc2_kernel": ["factor.cu", "common.cuh"],
    "st_iterate_pipe_kernel": ["structured.cu", "common.cuh"],
}
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # SMs x DFMA/clk/SM (ncu: sm__sass_thread_inst_executed_op_dfma_pred_on
                                                    # .sum.peak_sustained = 64 per SM) x 2 flop x clocks.max.sm


def measured_peaks():
    f = ROOT / "MEASURED_PEAKS.json"
    if f.exists():
        try:
            d = json.loads(f.read_text())
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def hbm_roofline(achieved, peak, **extra):
    """An HBM roofline object. MEASURED_PEAKS.json's hbm_gbs is a COPY bandwidth (half reads, half writes); the iterate
    kernels are 98 % reads and have been measured a few per cent above it with ncu DRAM traffic equal to the algorithmic
    bytes, so the figure is a yardstick, not a ceiling: a fraction above 1 is flagged here instead of passing silently
    (well above 1 would mean reuse out of the L2 or a wrong byte count)."""
    r = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak}
    r.update(extra)
    if achieved > peak:
        r["frac_above_1"] = ("achieved exceeds the copy-measured peak: read-dominated stream against a read+write "
                             "copy figure; check `traffic` against the algorithmic bytes" if achieved <= 1.2 * peak else
                             "achieved is more than 1.2 x the measured peak: L2 reuse or a wrong byte count, not HBM speed")
    return r


def source_hash(kernel: str) -> str:
    import hashlib
    h = hashlib.sha256()
    for name in KERNEL_SOURCES[kernel]:
        h.update((ROOT / "paper_2503_00264_b200" / "csrc" / name).read_bytes())
    return h.hexdigest()[:16]


def ncu_traffic(kernel: str, workload: str):
    """(bytes per launch or None, note). None unless the capture on file was taken with exactly these kernel sources."""
    f = ROOT / TRAFFIC_FILE
    if not f.exists():
        return None, f"{TRAFFIC_FILE} missing"
    want = source_hash(kernel)
    stale = None
    for line in f.read_text().splitlines():
        c = [x.strip() for x in line.split(",")]
        if len(c) < 6 or c[0] != kernel or c[2] != workload:
            continue
        if c[1] == want:
            return int(c[3]) + int(c[4]), f"{TRAFFIC_FILE}: {c[5]} (source hash {want})"
        stale = c[1]
    if stale:
        return None, f"capture on file is of other sources (hash {stale}, built from {want}): not quoted"
    return None, f"no capture of {kernel} on {workload} in {TRAFFIC_FILE}"


def structured_bytes_per_cell_solve(n: int, G: int) -> int:
    """DESIGN.md section 5 (structured cell solve): L^-1 blocks, two of their four rows (16 n) + c (8n)
    + neighbour edge flux (4n) + Psi write (8n) + C^-1 (128 G^2) + K (8 G^2) + dx (8) + phi read/write (64 G)."""
    return 36 * n + 136 * G * G + 64 * G + 8


def algorithmic_bytes_per_cell_solve(n: int, G: int) -> int:
    """A_j^{-1} (8 n^2) + c (8n) + neighbour edge flux (4n) + index/perm (4n) + Psi write (8n) +
    phi old/new (64 G)."""
    return 8 * n * n + 24 * n + 64 * G


def max_over_ranks(value: float, device="cuda") -> float:
    """Timing contract: the slowest rank's time. No-op without an initialised process group (N = 1)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, J: int, iterations_per_rank: int, ms: float) -> float:
    """Replicas only: every rank solves the same problem, so the job did world x J x iterations
    cell-solves in the slowest rank's time."""
    return world * J * iterations_per_rank / (ms * 1e-3)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.25)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
                for nm, val in zip(names, r[4:8]):
                    if val.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


# ---------------------------------------------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline and --impl reference): the ONLY places this file touches oracle/
# ---------------------------------------------------------------------------------------------------------------
def oracle_pass(problem, dts):
    """One converged time step per dt (factor + iterate to convergence + advance) with the unmodified oracle."""
    from oracle import Oracle, num_threads
    o = Oracle(problem, dt=dts[0])
    solves, t0 = 0, time.perf_counter()
    per_dt = []
    for dt in dts:
        t1 = time.perf_counter()
        o.set_dt(dt)
        o.factor()
        it, _ = o.oci_step(tol=TOL, max_iters=MAX_ITERS)
        per_dt.append({"dt": dt, "iters": int(it), "s": time.perf_counter() - t1})
        solves += problem.J * it
    return solves, time.perf_counter() - t0, per_dt, num_threads()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    full = W.config5()
    sample = full.head(args.ref_cells)
    from oracle import Oracle, num_threads
    o = Oracle(sample, dt=SWEEP[0])
    step_s, solves = [], 0
    for i in range(args.warmup + args.steps):
        dt = SWEEP[i % len(SWEEP)]
        t = time.perf_counter()
        o.set_dt(dt)
        o.factor()
        it, _ = o.oci_step(tol=TOL, max_iters=MAX_ITERS)
        el = time.perf_counter() - t
        if i >= args.warmup:
            step_s.append(el)
            solves += sample.J * it
    total = sum(step_s)
    value = solves / total
    which = "all" if sample.J == full.J else f"first {sample.J} of"
    desc = f"{which} {full.J} cells of config 5, one converged time step per timed step, dt cycling {SWEEP}"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[4] (config 5): G1 S16 n=64 J=65536, dt sweep", "sample": desc},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": num_threads(), "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ---------------------------------------------------------------------------------------------------------------
# GPU arm
# ---------------------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2503_00264_b200 import OCISolver

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    p = W.config5()
    n, J, G = p.n, p.J, p.G
    oci = OCISolver(p, dt=SWEEP[0], device=f"cuda:{local}")
    si = OCISolver(p, dt=SWEEP[0], device=f"cuda:{local}")
    K, Wm = args.steps, args.warmup

    def oci_step(i, solver=oci):
        solver.set_dt(SWEEP[i % len(SWEEP)])
        return solver.step(tol=TOL, max_iters=MAX_ITERS, check_every=CHECK_EVERY)

    # ---- device-resident leg -------------------------------------------------------------------------------
    for i in range(Wm):
        oci_step(i)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    per_dt = {dt: {"dt": dt, "oci_iters": [], "oci_ms": [], "factor_ms": [], "iter_kernel_ms": []} for dt in SWEEP}
    iters_total = launches = 0
    kernel_ms_total = 0.0
    barrier()
    with ClockSampler(local) as clocks:
        ev0.record()
        for i in range(Wm, Wm + K):
            t = time.perf_counter()
            it, conv, _ = oci_step(i)
            oci.synchronize()                      # (the advance kernel may still be in flight when oci_step returns)
            el = (time.perf_counter() - t) * 1e3   # host time of the call = its device time + launch gaps
            kms, ln = oci.last_timing(1)
            fms, _ = oci.last_timing(0)
            d = per_dt[SWEEP[i % len(SWEEP)]]
            d["oci_iters"].append(it); d["oci_ms"].append(el); d["factor_ms"].append(fms); d["iter_kernel_ms"].append(kms)
            iters_total += it
            launches += ln
            kernel_ms_total += kms
        ev1.record()
        barrier()
    ms_total = max_over_ranks(ev0.elapsed_time(ev1))
    value = whole_job_value(world, J, iters_total, ms_total)

    # ---- structured cell solve, same sequence, reported beside (not part of `value`) -----------
    st = OCISolver(p, dt=SWEEP[0], device=f"cuda:{local}", options={"solve_mode": 1})
    for i in range(Wm):
        oci_step(i, st)
    st_iters = 0
    st_kernel_ms = 0.0
    st_factor_ms = []
    barrier()
    ev0.record()
    for i in range(Wm, Wm + K):
        t = time.perf_counter()
        it, conv, _ = oci_step(i, st)
        st.synchronize()
        el = (time.perf_counter() - t) * 1e3
        d = per_dt[SWEEP[i % len(SWEEP)]]
        d.setdefault("st_iters", []).append(it); d.setdefault("st_ms", []).append(el)
        st_iters += it
        st_kernel_ms += st.last_timing(1)[0]
        st_factor_ms.append(st.last_timing(0)[0])
    ev1.record()
    barrier()
    st_ms_total = max_over_ranks(ev0.elapsed_time(ev1))
    st_diff = float((oci.scalar_flux() - st.scalar_flux()).abs().max().item())

    # ---- SI comparator, same sequence (reported beside, not part of `value`) ----------------------------------
    for i in range(0 if args.no_si else Wm):
        si.set_dt(SWEEP[i % len(SWEEP)]); si.si_step(tol=TOL, max_iters=MAX_ITERS, check_every=CHECK_EVERY)
    for i in range(Wm, Wm if args.no_si else Wm + K):
        dt = SWEEP[i % len(SWEEP)]
        si.set_dt(dt)
        torch.cuda.synchronize(); t = time.perf_counter()
        it, conv, _ = si.si_step(tol=TOL, max_iters=MAX_ITERS, check_every=CHECK_EVERY)
        si.synchronize()
        el = (time.perf_counter() - t) * 1e3
        per_dt[dt].setdefault("si_iters", []).append(it)
        per_dt[dt].setdefault("si_ms", []).append(el)
    diff = None if args.no_si else float((oci.scalar_flux() - si.scalar_flux()).abs().max().item())
    # the same SI iteration with the sweep evaluated as a parallel scan (NOT north_star's comparator)
    if not args.no_si:
        si2 = OCISolver(p, dt=SWEEP[0], device=f"cuda:{local}", options={"si_sweep": 1})
        for i in range(Wm + K):
            dt = SWEEP[i % len(SWEEP)]
            si2.set_dt(dt)
            torch.cuda.synchronize(); t = time.perf_counter()
            si2.si_step(tol=TOL, max_iters=MAX_ITERS, check_every=CHECK_EVERY)
            si2.synchronize()
            if i >= Wm:
                per_dt[dt].setdefault("si_scan_ms", []).append((time.perf_counter() - t) * 1e3)
        del si2

    # ---- end-to-end leg: host buffers through oci_step_host, copies inside the timed region ------------------
    e2e = OCISolver(p, dt=SWEEP[0], device=f"cuda:{local}")
    q_host = torch.from_numpy(np.ascontiguousarray(p.q)).pin_memory()
    phi_host = torch.empty((J, G, 4), dtype=torch.float64).pin_memory()
    for i in range(Wm):
        e2e.set_dt(SWEEP[i % len(SWEEP)])
        e2e.step_host(0, q_host, phi_host, tol=TOL, max_iters=MAX_ITERS, check_every=CHECK_EVERY)
    barrier()
    t0 = time.perf_counter()
    e2e_iters = 0
    for i in range(Wm, Wm + K):
        e2e.set_dt(SWEEP[i % len(SWEEP)])
        it, _, _ = e2e.step_host(0, q_host, phi_host, tol=TOL, max_iters=MAX_ITERS, check_every=CHECK_EVERY)
        e2e_iters += it
    barrier()
    e2e_s = max_over_ranks(time.perf_counter() - t0)
    e2e_value = whole_job_value(world, J, e2e_iters, e2e_s * 1e3)
    nbytes = J * G * 4 * 8

    if rank != 0:
        return
    # ---- roofline of the dominant kernel (oci_iterate_wpc_kernel<2,0>), from the timed region -----------------------
    peak, peak_src = measured_peaks()
    launch_ms = kernel_ms_total / max(iters_total, 1)
    alg_bytes = algorithmic_bytes_per_cell_solve(n, G) * J
    achieved = alg_bytes / (launch_ms * 1e-3) / 1e9
    wl = "config5"
    tr, tr_note = ncu_traffic("oci_iterate_wpc_kernel", wl)
    roofline = hbm_roofline(achieved, peak, kernel="oci_iterate_wpc_kernel<2,0>", traffic=tr, traffic_source=tr_note,
                            peak_source=peak_src, algorithmic_bytes_per_launch=alg_bytes, avg_launch_ms=launch_ms,
                            kernel_share_of_step=kernel_ms_total / ms_total)
    factor_ms = statistics.mean(x for d in per_dt.values() for x in d["factor_ms"])
    exec_flops, alg_flops = 2.0 * n ** 3 * J, (2.0 / 3.0) * n ** 3 * J
    factor_tf = exec_flops / (factor_ms * 1e-3) / 1e12
    tr, tr_note = ncu_traffic("factor_wc2_kernel", wl)
    roofline_factor = {"bound": "alu", "kernel": "factor_wc2_kernel", "achieved": factor_tf, "peak": FP64_PEAK_TFLOPS,
                       "unit": "TFLOP/s", "frac": factor_tf / FP64_PEAK_TFLOPS,
                       "frac_algorithmic": alg_flops / (factor_ms * 1e-3) / 1e12 / FP64_PEAK_TFLOPS,
                       "executed_flops": exec_flops, "algorithmic_flops": alg_flops,
                       "flops_note": "executed = 2 n^3 per cell (Gauss-Jordan with partial pivoting carried to the inverse, "
                                     "what the kernel does); algorithmic = (2/3) n^3 per cell (the LU of SURVEY 8(d))",
                       "traffic": tr, "traffic_source": tr_note,
                       "peak_source": "derived: 148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz (DESIGN.md section 7); DMMA "
                                      "reaches the same 64 FMA/clk/SM (profiles/r02_fp64_pipe.md)",
                       "avg_launch_ms": factor_ms, "kernel_share_of_step": factor_ms * K / ms_total}

    st_launch_ms = st_kernel_ms / max(st_iters, 1)
    st_bytes = structured_bytes_per_cell_solve(n, G) * J
    st_achieved = st_bytes / (st_launch_ms * 1e-3) / 1e9
    st_tr, st_tr_note = ncu_traffic("st_iterate_pipe_kernel", wl)
    structured = {
        "what": "SURVEY 8(f) row f1: structured cell solve A_j = D - U V^T (solve_mode = 1), same steps, same stop rule",
        "value": whole_job_value(world, J, st_iters, st_ms_total), "unit": UNIT, "ms_per_step": st_ms_total / K,
        "iterations_total": st_iters, "factor_ms": statistics.mean(st_factor_ms),
        "max_abs_phi_minus_dense_path": st_diff,
        "roofline": {"bound": "hbm", "kernel": "st_iterate_pipe_kernel<0,1>", "achieved": st_achieved, "peak": peak, "unit": "GB/s",
                     "frac": st_achieved / peak, "traffic": st_tr, "traffic_source": st_tr_note, "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": st_bytes, "avg_launch_ms": st_launch_ms,
                     "kernel_share_of_step": st_kernel_ms / st_ms_total},
    }

    # ---- CPU oracle on the same workload (bounded sample), rank 0, N = 1 only ---------------------------------------
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        sample = p.head(args.cpu_cells)
        solves = secs = 0.0
        passes = 0
        while secs < args.cpu_seconds and passes < 64:   # bounded: about 10-30 s of host work
            s_, t_, cpu_dt, cores = oracle_pass(sample, SWEEP)
            solves += s_; secs += t_; passes += 1
        cpu = {"value": solves / secs, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"first {sample.J} of {J} cells of config 5, {passes} pass(es) of one converged time step at each "
                         f"dt of {SWEEP} (factor + iterate + advance), {secs:.1f} s",
               "iters": [d["iters"] for d in cpu_dt]}

    per_config = true_error = as_specified = None
    if world == 1 and not args.quick:
        per_config = run_per_config(f"cuda:{local}", peak)
        true_error = run_true_error(p, f"cuda:{local}")
        as_specified = run_as_specified(p, f"cuda:{local}", args.no_si)

    table = []
    for dt in SWEEP:
        d = per_dt[dt]
        if not d["oci_iters"]:
            continue
        table.append({"dt": dt, "oci_iters": d["oci_iters"], "si_iters": d.get("si_iters"),
                      "oci_ms_per_step": statistics.mean(d["oci_ms"]), "oci_factor_ms": statistics.mean(d["factor_ms"]),
                      "oci_iter_kernel_ms": statistics.mean(d["iter_kernel_ms"]),
                      "structured_iters": d.get("st_iters"),
                      "structured_ms_per_step": statistics.mean(d["st_ms"]) if d.get("st_ms") else None,
                      "si_ms_per_step": statistics.mean(d["si_ms"]) if d.get("si_ms") else None,
                      "si_scan_variant_ms_per_step": statistics.mean(d["si_scan_ms"]) if d.get("si_scan_ms") else None})
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[4] (config 5): G1 S16 n=64 J=65536, one converged time step per "
                               "step, dt cycling {1,1e-1,1e-2,1e-3,1e-4}, tol 1e-8, check_every 8",
                   "J": J, "N": p.N, "G": G, "n": n, "l2_flush": "not needed: 2.1 GB of factors streamed per iteration (17x L2)",
                   "parallelism": "replicas" if world > 1 else "single"},
        "clocks": clocks.summary(),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "roofline_factor": roofline_factor,
        "structured": structured,
        "cpu_baseline": cpu,
        "oci_vs_si": table,
        "as_specified": as_specified,
        "true_error": true_error,
        "per_config": per_config,
        "max_abs_phi_oci_minus_si": diff,
        "iterations_total": iters_total,
    }
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


# ---------------------------------------------------------------------------------------------------------------
# Legs reported beside the headline (none of them is part of `value`)
# ---------------------------------------------------------------------------------------------------------------
def empty_launch_us(solver, torch, n=200):
    """Device time per launch of an empty kernel in a stream of back-to-back launches (the floor of one iteration)."""
    solver.debug_empty_launches(20)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    solver.debug_empty_launches(n)
    e1.record()
    torch.cuda.synchronize()
    return 1e3 * e0.elapsed_time(e1) / n


def run_per_config(device, peak):
    """BASELINE.json configs 1-4 (+ variant 4b), each run as configured for a few steps on the dense path (the
    structured path beside it): iterations OCI vs SI, ms per converged step, us per iteration, factor ms, and for the
    HBM-bound ones (3, 4) the roofline fraction of the iterate kernel; for the L2-resident ones (1, 2) the iteration
    time against the measured empty-launch floor (no roofline fraction is meaningful there)."""
    import torch
    from paper_2503_00264_b200 import OCISolver
    cases = [("config1", W.config1(), 0.1, 5), ("config2@dt=1", W.config2(dt=1.0), 1.0, 3),
             ("config2@dt=0.1", W.config2(dt=0.1), 0.1, 5), ("config2@dt=0.01", W.config2(dt=0.01), 0.01, 5),
             ("config3", W.config3(), 1e-8, 5), ("config4", W.config4(), 1e-3, 5),
             ("config4b(v=1000)", W.config4(v=1000.0), 1e-3, 3)]
    out = []
    floor = None
    for name, p, dt, steps in cases:
        row = {"config": name, "J": p.J, "N": p.N, "G": p.G, "n": p.n, "dt": dt, "steps": steps}
        for key, scheme, opts in (("oci_dense", 0, {}), ("oci_structured", 0, {"solve_mode": 1}), ("si", 1, {})):
            sol = OCISolver(p, dt=dt, device=device, options=opts)
            if floor is None:
                floor = empty_launch_us(sol, torch)
            if scheme == 0:
                sol.factor()                       # warm-up of the factor kernel; re-done (timed) below
                sol.set_dt(dt * (1 + 1e-12)); sol.factor()
                row[key + "_factor_ms"] = sol.last_timing(0)[0]
            iters, ms, kms = [], [], []
            for st in range(steps):
                sol.set_source(p.source_at_step(st))
                torch.cuda.synchronize(); t = time.perf_counter()
                it, conv, _ = (sol.step if scheme == 0 else sol.si_step)(tol=p.tol, max_iters=20000, check_every=CHECK_EVERY)
                sol.synchronize()
                ms.append((time.perf_counter() - t) * 1e3)
                iters.append(it)
                kms.append(sol.last_timing(1 if scheme == 0 else 2)[0])
            row[key + "_iters"] = iters
            row[key + "_ms_per_step"] = statistics.mean(ms)
            row[key + "_us_per_iteration"] = 1e3 * sum(kms) / max(sum(iters), 1)
            if key == "oci_dense":
                us = row[key + "_us_per_iteration"]
                if p.J * p.n * p.n * 8 > (126 << 20):     # factors exceed the L2: HBM roofline
                    gbs = algorithmic_bytes_per_cell_solve(p.n, p.G) * p.J / (us * 1e-6) / 1e9
                    row["oci_dense_roofline"] = hbm_roofline(gbs, peak)
                else:
                    row["oci_dense_iteration_over_launch_floor"] = us / floor
                fl = 2.0 * p.n ** 3 * p.J
                row["oci_dense_factor_tflops_executed"] = fl / (row[key + "_factor_ms"] * 1e-3) / 1e12
                row["oci_dense_factor_frac_of_fp64_peak_executed"] = row["oci_dense_factor_tflops_executed"] / FP64_PEAK_TFLOPS
                row["oci_dense_factor_frac_of_fp64_peak_algorithmic"] = row["oci_dense_factor_frac_of_fp64_peak_executed"] / 3.0
            del sol
        out.append(row)
    return {"empty_launch_us": floor, "rows": out}


def run_true_error(p, device):
    """what the stop rule leaves. Per dt of the sweep, first time step from the initial condition:
    |phi(tol 1e-8, rule 0) - phi(tol 1e-13)|_inf, for OCI and SI, and the same with the paper's rule (Eq. 12-13)."""
    from paper_2503_00264_b200 import OCISolver
    rows = []
    for dt in SWEEP:
        tight = OCISolver(p, dt=dt, device=device)
        it_t, _, _ = tight.step(tol=1e-13, max_iters=20000, check_every=CHECK_EVERY, advance=False)
        ref = tight.scalar_flux()
        row = {"dt": dt, "tight_iters": it_t}
        for key, fn, rule in (("oci_rule0", "step", 0), ("oci_rule1_paper", "step", 1), ("si_rule0", "si_step", 0)):
            s_ = OCISolver(p, dt=dt, device=device)
            it, _, _ = getattr(s_, fn)(tol=TOL, max_iters=20000, check_every=CHECK_EVERY, stop_rule=rule, advance=False)
            row[key] = {"iters": it, "true_error_inf": float((s_.scalar_flux() - ref).abs().max().item())}
            del s_
        rows.append(row)
        del tight
    return rows


def run_as_specified(p, device, no_si):
    """BASELINE.json config 5 as written: for every dt of the sweep 10 time steps; a1 + a2 once per dt (the matrices do
    not change inside a block)."""
    import torch
    from paper_2503_00264_b200 import OCISolver
    oci, si = OCISolver(p, dt=SWEEP[0], device=device), OCISolver(p, dt=SWEEP[0], device=device)
    rows, tot_ms, tot_it = [], 0.0, 0
    for dt in SWEEP:
        row = {"dt": dt, "steps": p.n_steps}
        oci.set_dt(dt)
        torch.cuda.synchronize(); t = time.perf_counter()
        its = [oci.step(tol=TOL, max_iters=MAX_ITERS, check_every=CHECK_EVERY)[0] for _ in range(p.n_steps)]
        oci.synchronize()
        row["oci_ms_total"] = (time.perf_counter() - t) * 1e3
        row["oci_iters"] = its
        row["oci_ms_per_step"] = row["oci_ms_total"] / p.n_steps
        tot_ms += row["oci_ms_total"]; tot_it += sum(its)
        if not no_si:
            si.set_dt(dt)
            torch.cuda.synchronize(); t = time.perf_counter()
            its = [si.si_step(tol=TOL, max_iters=MAX_ITERS, check_every=CHECK_EVERY)[0] for _ in range(p.n_steps)]
            si.synchronize()
            row["si_ms_per_step"] = (time.perf_counter() - t) * 1e3 / p.n_steps
            row["si_iters"] = its
        rows.append(row)
    return {"what": "config 5 as specified: 10 steps per dt, factors computed once per dt", "rows": rows,
            "oci_cell_solves_per_s": p.J * tot_it / (tot_ms * 1e-3), "oci_ms_total": tot_ms, "oci_iterations_total": tot_it}


# ---------------------------------------------------------------------------------------------------------------
# the paper's own timing experiment (Figs. 7-8) on this GPU. Not the headline.
# ---------------------------------------------------------------------------------------------------------------
def run_table2(args):
    """Two-group problem of Table 2, L = 100 cm, vacuum, psi_0 = 0, first time step, delta =
    Sigma_t,2 dx swept through dx, S16 and S32, dt = 10 s and 0.1 s. Like the paper, the time is that of the convergence
    loop only (CUDA events around the iteration kernels; no assembly / elimination), stop rule = the paper's Eq. 12."""
    import torch
    from paper_2503_00264_b200 import OCISolver
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --table2 needs a CUDA device")
    sig2, L, eps = 0.45468, 100.0, 1e-8
    rows = []
    for dt in (10.0, 0.1):
        for N in (16, 32):
            for delta in (10.0, 4.0, 1.0, 0.4, 0.1, 0.04, 0.01):
                J = max(2, int(round(L * sig2 / delta)))
                p = W.table2(J, N, dt, L)
                row = {"dt": dt, "N": N, "n": p.n, "J": J, "delta": sig2 * L / J}
                for name, scheme, opts in (("oci_dense", 0, {}), ("oci_structured", 0, {"solve_mode": 1}), ("si", 1, {})):
                    best = None
                    for rep in range(2):     # second repetition is warm
                        s = OCISolver(p, options=opts)
                        if scheme == 0:
                            s.factor()
                            it, conv, _ = s.step(tol=eps, max_iters=60000, check_every=16, stop_rule=1, advance=False)
                            ms = s.last_timing(1)[0]
                        else:
                            it, conv, _ = s.si_step(tol=eps, max_iters=60000, check_every=16, stop_rule=1, advance=False)
                            ms = s.last_timing(2)[0]
                        best = ms if best is None else min(best, ms)
                        del s
                    row[name + "_iters"] = it
                    row[name + "_converged"] = bool(conv)
                    row[name + "_loop_ms"] = best
                row["speedup_dense_over_si"] = row["si_loop_ms"] / row["oci_dense_loop_ms"]
                row["speedup_structured_over_si"] = row["si_loop_ms"] / row["oci_structured_loop_ms"]
                rows.append(row)
    print(json.dumps({"experiment": "table2 delta sweep (PAPER.md:510-520, Figs. 7-8)", "unit": "ms per convergence loop",
                      "stop_rule": "Eq. 12-13, eps = 1e-8", "rows": rows}))


def run_factor_ab(args):
    """The a1 + a2 kernels for n = 64 side by side on config 5 (the DMMA decision): the production
    kernel (two warps per cell, look-ahead, DMMA), the one-warp-per-cell kernel with its rank-8 updates as DMMA and as
    DFMA (everything else identical), and the generic one-CTA-per-cell kernel. One JSON line."""
    import torch
    from paper_2503_00264_b200 import OCISolver
    p = W.config5(dt=1e-3)
    n, J = p.n, p.J
    rows = []
    for name, opts in (("factor_wc2_kernel: 2 warps/cell, look-ahead, DMMA, panels paired [production]", {}),
                       ("factor_wc2_kernel: the same, one rank-8 pass per panel", {"factor_update": 1}),
                       ("factor_wc_kernel<DMMA>: 1 warp/cell", {"factor_kernel": 4, "factor_update": 1}),
                       ("factor_wc_kernel<DFMA>: 1 warp/cell", {"factor_kernel": 4, "factor_update": 0}),
                       ("factor_gj_kernel: generic, one CTA per cell, DFMA", {"factor_kernel": 0})):
        s = OCISolver(p, options=opts)
        ts = []
        for r in range(4):
            s.set_dt(p.dt * (1 + 1e-9 * (r + 1)))
            assert s.factor() == 0
            ts.append(s.last_timing(0)[0])
        ms = min(ts[1:])
        rows.append({"kernel": name, "ms": ms, "tflops_executed": 2.0 * n ** 3 * J / (ms * 1e-3) / 1e12,
                     "frac_of_fp64_peak_executed": 2.0 * n ** 3 * J / (ms * 1e-3) / 1e12 / FP64_PEAK_TFLOPS})
        del s
    print(json.dumps({"experiment": "factor kernels for n = 64 on config 5 (J = 65536)", "rows": rows}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--cpu-cells", type=int, default=65536, help="cells of the cpu_baseline sample")
    ap.add_argument("--cpu-seconds", type=float, default=10.0, help="minimum host time spent on the cpu_baseline sample")
    ap.add_argument("--ref-cells", type=int, default=65536,
                    help="cells per step of --impl reference (default: all of config 5, the workload of the GPU arm)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-si", action="store_true", help="skip the SI comparator leg (profiling runs)")
    ap.add_argument("--quick", action="store_true",
                    help="skip the per_config / true_error / as_specified legs (profiling runs)")
    ap.add_argument("--factor-ab", action="store_true",
                    help="instead of the headline benchmark: the n = 64 factor kernels side by side (DMMA vs DFMA evidence)")
    ap.add_argument("--table2", action="store_true",
                    help="instead of the headline benchmark: the paper's Table-2 delta sweep, OCI vs SI (SURVEY 8f row f3)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.factor_ab:
        run_factor_ab(args)
    elif args.table2:
        run_table2(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
