#!/usr/bin/env python
"""bench.py - transit-model evaluations/s of the CUDA library on the BASELINE.json workloads.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 0..4] [--precision fp64|fp32]
    python bench.py --impl reference ...          # the CPU oracle, as it stands, on the host cores

A "step" is one pass of the whole hot path over one batch of synthetic input:
rr_build_ld_table (kernel 1) + rr_evaluate (per-pv prep, kernels 2+3 fused; kernel 4's tile table
was built once by rr_set_data, the paper's call pattern PAPER.md:207-218).  Default workload:
config 4 of BASELINE.json (the largest population workload, the one the north-star target is
stated on), fp64.  One JSON line on stdout (rank 0).  See DESIGN.md s8 for every field.

Multi-GPU (torchrun, one process per GPU): the path shards over parameter vectors with no exchange,
so each rank evaluates its own full population (weak scaling) and the only communication is the
barrier and the max-over-ranks of the device time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "transit-model evaluations/sec (pv x time x supersample)"
UNIT = "evaluations/s"
# B200 FP64 FMA pipe = 64 lanes/clk/SM (37.2 TFLOP/s nominal at 148 SMs, 1965 MHz)
FP64_LANES_PER_SM, FP32_LANES_PER_SM, SM_COUNT = 64, 128, 148
# algorithmic FMA-pipe instructions (DFMA/DMUL/DADD; fp32 mode: FFMA-class, with the
# fp64 phase instructions counted twice) per unit of each class of the flux kernel.  Sub-samples in
# merged out-of-window fill runs cost no arithmetic.
ALG_OPS = {
    "fp64": dict(skipped=1, circular=16, eccentric_fixed=24, solver_iter=31, occulting=13,
                 ingress=62),
    "fp32": dict(skipped=4, circular=19, eccentric_fixed=32, solver_iter=24, occulting=11,
                 ingress=61),
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32", "mixed"],
                    help="mixed = fp32 z and Ip*Ap, fp64 averaging / subtraction / flux (PAPER.md:293)")
    ap.add_argument("--npv", type=int, default=None, help="shrink the population (debugging)")
    ap.add_argument("--npt", type=int, default=None, help="shrink the time axis (debugging)")
    ap.add_argument("--table-mode", default="lazy", choices=["lazy", "full", "direct"],
                    help="kernel 1: rows for each pv's k at evaluate time (default), the full table, "
                         "or the paper's direct model (weights at each pv's own k, no k grid)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def workload_config(wl, precision, extra=None):
    cfg = {
        "workload": wl.name, "npv": wl.npv, "npt": wl.npt, "nlc": wl.nlc,
        "supersampling": [int(x) for x in wl.supersampling],
        "evaluations_per_step_per_gpu": wl.evaluations,
        "ld": wl.ld_kind, "nz": wl.model.nz, "ng": wl.model.ng, "nk": wl.model.nk,
        "npb": wl.model.npb, "precision": precision,
    }
    cfg.update(extra or {})
    return cfg


def ncu_traffic(workload: str, precision: str):
    """dram read + write bytes per launch of rr_flux_kernel from the committed ncu capture."""
    try:
        with open(os.path.join(ROOT, "profiles", "flux_kernel_dram_traffic.csv")) as f:
            for line in f.read().splitlines()[1:]:
                w, p, rd, wr, _ = line.split(",")
                if w == workload and p == precision:
                    return int(rd) + int(wr)
    except (OSError, ValueError):
        pass
    return None


# ---- clocks ------------------------------------------------------------------------------------
CLOCK_FIELDS = ["clocks.sm", "clocks.max.sm", "power.draw",
                "clocks_event_reasons.hw_slowdown", "clocks_event_reasons.hw_thermal_slowdown",
                "clocks_event_reasons.sw_thermal_slowdown", "clocks_event_reasons.sw_power_cap"]


class ClockSampler:
    def __init__(self, index: int):
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={','.join(CLOCK_FIELDS)}",
                 "--format=csv,noheader,nounits", "-lms", "50", "-i", str(index)],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, smax, power, reasons = [], [], [], set()
        for line in out.splitlines():
            parts = [p.strip() for p in line.split(",")]
            if len(parts) != len(CLOCK_FIELDS):
                continue
            try:
                sm.append(float(parts[0]))
                smax.append(float(parts[1]))
                power.append(float(parts[2]))
            except ValueError:
                continue
            for name, val in zip(CLOCK_FIELDS[3:], parts[3:]):
                if val.lower().startswith("active"):
                    reasons.add(name.split(".")[-1])
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)),
                "power_w_max": float(max(power)), "samples": len(sm), "reasons": sorted(reasons)}


# ---- the reference arm: the oracle on the host cores ---------------------------------------------
def oracle_rate(wl, target_s: float, nthreads: int = 0):
    """Oracle (table build + evaluate) on the first n pvs of the workload, n calibrated so that
    the run takes about target_s.  Returns (evaluations/s, seconds, n_pv)."""
    import oracle
    om = oracle.OracleModel.from_config(wl.model)

    def run(n):
        sub = wl.subset_pv(np.arange(n))
        t = time.perf_counter()
        om.build_ld_table(sub.ldp(om.mu))
        om.evaluate(sub.times, sub.lc_index, sub.passband_index, sub.supersampling,
                    sub.exposure_time, sub.pv, nthreads=nthreads)
        return time.perf_counter() - t, sub.evaluations

    cores = os.cpu_count() or 1
    n0 = min(wl.npv, max(1, cores))
    dt, ev = run(n0)
    n = int(min(wl.npv, max(n0, n0 * target_s / max(dt, 1e-6))))
    if n > n0:
        dt, ev = run(n)
    return ev / dt, dt, n


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl = workloads.make_workload(args.config, npv=args.npv, npt=args.npt)
    cores = os.cpu_count() or 1
    steps, warm = max(1, args.steps), max(0, args.warmup)
    target = min(10.0, 150.0 / (steps + warm))
    for _ in range(warm):
        oracle_rate(wl, target)
    t_total, ev_total, n_used = 0.0, 0, 0
    for _ in range(steps):
        rate, dt, n = oracle_rate(wl, target)
        t_total += dt
        ev_total += rate * dt
        n_used = n
    value = ev_total / t_total
    sample = f"first {n_used} of {wl.npv} parameter vectors x all {wl.npt} exposures per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warm, "ms_per_step": 1e3 * t_total / steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(wl, "fp64"),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ---- our arm ----------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import paper_2009_08500_b200 as rr
    from paper_2009_08500_b200 import shard

    rank, local_rank, world = shard.env_rank()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        shard.init_process_group("nccl")
    rr.load()

    precision = {"fp64": rr.RR_FP64, "fp32": rr.RR_FP32, "mixed": rr.RR_MIXED}[args.precision]
    npdt = np.float32 if precision != rr.RR_FP64 else np.float64
    wl = workloads.make_workload(args.config, npv=args.npv, npt=args.npt)
    if rank:   # weak scaling: every rank gets a full population, rotated so that data differ
        sh = (rank * 97) % wl.npv
        wl.pv = np.ascontiguousarray(np.roll(wl.pv, sh, axis=0))
        wl.ld_coeffs = np.ascontiguousarray(np.roll(wl.ld_coeffs, sh, axis=0))

    model = rr.RoadRunner.from_config(wl.model, precision)
    rr.rr_set_table_mode(model.ctx, {"lazy": rr.RR_TABLE_LAZY, "full": rr.RR_TABLE_FULL,
                                     "direct": rr.RR_TABLE_DIRECT}[args.table_mode])
    model.set_data(wl.times, wl.lc_index, wl.passband_index, wl.supersampling, wl.exposure_time)
    ldp_h = np.ascontiguousarray(wl.ldp(model.mu), dtype=npdt)
    ldp = torch.as_tensor(ldp_h).to(dev)
    pv = torch.as_tensor(wl.pv).to(dev)
    flux = torch.empty((wl.npv, wl.npt), dtype=model.flux_dtype, device=dev)
    status = torch.empty(wl.npv, dtype=torch.int32, device=dev)
    ctx = model.ctx
    npv = wl.npv

    def step():
        rr.rr_build_ld_table(ctx, ldp, npv)
        rr.rr_evaluate(ctx, pv, flux, status)

    steps, warm = max(1, args.steps), max(3, args.warmup)
    for _ in range(warm):
        step()
    torch.cuda.synchronize()

    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
    launches0 = rr.rr_launch_count(ctx)
    sampler = ClockSampler(local_rank) if rank == 0 else None
    shard.barrier()
    torch.cuda.synchronize()
    rr.rr_enable_kernel_timing(ctx, True)    # the library's own CUDA events around its kernels
    for s in range(steps):
        ev[s][0].record()
        rr.rr_build_ld_table(ctx, ldp, npv)
        ev[s][1].record()
        rr.rr_evaluate(ctx, pv, flux, status)
        ev[s][2].record()
    torch.cuda.synchronize()
    shard.barrier()
    clocks = sampler.stop() if sampler else None
    launches = rr.rr_launch_count(ctx) - launches0
    ktimes = rr.rr_get_kernel_times(ctx)
    rr.rr_enable_kernel_timing(ctx, False)
    ms_total = ev[0][0].elapsed_time(ev[-1][2])
    ms_table = float(np.mean([e[0].elapsed_time(e[1]) for e in ev]))
    ms_eval = float(np.mean([e[1].elapsed_time(e[2]) for e in ev]))
    ms_flux = ktimes["flux_ms"] / max(1, ktimes["calls"])      # rr_flux_kernel alone
    ms_rows = ktimes["rows_ms"] / max(1, ktimes["calls"])
    ms_total = shard.max_over_ranks(ms_total, dev)
    evals_all = shard.sum_over_ranks(float(wl.evaluations), dev)
    value = evals_all * steps / (ms_total * 1e-3)

    # ---- class counts of one evaluation (outside the timed region) -> algorithmic work
    rr.rr_enable_counters(ctx, True)
    rr.rr_evaluate(ctx, pv, flux, status)
    counts = rr.rr_get_counters(ctx)
    rr.rr_enable_counters(ctx, False)
    n_bad = int((status != 0).sum().item())

    # ---- end to end: host buffers in, host flux out, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        try:
            flux_h_t = torch.empty((wl.npv, wl.npt), dtype=model.flux_dtype, pin_memory=True)
            ldp_h_t = torch.as_tensor(ldp_h).pin_memory()
            pv_h_t = torch.as_tensor(wl.pv).pin_memory()
            pinned = True
        except RuntimeError:
            flux_h_t = torch.empty((wl.npv, wl.npt), dtype=model.flux_dtype)
            ldp_h_t, pv_h_t = torch.as_tensor(ldp_h), torch.as_tensor(wl.pv)
            pinned = False
        status_h = np.empty(wl.npv, np.int32)
        fh, lh, ph = flux_h_t.numpy(), ldp_h_t.numpy(), pv_h_t.numpy()
        rr.rr_evaluate_host(ctx, lh, ph, fh, status_h)          # warm-up (allocates staging)
        e2e_steps = max(1, min(steps, 3))
        shard.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            rr.rr_evaluate_host(ctx, lh, ph, fh, status_h)      # synchronous
        dt = time.perf_counter() - t0
        dt = shard.max_over_ranks(dt, dev)
        e2e = {"value": evals_all * e2e_steps / dt, "unit": UNIT,
               "h2d_bytes_per_step": int(lh.nbytes + ph.nbytes),
               "d2h_bytes_per_step": int(fh.nbytes + status_h.nbytes),
               "steps": e2e_steps, "ms_per_step": 1e3 * dt / e2e_steps,
               "host_memory": "pinned" if pinned else "pageable",
               "call": "rr_evaluate_host (H2D ldp+pv, kernels 1-3, D2H flux+status, chunked on 2 streams)",
               "timer": "host perf_counter around the synchronous call (its copies and kernels "
                        "run on the library's own streams), max over ranks",
               "flux_checksum": float(fh[::max(1, wl.npv // 64), ::997].astype(np.float64).sum())}
        del flux_h_t, fh

    if rank != 0:
        return 0

    # ---- roofline of the dominant kernel (rr_flux_kernel), DESIGN.md s7 ----
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except (OSError, ValueError):
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    hbm_src = "MEASURED_PEAKS.json hbm_gbs (of measured)" if "hbm_gbs" in peaks else \
        "6650 GB/s (of fallback)"
    es = 4 if precision == rr.RR_FP32 else 8            # flux element
    nrows = wl.npv * wl.model.npb
    # algorithmic bytes per launch: flux written once, times read once, two table rows + Istar +
    # the per-pv constants read once per (pv, passband)
    alg_bytes = (wl.npv * wl.npt * es + wl.npt * 12 + nrows * (2 * wl.model.ng + 1) * es
                 + wl.npv * 184)
    t_flux = ms_flux * 1e-3
    ops = dict(ALG_OPS["fp64" if args.precision == "fp64" else "fp32"])
    if args.precision == "fp64":
        # circular orbits: per exposure phase 4 + sin/cos polynomials 15, per sub-sample one plane
        # rotation 4 + z^2 2
        ops["circular"] = 6.0 + 19.0 * wl.npt / wl.evaluations_per_pv
    alg_fma = (counts["skipped"] * ops["skipped"] + counts["circular"] * ops["circular"]
               + counts["eccentric"] * ops["eccentric_fixed"]
               + counts["solver_iters"] * ops["solver_iter"]
               + counts["occulting"] * ops["occulting"] + counts["ingress"] * ops["ingress"])
    lanes = FP32_LANES_PER_SM if precision != rr.RR_FP64 else FP64_LANES_PER_SM
    sm_max = (clocks or {}).get("sm_max_mhz") or float(peaks.get("sm_max_mhz", 1965.0))
    alu_peak_tflops = 2.0 * lanes * SM_COUNT * sm_max * 1e6 / 1e12
    fma_live = rr.rr_measure_fma_peak(precision)
    hbm_achieved = alg_bytes / t_flux / 1e9
    alu_achieved = 2.0 * alg_fma / t_flux / 1e12
    t_hbm, t_alu = alg_bytes / (hbm_peak * 1e9), 2.0 * alg_fma / (alu_peak_tflops * 1e12)
    if t_hbm >= t_alu:
        roofline = {"bound": "hbm", "achieved": hbm_achieved, "peak": hbm_peak, "unit": "GB/s",
                    "frac": hbm_achieved / hbm_peak, "traffic": None, "peak_source": hbm_src}
    else:
        roofline = {"bound": "alu", "achieved": alu_achieved, "peak": alu_peak_tflops,
                    "unit": "TFLOP/s", "frac": alu_achieved / alu_peak_tflops, "traffic": None,
                    "peak_source": f"{lanes} FMA lanes/clk/SM x {SM_COUNT} SMs x {sm_max:.0f} MHz "
                                   "x 2 (DESIGN.md s7)"}
    roofline["traffic"] = ncu_traffic(wl.name, args.precision)
    roofline.update({
        "kernel": "rr_flux_kernel", "kernel_ms": ms_flux, "ld_table_kernel_ms": ms_table + ms_rows,
        "ld_table_parts_ms": {"rr_build_ld_table": ms_table, "rows_in_rr_evaluate": ms_rows},
        "rr_evaluate_ms": ms_eval, "table_mode": args.table_mode,
        "algorithmic_bytes": int(alg_bytes), "algorithmic_fma": int(alg_fma),
        "algorithmic_ops_per_unit": ops,
        "hbm_frac": hbm_achieved / hbm_peak, "alu_frac": alu_achieved / alu_peak_tflops,
        "fma_peak_measured_live_tflops": 2.0 * fma_live / 1e12,
        "class_counts": counts,
        "note": "kernel_ms = CUDA events recorded by the library around rr_flux_kernel on the "
                "launching stream, inside the timed region, mean over the timed steps; frac = "
                "achieved / peak; traffic: see profiles/",
    })

    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        rate, dt, n = oracle_rate(wl, 24.0)
        cpu_baseline = {"value": rate, "unit": UNIT, "cores": os.cpu_count() or 1,
                        "kind": "oracle", "seconds": dt,
                        "sample": f"first {n} of {wl.npv} parameter vectors x all {wl.npt} "
                                  f"exposures (table build + evaluate), OpenMP over pv"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps,
        "warmup": warm, "ms_per_step": ms_total / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": {"fp64": "f64", "fp32": "f32", "mixed": "f32 (sum and flux f64)"}[args.precision],
        "data": "synthetic",
        "config": workload_config(wl, args.precision, {
            "parallelism": f"pv-sharded x{world}, no collective",
            "l2": "working set per step (flux + LD table) is far larger than the 126 MB L2; "
                  "no flush needed" if wl.npv * wl.npt * es > 2 ** 28 else
                  "working set fits L2: small config, latency-bound, no roofline claim",
            "invalid_pv": n_bad}),
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
        "cpu_baseline": cpu_baseline,
        "paper_context": "paper reports no absolute throughput; OpenCL fp32 GPU 10-20x over its "
                         "CPU code on unnamed hardware (PAPER.md:194)",
    }
    print(json.dumps(line))
    model.close()
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
