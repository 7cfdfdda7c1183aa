#!/usr/bin/env python
"""bench.py - transit-model evaluations/s of the CUDA library on the BASELINE.json workloads.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 0..4|4b] [--precision fp64|fp32|mixed]
                    [--scaling weak|strong] [--ld-law quadratic] [--no-all-configs]
    python bench.py --impl reference ...          # the CPU oracle, as it stands, on the host cores

A "step" is one pass of the whole hot path over one batch of synthetic input:
rr_build_ld_table (kernel 1) + rr_evaluate (per-pv prep, kernels 2+3 fused; kernel 4's tile table
was built once by rr_set_data, the paper's call pattern PAPER.md:207-218).  Default workload:
config 4 of BASELINE.json (the largest population workload, the one the north-star target is
stated on), fp64.  One JSON line on stdout (rank 0).  See DESIGN.md s8 for every field.

After the headline timing the default single-GPU run also times every other BASELINE config and
precision for a few steps each (``all_configs``: evaluations/s, kernel times, roofline fraction and the
largest |flux - oracle| on a sample), SURVEY.md 8(d)'s per-config report.

Multi-GPU (torchrun, one process per GPU): the path shards over parameter vectors with no exchange.
``--scaling weak`` (default): each rank evaluates its own full population; ``--scaling strong``: ONE
population is split with ``shard.pv_slice``.  The only communication is the barrier and the
max-over-ranks of the device time.
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
# ALGORITHMIC FMA-pipe instructions per unit of each class of the flux kernel: the
# count of the direct formulation (Kepler solve by Halley steps on d = E - E_tr, analytic lens area with
# its two arctangents, the paper's cc_intersection_area), counted in the SASS of the build that
# evaluates exactly that (profiles/r02c; DFMA/DMUL/DADD in fp64 mode, FFMA/FMUL/FADD in fp32 and mixed
# mode, where the fp64 phase arithmetic runs on the other pipe and is not counted).  Compares, selects,
# conversions, loads and the MUFU seeds are not counted; sub-samples in merged out-of-window fill runs
# cost no arithmetic.  `roofline.frac` = this work / time / peak: the EFFECTIVE fraction.  Where the
# kernel reaches the same result with fewer instructions (fp64: the lens area between the contacts from
# per-pv polynomials, EXECUTED_OPS below) the line says so: `counter_based.frac` is what the pipe
# really executes, `algorithmic_over_executed` the ratio.
CIRC_PER_SUBSAMPLE, CIRC_PER_EXPOSURE = 6.0, 22.0   # fp64 circular path: rotation + z^2; phase + sincos
ALG_OPS = {
    "fp64": dict(skipped=1, circular=28, eccentric_fixed=23, solver_iter=30, occulting=11,
                 ingress=60),
    "fp32": dict(skipped=0, circular=7, eccentric_fixed=20, solver_iter=24, occulting=11,
                 ingress=45),
}
# what the committed kernels execute per unit where that differs from the direct formulation
EXECUTED_OPS = {"fp64": dict(ingress=24), "fp32": dict(ingress=24)}
ZPOLY_OPS = 15      # an eccentric sub-sample through the z^2 polynomials: t, w, Horner 12, |.| + tiny


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="4", choices=["0", "1", "2", "3", "4", "4b"],
                    help="BASELINE.json config; 4b = config 4 with literal 2-minute spacing (SURVEY 8(d))")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32", "mixed"],
                    help="mixed = fp32 z and Ip*Ap, fp64 averaging / subtraction / flux (PAPER.md:293)")
    ap.add_argument("--npv", type=int, default=None, help="shrink the population (debugging)")
    ap.add_argument("--npt", type=int, default=None, help="shrink the time axis (debugging)")
    ap.add_argument("--table-mode", default="lazy", choices=["lazy", "full", "direct"],
                    help="kernel 1: rows for each pv's k at evaluate time (default), the full table, "
                         "or the paper's direct model (weights at each pv's own k, no k grid)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: a full population per rank (weak) or one population split by "
                         "shard.pv_slice (strong)")
    ap.add_argument("--ld-law", default=None, choices=["quadratic"],
                    help="time the step with rr_build_ld_table_law (the law evaluated on the device "
                         "from its coefficients, PAPER.md:143-156) instead of rr_build_ld_table")
    ap.add_argument("--no-orbit-poly", action="store_true",
                    help="solve Kepler's equation per eccentric sub-sample (rr_set_orbit_poly(ctx, 0)) "
                         "instead of evaluating the per-pv z^2 polynomials")
    ap.add_argument("--direct-formulation", action="store_true",
                    help="the direct formulation throughout: a Kepler solve per eccentric sub-sample and "
                         "the two-arctangent lens area per ingress sub-sample (rr_set_orbit_poly(ctx, 0), "
                         "rr_set_lens_poly(ctx, 0)): executed work = algorithmic work")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-all-configs", action="store_true",
                    help="skip the per-config / per-precision report after the headline timing")
    args = ap.parse_args()
    args.config = args.config if args.config == "4b" else int(args.config)
    return args


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


def ncu_capture(workload: str, precision: str):
    """The committed `ncu --set full` capture of rr_flux_kernel for this workload and precision
    (profiles/flux_kernel_ncu.csv, one row per capture): dram bytes and executed arithmetic
    thread-instructions per launch, or None."""
    try:
        with open(os.path.join(ROOT, "profiles", "flux_kernel_ncu.csv")) as f:
            rows = [ln.split(",") for ln in f.read().splitlines() if ln and not ln.startswith("#")]
        cols = rows[0]
        for r in rows[1:]:
            d = dict(zip(cols, r))
            if d["workload"] == workload and d["precision"] == precision:
                return d
    except (OSError, ValueError, KeyError, IndexError):
        pass
    return None


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


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
def oracle_sample(wl, stride: int):
    """Every stride-th parameter vector of the workload, all exposures."""
    return wl.subset_pv(np.arange(0, wl.npv, max(1, stride)))


def oracle_run(sub, nthreads: int):
    """Oracle as it stands (table build + evaluate) on a sub-population: evaluations/s, seconds.
    nthreads = 0: all cores (passed explicitly: the OpenMP thread count is sticky)."""
    import oracle
    nthreads = nthreads or (os.cpu_count() or 1)
    om = oracle.OracleModel.from_config(sub.model)
    t = time.perf_counter()
    om.build_ld_table(sub.ldp(om.mu))
    om.evaluate(sub.times, sub.lc_index, sub.passband_index, sub.supersampling,
                sub.exposure_time, sub.pv, nthreads=nthreads)
    dt = time.perf_counter() - t
    return sub.evaluations / dt, dt


def oracle_stride_for(wl, nthreads: int, target_s: float) -> int:
    """Stride of the pv sample so that one oracle pass takes about target_s (calibrated on a
    handful of parameter vectors; strides are powers of two, 1 = the whole population)."""
    cores = os.cpu_count() or 1
    n0 = min(wl.npv, max(1, cores if nthreads == 0 else 1))
    rate, _ = oracle_run(wl.subset_pv(np.arange(0, wl.npv, max(1, wl.npv // n0))[:n0]), nthreads)
    want = max(1.0, rate * target_s / max(1, wl.evaluations_per_pv))     # pvs in target_s
    stride = 1
    while wl.npv / stride > want and stride < wl.npv:
        stride *= 2
    return stride


def cpu_baseline_of(wl, target_s: float = 10.0) -> dict:
    """the oracle on the GPU box's host cores, 1 thread and all cores, on every
    stride-th parameter vector (all exposures), extrapolation-free: evaluations of the sample / time."""
    cores = os.cpu_count() or 1
    s_all = oracle_stride_for(wl, 0, target_s)
    s_one = oracle_stride_for(wl, 1, target_s)
    sub_all, sub_one = oracle_sample(wl, s_all), oracle_sample(wl, s_one)
    r_all, t_all = oracle_run(sub_all, 0)
    r_one, t_one = oracle_run(sub_one, 1)
    return {"value": r_all, "unit": UNIT, "cores": cores, "kind": "oracle",
            "all_cores": r_all, "one_thread": r_one, "cpu_model": cpu_model(),
            "seconds": {"all_cores": t_all, "one_thread": t_one},
            "sample": f"every {s_all}th parameter vector ({sub_all.npv} of {wl.npv}) x all {wl.npt} "
                      f"exposures on {cores} threads (OpenMP over pv); one_thread: every {s_one}th "
                      f"({sub_one.npv}); table build + evaluate"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl = workloads.make_workload(args.config, npv=args.npv, npt=args.npt)
    cores = os.cpu_count() or 1
    steps, warm = max(1, args.steps), max(0, args.warmup)
    target = min(10.0, 150.0 / (steps + warm))
    stride = oracle_stride_for(wl, 0, target)
    sub = oracle_sample(wl, stride)
    for _ in range(warm):
        oracle_run(sub, 0)
    t_total = 0.0
    for _ in range(steps):
        _, dt = oracle_run(sub, 0)
        t_total += dt
    value = sub.evaluations * steps / t_total
    sample = (f"every {stride}th parameter vector ({sub.npv} of {wl.npv}) x all {wl.npt} exposures; "
              f"each of the {steps} steps re-runs this same sample (table build + evaluate, "
              f"~{t_total / steps:.1f} s of oracle on {cores} threads)")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warm, "ms_per_step": 1e3 * t_total / steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(wl, "fp64"),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": sample, "cpu_model": cpu_model()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ---- our arm ----------------------------------------------------------------------------------------
PRECISIONS = {"fp64": 0, "fp32": 1, "mixed": 2}
DTYPE_NAME = {"fp64": "f64", "fp32": "f32", "mixed": "f32 (sum and flux f64)"}


class Case:
    """One workload in one precision, resident on the device: ctx, inputs, output buffers."""

    def __init__(self, rr, wl, precision: str, table_mode: str, dev, ld_law=None, orbit_poly=True,
                 lens_poly=True):
        import torch
        self.rr, self.wl, self.precision, self.dev = rr, wl, precision, dev
        self.orbit_poly, self.lens_poly = orbit_poly, lens_poly
        code = PRECISIONS[precision]
        self.npdt = np.float32 if code != rr.RR_FP64 else np.float64
        self.model = rr.RoadRunner.from_config(wl.model, code)
        self.ctx = self.model.ctx
        rr.rr_set_table_mode(self.ctx, {"lazy": rr.RR_TABLE_LAZY, "full": rr.RR_TABLE_FULL,
                                        "direct": rr.RR_TABLE_DIRECT}[table_mode])
        rr.rr_set_orbit_poly(self.ctx, orbit_poly)
        rr.rr_set_lens_poly(self.ctx, lens_poly)
        self.model.set_data(wl.times, wl.lc_index, wl.passband_index, wl.supersampling,
                            wl.exposure_time)
        self.ldp_h = np.ascontiguousarray(wl.ldp(self.model.mu), dtype=self.npdt)
        self.ldp = torch.as_tensor(self.ldp_h).to(dev)
        self.pv = torch.as_tensor(wl.pv).to(dev)
        self.flux = torch.empty((wl.npv, wl.npt), dtype=self.model.flux_dtype, device=dev)
        self.status = torch.empty(wl.npv, dtype=torch.int32, device=dev)
        self.ld_law = ld_law
        self.ldc = None
        if ld_law is not None:
            if wl.ld_kind != ld_law:
                raise SystemExit(f"--ld-law {ld_law}: workload {wl.name} uses the {wl.ld_kind} law")
            self.ldc = torch.as_tensor(np.ascontiguousarray(wl.ld_coeffs, np.float64)).to(dev)

    def build_table(self):
        if self.ldc is not None:
            self.rr.rr_build_ld_table_law(self.ctx, self.ld_law, self.ldc, self.wl.npv)
        else:
            self.rr.rr_build_ld_table(self.ctx, self.ldp, self.wl.npv)

    def step(self):
        self.build_table()
        self.rr.rr_evaluate(self.ctx, self.pv, self.flux, self.status)

    def timed(self, steps: int, warm: int, sync, sampler_rank0=None):
        """W warm-up steps, then K steps between synchronisations: CUDA events around the steps and
        the library's own events around its kernels.  Returns per-step times in ms."""
        import torch
        rr = self.rr
        for _ in range(warm):
            self.step()
        torch.cuda.synchronize()
        ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
        launches0 = rr.rr_launch_count(self.ctx)
        sampler = sampler_rank0() if sampler_rank0 else None
        sync()
        rr.rr_enable_kernel_timing(self.ctx, True)   # the library's own CUDA events around its kernels
        for s in range(steps):
            ev[s][0].record()
            self.build_table()
            ev[s][1].record()
            rr.rr_evaluate(self.ctx, self.pv, self.flux, self.status)
            ev[s][2].record()
        sync()
        clocks = sampler.stop() if sampler else None
        launches = rr.rr_launch_count(self.ctx) - launches0
        kt = rr.rr_get_kernel_times(self.ctx)
        rr.rr_enable_kernel_timing(self.ctx, False)
        return {
            "ms_total": ev[0][0].elapsed_time(ev[-1][2]),
            "ms_table": float(np.mean([e[0].elapsed_time(e[1]) for e in ev])),
            "ms_eval": float(np.mean([e[1].elapsed_time(e[2]) for e in ev])),
            "ms_flux": kt["flux_ms"] / max(1, kt["calls"]),       # rr_flux_kernel alone
            "ms_rows": kt["rows_ms"] / max(1, kt["calls"]),
            "launches": int(launches), "clocks": clocks,
        }

    def graph_us_per_step(self, n=300):
        """One step captured into a CUDA graph and replayed (the step allocates and synchronises
        nothing in steady state): microseconds per replay."""
        import torch
        side, graph = torch.cuda.Stream(), torch.cuda.CUDAGraph()
        with torch.cuda.stream(side):
            self.step()
            torch.cuda.synchronize()
            with torch.cuda.graph(graph, stream=side):
                self.step()
        for _ in range(10):
            graph.replay()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            graph.replay()
        e1.record()
        torch.cuda.synchronize()
        return 1e3 * e0.elapsed_time(e1) / n

    def class_counts(self):
        """Class counts of one evaluation (untimed launches with the kernel's counters on): those of
        the direct formulation (every eccentric sub-sample solves Kepler's equation: the algorithmic
        work) plus `eccentric_poly`, the sub-samples the committed kernel takes from the per-pv z^2
        polynomials instead."""
        rr = self.rr
        rr.rr_enable_counters(self.ctx, True)
        rr.rr_set_orbit_poly(self.ctx, False)
        rr.rr_evaluate(self.ctx, self.pv, self.flux, self.status)
        counts = rr.rr_get_counters(self.ctx)
        rr.rr_set_orbit_poly(self.ctx, self.orbit_poly)
        rr.rr_evaluate(self.ctx, self.pv, self.flux, self.status)
        as_run = rr.rr_get_counters(self.ctx)
        rr.rr_enable_counters(self.ctx, False)
        counts["eccentric_poly"] = as_run["eccentric_poly"]
        counts["solver_iters_as_run"] = as_run["solver_iters"]
        counts["lens_poly"] = int(bool(self.lens_poly))
        return counts

    def sample_error(self, n_pv=8, n_cols=600):
        """Largest |flux - oracle| over sampled (pv, exposure) pairs of the flux now in self.flux:
        n_pv parameter vectors x (n_cols random exposures + the 40 nearest to each one's t0).
        With --ld-law the oracle takes the law's closed-form Istar as the library does (the
        paper's "integrated analytically") instead of reading R6."""
        import oracle
        import torch
        wl = self.wl
        rng = np.random.default_rng(7)
        pvs = np.sort(rng.choice(wl.npv, min(n_pv, wl.npv), replace=False))
        cols = rng.choice(wl.npt, min(n_cols, wl.npt), replace=False)
        t0 = wl.pv[pvs, wl.model.nkpb]
        near = [np.argsort(np.abs(wl.times - t))[:40] for t in t0]
        cols = np.unique(np.concatenate([cols] + near))
        got = self.flux[torch.as_tensor(pvs, device=self.dev)][:, torch.as_tensor(cols, device=self.dev)]
        got = got.cpu().numpy().astype(np.float64)
        sub = wl.subset_pv(pvs).subset_times(cols)
        if self.ld_law is None:
            want, _ = oracle.evaluate_workload(sub, nthreads=0)
        else:
            from oracle import truth
            om = oracle.OracleModel.from_config(sub.model)
            ist = np.array([[truth.law(self.ld_law, c)[1] for c in row] for row in sub.ld_coeffs])
            om.build_ld_table(sub.ldp(om.mu), istar_override=ist)
            want, _ = om.evaluate(sub.times, sub.lc_index, sub.passband_index, sub.supersampling,
                                  sub.exposure_time, sub.pv, nthreads=0)
        ok = ~np.isnan(want)
        return float(np.max(np.abs(got[ok] - want[ok]))), int(ok.sum()), int((want[ok] < 1).sum())

    def close(self):
        self.model.close()
        self.ldp = self.pv = self.flux = self.status = self.ldc = None


def roofline_of(rr, wl, precision: str, t: dict, counts: dict, table_mode: str, clocks, peaks,
                capture_key=None):
    """algorithmic bytes and FMA-pipe instructions per launch of rr_flux_kernel against
    the HBM and ALU peaks; the larger time bound names the binding roofline."""
    code = PRECISIONS[precision]
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    hbm_src = "MEASURED_PEAKS.json hbm_gbs (of measured)" if "hbm_gbs" in peaks else \
        "6650 GB/s (of fallback)"
    es = 4 if code == rr.RR_FP32 else 8            # flux element
    nrows = wl.npv * wl.model.npb
    # algorithmic bytes per launch: flux written once, times read once, two table rows + Istar +
    # the per-pv constants read once per (pv, passband)
    alg_bytes = (wl.npv * wl.npt * es + wl.npt * 12 + nrows * (2 * wl.model.ng + 1) * es
                 + wl.npv * 184)
    t_flux = max(t["ms_flux"], 1e-6) * 1e-3
    ops = dict(ALG_OPS["fp64" if precision == "fp64" else "fp32"])
    if precision == "fp64":
        # circular orbits: per exposure phase + sin/cos polynomials, per sub-sample one plane
        # rotation + z^2
        ops["circular"] = CIRC_PER_SUBSAMPLE + CIRC_PER_EXPOSURE * wl.npt / wl.evaluations_per_pv
    alg_fma = (counts["skipped"] * ops["skipped"] + counts["circular"] * ops["circular"]
               + counts["eccentric"] * ops["eccentric_fixed"]
               + counts["solver_iters"] * ops["solver_iter"]
               + counts["occulting"] * ops["occulting"] + counts["ingress"] * ops["ingress"])
    lanes = FP32_LANES_PER_SM if code != rr.RR_FP64 else FP64_LANES_PER_SM
    sm_max = (clocks or {}).get("sm_max_mhz") or float(peaks.get("sm_max_mhz", 1965.0))
    alu_peak_tflops = 2.0 * lanes * SM_COUNT * sm_max * 1e6 / 1e12
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
    cap = ncu_capture(wl.name, capture_key or precision)
    counter_based = None
    if cap is not None:
        roofline["traffic"] = int(cap["dram_read_bytes"]) + int(cap["dram_write_bytes"])
        executed = int(cap["arith_thread_inst"])
        # executed arithmetic thread-instructions of the committed capture (DFMA + DADD + DMUL, or
        # FFMA + FADD + FMUL: a property of the build and the workload, not of the run) over the
        # lanes x cycles of THIS run's kernel time: the counter-based pipe-feeding fraction
        counter_based = {"arith_thread_inst_per_launch": executed,
                         "frac": executed / (lanes * SM_COUNT * sm_max * 1e6 * t_flux),
                         "algorithmic_over_executed": alg_fma / max(1, executed),
                         "pipe_cycles_active_pct_ncu": float(cap["pipe_active_pct"]),
                         "issue_active_pct_ncu": float(cap["issue_active_pct"]),
                         "capture": cap["capture"]}
    exe_ops = dict(ops)
    if counts.get("lens_poly", 1):
        exe_ops.update(EXECUTED_OPS.get("fp64" if precision == "fp64" else "fp32", {}))
    exe_fma = alg_fma + sum(counts[c] * (exe_ops[c] - ops[c]) for c in ("ingress",))
    if counts.get("eccentric_poly"):
        # sub-samples taken from the z^2 polynomials: ZPOLY_OPS instead of the fixed part and their solves
        exe_fma += (counts["eccentric_poly"] * (ZPOLY_OPS - ops["eccentric_fixed"])
                    - (counts["solver_iters"] - counts["solver_iters_as_run"]) * ops["solver_iter"])
    roofline.update({
        "executed_ops_per_unit": exe_ops, "executed_fma_by_table": int(exe_fma),
        "executed_frac_by_table": 2.0 * exe_fma / t_flux / 1e12 / alu_peak_tflops,
        "kernel": "rr_flux_kernel", "kernel_ms": t["ms_flux"],
        "ld_table_kernel_ms": t["ms_table"] + t["ms_rows"],
        "ld_table_parts_ms": {"rr_build_ld_table": t["ms_table"], "rows_in_rr_evaluate": t["ms_rows"]},
        "rr_evaluate_ms": t["ms_eval"], "table_mode": table_mode,
        "algorithmic_bytes": int(alg_bytes), "algorithmic_fma": int(alg_fma),
        "algorithmic_ops_per_unit": ops,
        "hbm_frac": hbm_achieved / hbm_peak, "alu_frac": alu_achieved / alu_peak_tflops,
        "counter_based": counter_based,
        "class_counts": counts,
    })
    return roofline


def all_configs_report(rr, dev, peaks, args, headline):
    """every BASELINE config and precision, a few steps each (after the headline
    timing, rank 0 of a single-GPU run).  Config 0 is launch-latency-bound: microseconds per call, no
    roofline claim."""
    import torch
    out = []
    plan = [(0, "fp64"), (0, "fp32"), (1, "fp64"), (1, "fp32"), (2, "fp64"), (2, "fp32"),
            (3, "fp64"), (3, "fp32"), (4, "fp64"), (4, "fp32"), (4, "mixed"), ("4b", "fp64"),
            ("4b", "fp32")]
    cache = {}
    for config, precision in plan:
        if (config, precision) == headline:
            continue
        if config not in cache:
            cache.clear()
            cache[config] = workloads.make_workload(config)
        wl = cache[config]
        case = Case(rr, wl, precision, "lazy", dev)
        small = wl.evaluations < 10 ** 6
        steps = 200 if small else (10 if wl.evaluations < 2 * 10 ** 9 else 5)
        t = case.timed(steps, 3, torch.cuda.synchronize)
        counts = case.class_counts()
        err, n_s, n_in = case.sample_error()
        value = wl.evaluations * steps / (t["ms_total"] * 1e-3)
        entry = {"workload": wl.name, "precision": precision, "value": value, "unit": UNIT,
                 "steps": steps, "ms_per_step": t["ms_total"] / steps, "flux_ms": t["ms_flux"],
                 "table_ms": t["ms_table"] + t["ms_rows"],
                 "max_abs_err_vs_oracle_sample": err, "sampled_points": n_s,
                 "sampled_in_transit": n_in}
        if small:
            entry.update({"us_per_call": 1e3 * t["ms_total"] / steps, "bound": "launch latency",
                          "frac": None, "us_per_call_cuda_graph": case.graph_us_per_step()})
        else:
            r = roofline_of(rr, wl, precision, t, counts, "lazy", headline_clocks(args), peaks)
            entry.update({"bound": r["bound"], "frac": r["frac"], "hbm_frac": r["hbm_frac"],
                          "alu_frac": r["alu_frac"], "traffic": r["traffic"],
                          "counter_frac": (r["counter_based"] or {}).get("frac")})
        out.append(entry)
        case.close()
        del case
        torch.cuda.empty_cache()
    return out


def headline_clocks(args):
    return getattr(args, "_clocks", None)


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

    wl = workloads.make_workload(args.config, npv=args.npv, npt=args.npt)
    npv_job = wl.npv
    if world > 1 and args.scaling == "strong":
        b, e = shard.pv_slice(wl.npv, rank, world)      # ONE population, split over the ranks
        wl = wl.subset_pv(np.arange(b, e))
    elif rank:   # weak scaling: every rank gets a full population, rotated so that data differ
        sh = (rank * 97) % wl.npv
        wl.pv = np.ascontiguousarray(np.roll(wl.pv, sh, axis=0))
        wl.ld_coeffs = np.ascontiguousarray(np.roll(wl.ld_coeffs, sh, axis=0))

    case = Case(rr, wl, args.precision, args.table_mode, dev, ld_law=args.ld_law,
                orbit_poly=not (args.no_orbit_poly or args.direct_formulation),
                lens_poly=not args.direct_formulation)
    ctx, model = case.ctx, case.model
    steps, warm = max(1, args.steps), max(3, args.warmup)

    def sync():
        shard.barrier()
        torch.cuda.synchronize()
        shard.barrier()

    t = case.timed(steps, warm, sync, (lambda: ClockSampler(local_rank)) if rank == 0 else None)
    clocks = t["clocks"]
    args._clocks = clocks
    ms_total = shard.max_over_ranks(t["ms_total"], dev)
    evals_all = shard.sum_over_ranks(float(wl.evaluations), dev)
    value = evals_all * steps / (ms_total * 1e-3)
    counts = case.class_counts()
    n_bad = int((case.status != 0).sum().item())
    err_sample = case.sample_error() if rank == 0 else None
    precision = PRECISIONS[args.precision]

    # ---- end to end: host buffers in, host flux out, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        try:
            flux_h_t = torch.empty((wl.npv, wl.npt), dtype=model.flux_dtype, pin_memory=True)
            ldp_h_t = torch.as_tensor(case.ldp_h).pin_memory()
            pv_h_t = torch.as_tensor(wl.pv).pin_memory()
            pinned = True
        except RuntimeError:
            flux_h_t = torch.empty((wl.npv, wl.npt), dtype=model.flux_dtype)
            ldp_h_t, pv_h_t = torch.as_tensor(case.ldp_h), torch.as_tensor(wl.pv)
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
               "bound": "PCIe: the flux matrix leaves the device once per step "
                        f"({fh.nbytes / 1e9:.2f} GB D2H)",
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
    roofline = roofline_of(rr, wl, args.precision, t, counts, args.table_mode, clocks, peaks,
                           capture_key=args.precision + "-direct" if args.direct_formulation else None)
    roofline["fma_peak_measured_live_tflops"] = 2.0 * rr.rr_measure_fma_peak(precision) / 1e12
    roofline["note"] = ("kernel_ms = CUDA events recorded by the library around rr_flux_kernel on the "
                        "launching stream, inside the timed region, mean over the timed steps; frac = "
                        "achieved / peak from the op table of DESIGN.md s7; counter_based.frac = the "
                        "arithmetic thread-instructions ncu counted for this build and workload "
                        "(profiles/flux_kernel_ncu.csv) over lanes x cycles of this run's kernel time")

    es = 4 if precision == rr.RR_FP32 else 8
    line_config = workload_config(wl, args.precision, {
        "parallelism": f"pv-sharded x{world}, no collective"
                       + (f" (strong: {npv_job} parameter vectors split)" if world > 1 and
                          args.scaling == "strong" else ""),
        "l2": "working set per step (flux + LD table) is far larger than the 126 MB L2; "
              "no flush needed" if wl.npv * wl.npt * es > 2 ** 28 else
              "working set fits L2: small config, latency-bound, no roofline claim",
        "invalid_pv": n_bad,
        "ld_table_call": "rr_build_ld_table_law" if args.ld_law else "rr_build_ld_table",
        "lens_area": "two arctangents per ingress sub-sample" if args.direct_formulation else
                     "per-(pv, k) polynomials between the contacts for k <= 0.32, else the exact form",
        "orbit": "Kepler solve per eccentric sub-sample" if (args.no_orbit_poly or args.direct_formulation) else
                 "per-pv z^2 polynomials over the transit window where they converge, else the solve"})
    case.close()
    del case
    torch.cuda.empty_cache()

    all_configs = None
    if world == 1 and not args.no_all_configs and args.npv is None and args.npt is None:
        all_configs = all_configs_report(rr, dev, peaks, args, (args.config, args.precision))

    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        cpu_baseline = cpu_baseline_of(wl)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps,
        "warmup": warm, "ms_per_step": ms_total / steps, "higher_is_better": True,
        "scaling": args.scaling if world > 1 else "weak", "vs_baseline": None,
        "dtype": DTYPE_NAME[args.precision], "data": "synthetic",
        "config": line_config,
        "clocks": clocks, "e2e": e2e, "gpu_launches": t["launches"], "roofline": roofline,
        "max_abs_err_vs_oracle_sample": {"value": err_sample[0], "points": err_sample[1],
                                         "in_transit": err_sample[2]},
        "cpu_baseline": cpu_baseline,
        "all_configs": all_configs,
        "paper_context": "paper reports no absolute throughput; OpenCL fp32 GPU 10-20x over its "
                         "CPU code on unnamed hardware (PAPER.md:194)",
    }
    print(json.dumps(line))
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    try:
        return run_ours(args)
    finally:
        try:                                    # leave the process group cleanly under torchrun
            import torch.distributed as dist
            if dist.is_available() and dist.is_initialized():
                dist.destroy_process_group()
        except Exception:
            pass


if __name__ == "__main__":
    sys.exit(main())
