"""paper_2009_08500_b200 - thin Python binding of libroadrunner_b200.so (include/roadrunner.h).

Argument marshalling only: every step of the path (z grid and geometry weights, LD table, orbit,
fused flux, heterogeneous dispatch) runs in the library's sm_100a CUDA kernels.  PyTorch supplies
device memory and the current CUDA stream, nothing else.  There is no CPU fallback: loading fails
loudly if the library cannot be built or found, and every compute call raises ``RoadRunnerError``
when CUDA reports an error (e.g. no device).

Module-level ``rr_*`` functions mirror the C entry points one to one (torch tensors in place of
raw pointers); ``RoadRunner`` is a small convenience wrapper in the shape of the paper's
``RoadRunnerModel``: ``set_data`` once, ``build_ld_table`` + ``evaluate`` many
times.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

RR_FP64, RR_FP32, RR_MIXED = 0, 1, 2
RR_REDUCE_AUTO, RR_REDUCE_THREAD, RR_REDUCE_SHUFFLE = 0, 1, 2
RR_TABLE_LAZY, RR_TABLE_FULL, RR_TABLE_DIRECT = 0, 1, 2
LD_LAWS = {"uniform": 0, "linear": 1, "quadratic": 2, "quadratic-tri": 3, "general": 4,
           "nonlinear": 5, "logarithmic": 6, "exponential": 7, "power-2": 8, "power-2-pm": 9}
RR_PV_K_RANGE, RR_PV_E_RANGE, RR_PV_A_RANGE, RR_PV_P_RANGE, RR_PV_NONFINITE = 1, 2, 4, 8, 16

# every symbol include/roadrunner.h declares (tests check the library exports each of them)
SYMBOLS = (
    "rr_create", "rr_destroy", "rr_error_string", "rr_get_mu", "rr_get_ze", "rr_get_weights",
    "rr_set_data", "rr_build_ld_table", "rr_table_ptr", "rr_istar_ptr", "rr_get_table",
    "rr_evaluate",
    "rr_evaluate_flat", "rr_orbit_z", "rr_num_subsamples", "rr_num_tiles", "rr_get_tiles",
    "rr_set_reduction", "rr_evaluate_host", "rr_enable_counters", "rr_get_counters",
    "rr_launch_count", "rr_measure_fma_peak", "rr_set_table_mode", "rr_enable_kernel_timing",
    "rr_get_kernel_times", "rr_get_rows", "rr_set_mean_k_weights",
    "rr_set_small_planet", "rr_build_ld_table_law", "rr_math_probe", "rr_set_orbit_poly",
    "rr_orbit_z_noalloc", "rr_set_lens_poly",
)
PROBE_OPS = {"sqrt3": 0, "sqrt": 1, "div3": 2, "rcp": 3, "atan_t": 4, "atan_quadrant": 5,
             "atan2_pos": 6, "sincosm1": 7, "cell": 8}


class RoadRunnerError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {error_string(code)} (code {code})")


class rr_config(C.Structure):
    _fields_ = [("nzin", C.c_int32), ("nzlimb", C.c_int32), ("zcut", C.c_double),
                ("ng", C.c_int32), ("nk", C.c_int32), ("k0", C.c_double), ("k1", C.c_double),
                ("npb", C.c_int32), ("nkpb", C.c_int32), ("precision", C.c_int32)]


_lib = None
_VP, _I64, _I32, _DBL = C.c_void_p, C.c_int64, C.c_int32, C.c_double


def library_path() -> str:
    return _build.LIB


def load() -> C.CDLL:
    """Build (if stale) and load the CUDA library.  Raises if that is impossible."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build() if os.path.exists(_build.NVCC) else _build.LIB
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing and nvcc is not available to build it; "
                           "there is no CPU fallback")
    lib = C.CDLL(path)
    sig = {
        "rr_create": (C.c_int, [C.POINTER(rr_config), C.POINTER(_VP)]),
        "rr_destroy": (C.c_int, [_VP]),
        "rr_error_string": (C.c_char_p, [C.c_int]),
        "rr_get_mu": (C.c_int, [_VP, _VP]),
        "rr_get_ze": (C.c_int, [_VP, _VP]),
        "rr_get_weights": (C.c_int, [_VP, _VP]),
        "rr_set_data": (C.c_int, [_VP, _VP, _VP, _I64, _VP, _VP, _VP, _I32, _VP]),
        "rr_build_ld_table": (C.c_int, [_VP, _VP, _VP, _I64, _VP]),
        "rr_table_ptr": (_VP, [_VP]),
        "rr_istar_ptr": (_VP, [_VP]),
        "rr_get_table": (C.c_int, [_VP, _VP, _VP]),
        "rr_evaluate": (C.c_int, [_VP, _VP, _I32, _I64, _VP, _VP, _VP]),
        "rr_evaluate_flat": (C.c_int, [_VP, _VP, _VP, _I64, _VP, _VP, _VP, _I32, _VP, _I32, _I64,
                                       _VP, _VP, _VP]),
        "rr_orbit_z": (C.c_int, [_VP, _VP, _I32, _I64, _VP, _I32, _VP]),
        "rr_orbit_z_noalloc": (C.c_int, [_VP, _VP, _I32, _I64, _VP, _I32, _VP]),
        "rr_num_subsamples": (_I64, [_VP]),
        "rr_num_tiles": (_I64, [_VP]),
        "rr_get_tiles": (C.c_int, [_VP, _VP, _VP, _VP, _VP, _VP]),
        "rr_set_reduction": (C.c_int, [_VP, _I32]),
        "rr_evaluate_host": (C.c_int, [_VP, _VP, _VP, _I32, _I64, _VP, _VP]),
        "rr_enable_counters": (C.c_int, [_VP, _I32]),
        "rr_get_counters": (C.c_int, [_VP, _VP]),
        "rr_launch_count": (_I64, [_VP]),
        "rr_measure_fma_peak": (C.c_int, [_I32, C.POINTER(_DBL), _VP]),
        "rr_set_table_mode": (C.c_int, [_VP, _I32]),
        "rr_get_rows": (C.c_int, [_VP, _VP]),
        "rr_set_mean_k_weights": (C.c_int, [_VP, _I32]),
        "rr_set_orbit_poly": (C.c_int, [_VP, _I32]),
        "rr_set_lens_poly": (C.c_int, [_VP, _I32]),
        "rr_set_small_planet": (C.c_int, [_VP, _DBL]),
        "rr_build_ld_table_law": (C.c_int, [_VP, _I32, _VP, _I32, _I64, _VP]),
        "rr_math_probe": (C.c_int, [_I32, _I32, _VP, _VP, _I64, _VP, _VP, _VP]),
        "rr_enable_kernel_timing": (C.c_int, [_VP, _I32]),
        "rr_get_kernel_times": (C.c_int, [_VP, _VP, C.POINTER(_I64)]),
    }
    for name, (res, args) in sig.items():
        f = getattr(lib, name)
        f.restype, f.argtypes = res, args
    _lib = lib
    return lib


def error_string(code: int) -> str:
    return load().rr_error_string(int(code)).decode()


def _check(code: int, where: str):
    if code != 0:
        raise RoadRunnerError(code, where)


def _stream(stream=None) -> int:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return int(s.cuda_stream)


def _dev(t, dtype, name):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name} must be a CUDA tensor")
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name} must be contiguous {dtype}, got {t.dtype}")
    return t.data_ptr()


def _host(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


# What the library was told about each ctx (rr_create, rr_set_data, rr_build_ld_table*), kept so
# that the wrappers can refuse a tensor of the wrong dtype or size BEFORE the kernels read or write
# out of bounds: the C side sees raw pointers only.
_CTX: dict[int, dict] = {}


def _info(ctx: int, where: str) -> dict:
    try:
        return _CTX[int(ctx)]
    except KeyError:
        raise ValueError(f"{where}: unknown ctx handle (not made by rr_create, or destroyed)") from None


def _torch_dtype(code: str):
    import torch
    return {"f64": torch.float64, "f32": torch.float32}[code]


def _in_code(info) -> str:       # ldp, istar, table
    return "f32" if info["precision"] != RR_FP64 else "f64"


def _flux_code(info) -> str:     # flux (fp64 in RR_MIXED)
    return "f32" if info["precision"] == RR_FP32 else "f64"


def _numel(t, n: int, name: str, where: str):
    if int(t.numel() if hasattr(t, "numel") else t.size) != int(n):
        have = int(t.numel() if hasattr(t, "numel") else t.size)
        raise ValueError(f"{where}: {name} must hold {n} elements, got {have}")


# ---- one-to-one wrappers of the C entry points ----------------------------------------------------
def rr_create(nzin=50, nzlimb=50, zcut=0.7, ng=100, nk=50, k0=0.02, k1=0.2, npb=1, nkpb=1,
              precision=RR_FP64) -> int:
    cfg = rr_config(nzin, nzlimb, zcut, ng, nk, k0, k1, npb, nkpb, precision)
    h = _VP()
    _check(load().rr_create(C.byref(cfg), C.byref(h)), "rr_create")
    _CTX[int(h.value)] = dict(precision=int(precision), nz=int(nzin) + int(nzlimb), ng=int(ng),
                              nk=int(nk), npb=int(npb), nkpb=int(nkpb), npt=0, npv=0)
    return h.value


def rr_destroy(ctx: int):
    _check(load().rr_destroy(ctx), "rr_destroy")
    _CTX.pop(int(ctx), None)


def rr_get_mu(ctx: int, nz: int) -> np.ndarray:
    out = np.empty(nz)
    _check(load().rr_get_mu(ctx, out.ctypes.data), "rr_get_mu")
    return out


def rr_get_ze(ctx: int, nz: int) -> np.ndarray:
    out = np.empty(nz + 1)
    _check(load().rr_get_ze(ctx, out.ctypes.data), "rr_get_ze")
    return out


def rr_get_weights(ctx: int, nk: int, ng: int, nz: int) -> np.ndarray:
    out = np.empty((nk, ng, nz))
    _check(load().rr_get_weights(ctx, out.ctypes.data), "rr_get_weights")
    return out


def rr_set_data(ctx: int, times, lc_index, passband_index, supersampling, exposure_time,
                stream=None):
    """times f64 [npt] and lc_index i32 [npt]: CUDA tensors; the per-light-curve arrays: host."""
    import torch
    pb, ns, et = _host(passband_index, np.int32), _host(supersampling, np.int32), \
        _host(exposure_time, np.float64)
    if not (pb.size == ns.size == et.size):
        raise ValueError("passband_index, supersampling, exposure_time must have nlc entries each")
    if times.numel() != lc_index.numel():
        raise ValueError("times and lc_index must have npt entries each")
    _check(load().rr_set_data(ctx, _dev(times, torch.float64, "times"),
                              _dev(lc_index, torch.int32, "lc_index"), times.numel(),
                              pb.ctypes.data, ns.ctypes.data, et.ctypes.data, pb.size,
                              _stream(stream)), "rr_set_data")
    _info(ctx, "rr_set_data")["npt"] = int(times.numel())


def rr_build_ld_table(ctx: int, ldp, npv: int, istar=None, stream=None):
    """ldp [npv][npb][nz] CUDA tensor in the ctx input precision (fp32 for RR_FP32 / RR_MIXED);
    istar [npv][npb] optional, same dtype.  TypeError / ValueError on a dtype or size mismatch."""
    info = _info(ctx, "rr_build_ld_table")
    dt = _torch_dtype(_in_code(info))
    npv = int(npv)
    pl = _dev(ldp, dt, "ldp")
    _numel(ldp, npv * info["npb"] * info["nz"], "ldp [npv][npb][nz]", "rr_build_ld_table")
    pi = None
    if istar is not None:
        pi = _dev(istar, dt, "istar")
        _numel(istar, npv * info["npb"], "istar [npv][npb]", "rr_build_ld_table")
    _check(load().rr_build_ld_table(ctx, pl, pi, npv, _stream(stream)), "rr_build_ld_table")
    info["npv"] = npv


def rr_build_ld_table_law(ctx: int, law, ldc, npv: int, stream=None):
    """law: RR_LD_* code or a name of LD_LAWS; ldc f64 CUDA tensor [npv][npb][nldc] (or None for
    the uniform law)."""
    import torch
    info = _info(ctx, "rr_build_ld_table_law")
    code = LD_LAWS[law] if isinstance(law, str) else int(law)
    nldc = 0 if ldc is None else int(ldc.shape[-1])
    npv = int(npv)
    pc = None
    if ldc is not None:
        pc = _dev(ldc, torch.float64, "ldc")
        _numel(ldc, npv * info["npb"] * nldc, "ldc [npv][npb][nldc]", "rr_build_ld_table_law")
    _check(load().rr_build_ld_table_law(ctx, code, pc, nldc, npv, _stream(stream)),
           "rr_build_ld_table_law")
    info["npv"] = npv


def rr_evaluate(ctx: int, pv, flux, status=None, stream=None):
    """pv f64 [npv][npar] -> flux [npv][npt] (ctx precision), status i32 [npv] optional."""
    import torch
    info = _info(ctx, "rr_evaluate")
    npv, npar = pv.shape
    pf = _dev(flux, _torch_dtype(_flux_code(info)), "flux")
    if info["npt"] > 0 and npar == info["nkpb"] + 6:     # otherwise the library reports the state
        _numel(flux, npv * info["npt"], "flux [npv][npt]", "rr_evaluate")
    ps = None
    if status is not None:
        ps = _dev(status, torch.int32, "status")
        _numel(status, npv, "status [npv]", "rr_evaluate")
    _check(load().rr_evaluate(ctx, _dev(pv, torch.float64, "pv"), npar, npv, pf, ps,
                              _stream(stream)), "rr_evaluate")


def rr_evaluate_flat(ctx: int, times, lc_index, passband_index, supersampling, exposure_time, pv,
                     flux, status=None, stream=None):
    import torch
    pb, ns, et = _host(passband_index, np.int32), _host(supersampling, np.int32), \
        _host(exposure_time, np.float64)
    info = _info(ctx, "rr_evaluate_flat")
    npv, npar = pv.shape
    if not (pb.size == ns.size == et.size):
        raise ValueError("passband_index, supersampling, exposure_time must have nlc entries each")
    if times.numel() != lc_index.numel():
        raise ValueError("times and lc_index must have npt entries each")
    pf = _dev(flux, _torch_dtype(_flux_code(info)), "flux")
    _numel(flux, npv * int(times.numel()), "flux [npv][npt]", "rr_evaluate_flat")
    ps = None
    if status is not None:
        ps = _dev(status, torch.int32, "status")
        _numel(status, npv, "status [npv]", "rr_evaluate_flat")
    rc = load().rr_evaluate_flat(ctx, _dev(times, torch.float64, "times"),
                                 _dev(lc_index, torch.int32, "lc_index"), times.numel(),
                                 pb.ctypes.data, ns.ctypes.data, et.ctypes.data, pb.size,
                                 _dev(pv, torch.float64, "pv"), npar, npv, pf, ps, _stream(stream))
    if rc == 0 or rc == -5:      # RR_ESTATE comes from rr_evaluate: the data were set
        info["npt"] = int(times.numel())
    _check(rc, "rr_evaluate_flat")


def rr_orbit_z(ctx: int, pv, z, fp32_math=False, stream=None):
    import torch
    npv, npar = pv.shape
    pz = _dev(z, torch.float64, "z")
    nsub = rr_num_subsamples(ctx)
    if nsub >= 0:
        _numel(z, npv * nsub, "z [npv][nsub]", "rr_orbit_z")
    _check(load().rr_orbit_z(ctx, _dev(pv, torch.float64, "pv"), npar, npv, pz,
                             int(bool(fp32_math)), _stream(stream)), "rr_orbit_z")


RR_ESCRATCH = -7
RR_NOALLOC_SCRATCH_BYTES = 2 << 20


def rr_orbit_z_noalloc(ctx: int, pv, z, fp32_math=False, stream=None):
    """rr_orbit_z without any allocation (scratch in a static 2 MiB device array shared by all calls
    on the device: do not overlap calls); RoadRunnerError code RR_ESCRATCH beyond its limit."""
    import torch
    npv, npar = pv.shape
    pz = _dev(z, torch.float64, "z")
    nsub = rr_num_subsamples(ctx)
    if nsub >= 0:
        _numel(z, npv * nsub, "z [npv][nsub]", "rr_orbit_z_noalloc")
    _check(load().rr_orbit_z_noalloc(ctx, _dev(pv, torch.float64, "pv"), npar, npv, pz,
                                     int(bool(fp32_math)), _stream(stream)), "rr_orbit_z_noalloc")


def rr_num_subsamples(ctx: int) -> int:
    return int(load().rr_num_subsamples(ctx))


def rr_num_tiles(ctx: int) -> int:
    return int(load().rr_num_tiles(ctx))


def rr_get_tiles(ctx: int) -> dict:
    n = rr_num_tiles(ctx)
    if n < 0:
        raise RoadRunnerError(-5, "rr_get_tiles")
    start, count, lc = (np.empty(n, np.int32) for _ in range(3))
    tmin, tmax = np.empty(n), np.empty(n)
    _check(load().rr_get_tiles(ctx, start.ctypes.data, count.ctypes.data, lc.ctypes.data,
                               tmin.ctypes.data, tmax.ctypes.data), "rr_get_tiles")
    return dict(start=start, count=count, lc=lc, tmin=tmin, tmax=tmax)


def rr_set_reduction(ctx: int, mode: int):
    _check(load().rr_set_reduction(ctx, mode), "rr_set_reduction")


def rr_set_table_mode(ctx: int, mode: int):
    _check(load().rr_set_table_mode(ctx, mode), "rr_set_table_mode")


def rr_set_small_planet(ctx: int, k_threshold: float):
    _check(load().rr_set_small_planet(ctx, float(k_threshold)), "rr_set_small_planet")


def rr_set_orbit_poly(ctx: int, on: bool):
    _check(load().rr_set_orbit_poly(ctx, int(bool(on))), "rr_set_orbit_poly")


def rr_set_lens_poly(ctx: int, on: bool):
    _check(load().rr_set_lens_poly(ctx, int(bool(on))), "rr_set_lens_poly")


def rr_set_mean_k_weights(ctx: int, on: bool):
    _check(load().rr_set_mean_k_weights(ctx, int(bool(on))), "rr_set_mean_k_weights")


def rr_enable_kernel_timing(ctx: int, on: bool):
    _check(load().rr_enable_kernel_timing(ctx, int(bool(on))), "rr_enable_kernel_timing")


def rr_get_kernel_times(ctx: int) -> dict:
    """Summed device ms of the lazy row builder and of the flux kernel since the last read."""
    ms = np.zeros(2)
    calls = _I64(0)
    _check(load().rr_get_kernel_times(ctx, ms.ctypes.data, C.byref(calls)), "rr_get_kernel_times")
    return {"rows_ms": float(ms[0]), "flux_ms": float(ms[1]), "calls": int(calls.value)}


def rr_evaluate_host(ctx: int, ldp: np.ndarray, pv: np.ndarray, flux: np.ndarray,
                     status: np.ndarray | None = None):
    """Whole step from HOST arrays (numpy, or the .numpy() view of a pinned torch tensor)."""
    info = _info(ctx, "rr_evaluate_host")
    if not (ldp.flags.c_contiguous and pv.flags.c_contiguous and flux.flags.c_contiguous):
        raise TypeError("host arrays must be C-contiguous")
    want_in = np.float32 if info["precision"] != RR_FP64 else np.float64
    want_out = np.float32 if info["precision"] == RR_FP32 else np.float64
    if pv.dtype != np.float64 or ldp.dtype != want_in or flux.dtype != want_out:
        raise TypeError(f"pv must be float64, ldp {np.dtype(want_in)} and flux {np.dtype(want_out)} "
                        f"for this ctx; got {pv.dtype}, {ldp.dtype}, {flux.dtype}")
    npv, npar = pv.shape
    _numel(ldp, npv * info["npb"] * info["nz"], "ldp [npv][npb][nz]", "rr_evaluate_host")
    if info["npt"] > 0 and npar == info["nkpb"] + 6:
        _numel(flux, npv * info["npt"], "flux [npv][npt]", "rr_evaluate_host")
    if status is not None:
        if status.dtype != np.int32 or not status.flags.c_contiguous:
            raise TypeError("status must be C-contiguous int32")
        _numel(status, npv, "status [npv]", "rr_evaluate_host")
    _check(load().rr_evaluate_host(ctx, ldp.ctypes.data, pv.ctypes.data, npar, npv,
                                   flux.ctypes.data,
                                   None if status is None else status.ctypes.data),
           "rr_evaluate_host")


def rr_math_probe(op, a, b=None, fp32_math=False, stream=None):
    """Device math of the hot path applied element by element (tests): a, b fp64 CUDA tensors of
    n entries -> (out0, out1) fp64 CUDA tensors."""
    import torch
    code = PROBE_OPS[op] if isinstance(op, str) else int(op)
    n = a.numel()
    if b is not None and b.numel() != n:
        raise ValueError("rr_math_probe: a and b must have the same number of elements")
    o0 = torch.empty(n, dtype=torch.float64, device=a.device)
    o1 = torch.zeros(n, dtype=torch.float64, device=a.device)
    _check(load().rr_math_probe(code, int(bool(fp32_math)), _dev(a, torch.float64, "a"),
                                None if b is None else _dev(b, torch.float64, "b"), n,
                                o0.data_ptr(), o1.data_ptr(), _stream(stream)), "rr_math_probe")
    return o0, o1


def rr_enable_counters(ctx: int, on: bool):
    _check(load().rr_enable_counters(ctx, int(bool(on))), "rr_enable_counters")


COUNTER_NAMES = ("skipped", "circular", "eccentric", "occulting", "ingress", "solver_iters",
                 "tiles_filled", "tiles_evaluated", "eccentric_poly")


def rr_get_counters(ctx: int) -> dict:
    out = np.zeros(9, np.int64)
    _check(load().rr_get_counters(ctx, out.ctypes.data), "rr_get_counters")
    return dict(zip(COUNTER_NAMES, (int(x) for x in out)))


def rr_launch_count(ctx: int) -> int:
    return int(load().rr_launch_count(ctx))


def rr_measure_fma_peak(precision=RR_FP64, stream=None) -> float:
    v = _DBL()
    _check(load().rr_measure_fma_peak(precision, C.byref(v), _stream(stream)),
           "rr_measure_fma_peak")
    return v.value


# ---- convenience wrapper ----------------------------------------------------------------------------
class RoadRunner:
    """The paper's call pattern over the C-ABI.  Holds the ctx handle."""

    def __init__(self, nzin=50, nzlimb=50, zcut=0.7, ng=100, nk=50, k0=0.02, k1=0.2, npb=1,
                 nkpb=1, precision=RR_FP64):
        import torch
        self.nz, self.ng, self.nk, self.npb, self.nkpb = nzin + nzlimb, ng, nk, npb, nkpb
        self.precision = precision
        self.dtype = torch.float32 if precision != RR_FP64 else torch.float64     # ldp, istar, table
        self.flux_dtype = torch.float32 if precision == RR_FP32 else torch.float64
        self.ctx = rr_create(nzin, nzlimb, zcut, ng, nk, k0, k1, npb, nkpb, precision)
        self.mu = rr_get_mu(self.ctx, self.nz)
        self.ze = rr_get_ze(self.ctx, self.nz)
        self.npt = 0
        self.npv = 0

    @classmethod
    def from_config(cls, m, precision=RR_FP64):
        return cls(m.nzin, m.nzlimb, m.zcut, m.ng, m.nk, m.k0, m.k1, m.npb, m.nkpb, precision)

    def close(self):
        if getattr(self, "ctx", None):
            rr_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def weights(self) -> np.ndarray:
        return rr_get_weights(self.ctx, self.nk, self.ng, self.nz)

    def set_data(self, times, lc_index, passband_index, supersampling, exposure_time):
        import torch
        t = torch.as_tensor(np.ascontiguousarray(times, np.float64)).cuda()
        lc = torch.as_tensor(np.ascontiguousarray(lc_index, np.int32)).cuda()
        rr_set_data(self.ctx, t, lc, passband_index, supersampling, exposure_time)
        self.npt = t.numel()

    def build_ld_table(self, ldp, istar=None):
        """ldp: CUDA tensor or array [npv][npb][nz]."""
        import torch
        if not isinstance(ldp, torch.Tensor):
            ldp = torch.as_tensor(np.ascontiguousarray(ldp))
        ldp = ldp.to(device="cuda", dtype=self.dtype).reshape(-1, self.npb, self.nz).contiguous()
        if istar is not None:
            if not isinstance(istar, torch.Tensor):
                istar = torch.as_tensor(np.ascontiguousarray(istar))
            istar = istar.to(device="cuda", dtype=self.dtype).contiguous()
        self.npv = ldp.shape[0]
        rr_build_ld_table(self.ctx, ldp, self.npv, istar)

    def build_ld_table_law(self, law, ldc):
        """Named law on the device: ldc array or CUDA tensor [npv][npb][nldc] (fp64)."""
        import torch
        if ldc is not None and not isinstance(ldc, torch.Tensor):
            ldc = torch.as_tensor(np.ascontiguousarray(ldc, np.float64)).cuda()
        if ldc is not None:
            ldc = ldc.reshape(-1, self.npb, ldc.shape[-1]).contiguous()
        self.npv = int(ldc.shape[0]) if ldc is not None else self.npv
        rr_build_ld_table_law(self.ctx, law, ldc, self.npv)

    def profile_and_istar(self):
        """Diagnostics: Istar[npv][npb] of the last table build (numpy)."""
        npdt = np.float32 if self.precision != RR_FP64 else np.float64
        I = np.empty((self.npv, self.npb), npdt)
        _check(load().rr_get_table(self.ctx, None, I.ctypes.data), "rr_get_table")
        return I

    def table(self):
        """Copy of T[npv][npb][nk][ng] and Istar[npv][npb] as numpy arrays (diagnostics)."""
        npdt = np.float32 if self.precision != RR_FP64 else np.float64
        T = np.empty((self.npv, self.npb, self.nk, self.ng), npdt)
        I = np.empty((self.npv, self.npb), npdt)
        _check(load().rr_get_table(self.ctx, T.ctypes.data, I.ctypes.data), "rr_get_table")
        return T, I

    def rows(self):
        """Copy of the collapsed rows ldw[npv][npb][ng] of the last evaluate (lazy / direct mode)."""
        npdt = np.float32 if self.precision != RR_FP64 else np.float64
        out = np.empty((self.npv, self.npb, self.ng), npdt)
        _check(load().rr_get_rows(self.ctx, out.ctypes.data), "rr_get_rows")
        return out

    def evaluate(self, pv, want_status=False):
        """pv: CUDA tensor or array [npv][nkpb+6] -> flux CUDA tensor [npv][npt]."""
        import torch
        if not isinstance(pv, torch.Tensor):
            pv = torch.as_tensor(np.ascontiguousarray(pv, np.float64)).cuda()
        pv = pv.reshape(-1, self.nkpb + 6).contiguous()
        flux = torch.empty((pv.shape[0], self.npt), dtype=self.flux_dtype, device="cuda")
        status = torch.empty(pv.shape[0], dtype=torch.int32, device="cuda")
        rr_evaluate(self.ctx, pv, flux, status)
        return (flux, status) if want_status else flux

    def evaluate_ps(self, k, t0, p, a, i, e=0.0, w=0.0):
        """The paper's call ``evaluate(k, ldc, t0, p, a, i, e, w)`` with the
        profile already set by ``build_ld_table*``: scalars give flux of shape (npt,), arrays of
        npv entries give (npv, npt); k may be (npv,) or (npv, nkpb).  Marshalling only."""
        args = [np.atleast_1d(np.asarray(x, np.float64)) for x in (t0, p, a, i, e, w)]
        k = np.asarray(k, np.float64)
        scalar = k.ndim == 0 and all(x.size == 1 for x in args)
        k = k.reshape(1, -1) if k.ndim <= 1 and self.nkpb > 1 and k.size == self.nkpb else \
            k.reshape(-1, self.nkpb) if k.ndim == 2 else k.reshape(-1, 1)
        npv = max([k.shape[0]] + [x.size for x in args])
        if k.shape[1] == 1 and self.nkpb > 1:
            k = np.repeat(k, self.nkpb, axis=1)
        pv = np.empty((npv, self.nkpb + 6))
        pv[:, :self.nkpb] = np.broadcast_to(k, (npv, self.nkpb))
        for col, x in enumerate(args):
            pv[:, self.nkpb + col] = np.broadcast_to(x, (npv,))
        flux = self.evaluate(pv)
        return flux[0] if scalar else flux

    def orbit_z(self, pv, fp32_math=False):
        import torch
        if not isinstance(pv, torch.Tensor):
            pv = torch.as_tensor(np.ascontiguousarray(pv, np.float64)).cuda()
        pv = pv.reshape(-1, self.nkpb + 6).contiguous()
        z = torch.empty((pv.shape[0], rr_num_subsamples(self.ctx)), dtype=torch.float64,
                        device="cuda")
        rr_orbit_z(self.ctx, pv, z, fp32_math)
        return z

    def evaluate_host(self, ldp: np.ndarray, pv: np.ndarray, flux: np.ndarray | None = None,
                      status: np.ndarray | None = None):
        npdt = np.float32 if self.precision != RR_FP64 else np.float64
        ldp = np.ascontiguousarray(ldp, npdt).reshape(-1, self.npb, self.nz)
        pv = np.ascontiguousarray(pv, np.float64).reshape(-1, self.nkpb + 6)
        if flux is None:
            flux = np.empty((pv.shape[0], self.npt),
                            np.float32 if self.precision == RR_FP32 else np.float64)
        rr_evaluate_host(self.ctx, ldp, pv, flux, status)
        return flux
