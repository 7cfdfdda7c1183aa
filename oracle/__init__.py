"""oracle - TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Python face of ``roadrunner_oracle.c`` (plain scalar fp64 C, written from the paper; see its header
for layers, readings and pins) plus ``truth.py`` (Eq. (2) by quadrature).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference`` legs may import
this package.  It imports nothing from ``paper_2009_08500_b200`` and shares no code with it.

This file only marshals numpy arrays into the C functions; it holds no model arithmetic.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_lib = None
_D = C.POINTER(C.c_double)
_I = C.POINTER(C.c_int32)


def _dp(a):
    return a.ctypes.data_as(_D)


def _ip(a):
    return a.ctypes.data_as(_I)


def load():
    global _lib
    if _lib is not None:
        return _lib
    lib = C.CDLL(_build.build())
    lib.oracle_z_grid.argtypes = [C.c_double, C.c_int, C.c_int, _D, _D, _D]
    lib.oracle_z_grid.restype = None
    for name in ("oracle_lens_area", "oracle_lens_area_acos"):
        f = getattr(lib, name)
        f.argtypes = [C.c_double] * 3
        f.restype = C.c_double
    lib.oracle_weights.argtypes = [C.c_double, C.c_double, _D, C.c_int, _D]
    lib.oracle_weights.restype = None
    lib.oracle_weight_tensor.argtypes = [C.c_int, C.c_double, C.c_double, C.c_int, _D, C.c_int, _D]
    lib.oracle_weight_tensor.restype = None
    lib.oracle_ld_table.argtypes = [_D, C.c_int, C.c_int, C.c_int, _D, C.c_int64, _D]
    lib.oracle_ld_table.restype = None
    lib.oracle_istar.argtypes = [_D, C.c_int, _D, C.c_int64, _D]
    lib.oracle_istar.restype = None
    lib.oracle_direct_flux.argtypes = [C.c_double, C.c_double, _D, C.c_int, _D, C.c_double]
    lib.oracle_direct_flux.restype = C.c_double
    lib.oracle_kepler.argtypes = [C.c_double, C.c_double, _D]
    lib.oracle_kepler.restype = C.c_int
    lib.oracle_separation.argtypes = [C.c_double] * 7 + [C.POINTER(C.c_int)]
    lib.oracle_separation.restype = C.c_double
    lib.oracle_flux_from_table.argtypes = [C.c_double, C.c_double, _D, C.c_int, C.c_double,
                                           C.c_double, C.c_int, C.c_double]
    lib.oracle_flux_from_table.restype = C.c_double
    lib.oracle_evaluate.argtypes = [_D, _I, C.c_int64, _I, _I, _D, C.c_int32,
                                    _D, C.c_int32, C.c_int64, _D, _D,
                                    C.c_int32, C.c_int32, C.c_double, C.c_double, C.c_int32,
                                    _D, _I, _D, C.c_int32]
    lib.oracle_evaluate.restype = None
    lib.oracle_evaluate_mk.argtypes = [_D, _I, C.c_int64, _I, _I, _D, C.c_int32,
                                       _D, C.c_int32, C.c_int64, _D, _D,
                                       C.c_int32, C.c_int32, C.c_double, C.c_double, C.c_int32,
                                       C.c_int32, _D, _I, _D, C.c_int32]
    lib.oracle_evaluate_mk.restype = None
    lib.oracle_direct_rows.argtypes = [_D, C.c_int, C.c_int, _D, _D, C.c_int64, _D]
    lib.oracle_direct_rows.restype = None
    lib.oracle_direct_rows_sp.argtypes = [_D, _D, C.c_int, C.c_int, _D, _D, C.c_int64, C.c_double, _D]
    lib.oracle_direct_rows_sp.restype = None
    lib.oracle_direct_rows_pv.argtypes = [_D, _D, C.c_int, C.c_int, _D, C.c_int32, C.c_int32,
                                          C.c_int64, C.c_int32, _D, C.c_double, _D]
    lib.oracle_direct_rows_pv.restype = None
    lib.oracle_profile_at.argtypes = [C.c_double, _D, _D, C.c_int]
    lib.oracle_profile_at.restype = C.c_double
    lib.oracle_flux_from_row.argtypes = [C.c_double, C.c_double, _D, C.c_int, C.c_double]
    lib.oracle_flux_from_row.restype = C.c_double
    lib.oracle_evaluate_direct.argtypes = [_D, _I, C.c_int64, _I, _I, _D, _D, C.c_int32,
                                           C.c_int64, _D, _D, C.c_int32, C.c_int32, C.c_int32,
                                           _D, _I, C.c_int32]
    lib.oracle_evaluate_direct.restype = None
    _lib = lib
    return lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


# ---- scalar / small helpers ---------------------------------------------------------------------
def z_grid(zcut, nzin, nzlimb):
    nz = nzin + nzlimb
    ze, zm, mu = np.empty(nz + 1), np.empty(nz), np.empty(nz)
    load().oracle_z_grid(zcut, nzin, nzlimb, _dp(ze), _dp(zm), _dp(mu))
    return ze, zm, mu


def lens_area(r1, r2, d):
    return load().oracle_lens_area(float(r1), float(r2), float(d))


def lens_area_acos(r1, r2, d):
    return load().oracle_lens_area_acos(float(r1), float(r2), float(d))


def weights(c, k, ze):
    ze = _f64(ze)
    w = np.empty(ze.size - 1)
    load().oracle_weights(float(c), float(k), _dp(ze), ze.size - 1, _dp(w))
    return w


def istar(ze, ldp):
    ze, ldp = _f64(ze), _f64(ldp)
    rows = ldp.reshape(-1, ze.size - 1)
    out = np.empty(rows.shape[0])
    load().oracle_istar(_dp(ze), ze.size - 1, _dp(rows), rows.shape[0], _dp(out))
    return out.reshape(ldp.shape[:-1])


def direct_flux(k, c, ze, ldp, istar_value):
    ze, ldp = _f64(ze), _f64(ldp)
    return load().oracle_direct_flux(float(k), float(c), _dp(ze), ze.size - 1, _dp(ldp),
                                     float(istar_value))


def kepler(M, e):
    E = C.c_double()
    it = load().oracle_kepler(float(M), float(e), C.byref(E))
    return E.value, it


def separation(t, t0, p, a, inc, e, w):
    front = C.c_int()
    z = load().oracle_separation(float(t), float(t0), float(p), float(a), float(inc), float(e),
                                 float(w), C.byref(front))
    return z, bool(front.value)


# ---- the L2 model ---------------------------------------------------------------------------------
class OracleModel:
    """Interpolated RoadRunner model: grid + weight tensor built at creation."""

    def __init__(self, nzin=50, nzlimb=50, zcut=0.7, ng=100, nk=50, k0=0.02, k1=0.2, npb=1,
                 nkpb=1):
        self.nzin, self.nzlimb, self.zcut = int(nzin), int(nzlimb), float(zcut)
        self.ng, self.nk, self.k0, self.k1 = int(ng), int(nk), float(k0), float(k1)
        self.npb, self.nkpb = int(npb), int(nkpb)
        self.nz = self.nzin + self.nzlimb
        self.ze, self.zm, self.mu = z_grid(self.zcut, self.nzin, self.nzlimb)
        self.W = np.empty((self.nk, self.ng, self.nz))
        load().oracle_weight_tensor(self.nk, self.k0, self.k1, self.ng, _dp(self.ze), self.nz,
                                    _dp(self.W))
        self.T = None
        self.istar = None

    @classmethod
    def from_config(cls, m):
        return cls(m.nzin, m.nzlimb, m.zcut, m.ng, m.nk, m.k0, m.k1, m.npb, m.nkpb)

    def build_ld_table(self, ldp, istar_override=None):
        ldp = _f64(ldp).reshape(-1, self.npb, self.nz)
        npv = ldp.shape[0]
        self.T = np.empty((npv, self.npb, self.nk, self.ng))
        load().oracle_ld_table(_dp(self.W), self.nk, self.ng, self.nz, _dp(ldp), npv * self.npb,
                               _dp(self.T))
        if istar_override is None:
            self.istar = istar(self.ze, ldp)
        else:
            self.istar = _f64(istar_override).reshape(npv, self.npb).copy()
        return self.T, self.istar

    def evaluate(self, times, lc_index, passband_index, supersampling, exposure_time, pv,
                 nthreads=1, want_z=False, mean_k_weights=False):
        times, pv = _f64(times), _f64(pv)
        pv = pv.reshape(-1, self.nkpb + 6)
        lc_index, passband_index = _i32(lc_index), _i32(passband_index)
        supersampling, exposure_time = _i32(supersampling), _f64(exposure_time)
        npv, npt = pv.shape[0], times.size
        assert self.T is not None and self.T.shape[0] == npv, "build_ld_table first (same npv)"
        assert lc_index.size == npt and lc_index.min() >= 0 and lc_index.max() < passband_index.size
        assert passband_index.min() >= 0 and passband_index.max() < self.npb
        flux = np.empty((npv, npt))
        status = np.empty(npv, np.int32)
        z = None
        if want_z:
            nsub = int(supersampling.astype(np.int64)[lc_index].sum())
            z = np.empty((npv, nsub))
        load().oracle_evaluate_mk(_dp(times), _ip(lc_index), npt, _ip(passband_index),
                                  _ip(supersampling), _dp(exposure_time), passband_index.size,
                                  _dp(pv), self.nkpb, npv, _dp(self.T), _dp(self.istar),
                                  self.npb, self.nk, self.k0, self.k1, self.ng,
                                  int(bool(mean_k_weights)),
                                  _dp(flux), _ip(status), _dp(z) if want_z else None,
                                  int(nthreads))
        return (flux, status, z) if want_z else (flux, status)


class OracleDirectModel:
    """Direct RoadRunner model: weights at each pv's own k, g interpolation
    only.  Marshalling only; the arithmetic is oracle_direct_rows / oracle_evaluate_direct."""

    def __init__(self, nzin=50, nzlimb=50, zcut=0.7, ng=100, npb=1, nkpb=1):
        self.nzin, self.nzlimb, self.zcut = int(nzin), int(nzlimb), float(zcut)
        self.ng, self.npb, self.nkpb = int(ng), int(npb), int(nkpb)
        self.nz = self.nzin + self.nzlimb
        self.ze, self.zm, self.mu = z_grid(self.zcut, self.nzin, self.nzlimb)

    @classmethod
    def from_config(cls, m):
        return cls(m.nzin, m.nzlimb, m.zcut, m.ng, m.npb, m.nkpb)

    def rows(self, ldp, pv, mean_k_weights=False, small_planet_k=0.0):
        """ldw[npv][npb][ng] and Istar[npv][npb] for the k of every (pv, passband); with
        mean_k_weights the weights of every passband are taken at the pv's mean k.
        Rows of pvs with an invalid k are NaN (oracle_direct_rows_pv)."""
        ldp = _f64(ldp).reshape(-1, self.npb, self.nz)
        pv = _f64(pv).reshape(-1, self.nkpb + 6)
        npv = ldp.shape[0]
        out = np.empty((npv, self.npb, self.ng))
        load().oracle_direct_rows_pv(_dp(self.ze), _dp(self.zm), self.nz, self.ng, _dp(pv),
                                     self.nkpb, self.npb, npv, int(bool(mean_k_weights)), _dp(ldp),
                                     float(small_planet_k), _dp(out))
        return out, istar(self.ze, ldp)

    def evaluate(self, times, lc_index, passband_index, supersampling, exposure_time, pv, ldp,
                 nthreads=1, mean_k_weights=False, small_planet_k=0.0):
        times, pv = _f64(times), _f64(pv).reshape(-1, self.nkpb + 6)
        lc_index, passband_index = _i32(lc_index), _i32(passband_index)
        supersampling, exposure_time = _i32(supersampling), _f64(exposure_time)
        rows, ist = self.rows(ldp, pv, mean_k_weights, small_planet_k)
        npv, npt = pv.shape[0], times.size
        flux = np.empty((npv, npt))
        status = np.empty(npv, np.int32)
        load().oracle_evaluate_direct(_dp(times), _ip(lc_index), npt, _ip(passband_index),
                                      _ip(supersampling), _dp(exposure_time), _dp(pv), self.nkpb,
                                      npv, _dp(rows), _dp(ist), self.npb, self.ng,
                                      int(bool(mean_k_weights)), _dp(flux), _ip(status),
                                      int(nthreads))
        return flux, status


def profile_at(z, zm, ldp):
    zm, ldp = _f64(zm), _f64(ldp)
    return load().oracle_profile_at(float(z), _dp(zm), _dp(ldp), zm.size)


def flux_from_row(z, k, ldw, istar_value):
    ldw = _f64(ldw)
    return load().oracle_flux_from_row(float(z), float(k), _dp(ldw), ldw.size, float(istar_value))


def evaluate_workload(wl, nthreads=1, want_z=False):
    """Run a ``workloads.Workload`` through the L2 oracle (model built here)."""
    m = OracleModel.from_config(wl.model)
    m.build_ld_table(wl.ldp(m.mu))
    return m.evaluate(wl.times, wl.lc_index, wl.passband_index, wl.supersampling,
                      wl.exposure_time, wl.pv, nthreads=nthreads, want_z=want_z)
