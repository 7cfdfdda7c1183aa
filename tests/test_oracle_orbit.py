"""Pins for the oracle's orbit, supersampling and heterogeneous-indexing steps (CPU only).

Citations: PAPER.md lines; readings R* in DESIGN.md section 3.  None of these retypes the oracle's
own formula: each compares it with something fixed by the mathematics (Kepler's equation itself,
a vector-rotation construction of the orbit, scipy's root finder, closed-form special cases) or
with the same oracle called on differently arranged input.
"""
import math

import numpy as np
import pytest
from scipy.optimize import brentq

import oracle
from workloads import make_workload, paper_dummy_example


# ---- Kepler's equation ----------------------------------------------------------------------------
@pytest.mark.parametrize("e", [0.0, 1e-8, 0.1, 0.3, 0.5, 0.7, 0.9, 0.99])
def test_kepler_residual_and_iterations(e):
    """E - e sin E = M to 1e-15 for M over [-pi, pi); the safeguarded Newton converges in a handful
    of steps, never by running into the 50-iteration cap (R8)."""
    worst_it = 0
    for M in np.linspace(-math.pi, math.pi, 721, endpoint=False):
        E, it = oracle.kepler(M, e)
        assert abs(E - e * math.sin(E) - M) <= 4e-15, (M, e)
        worst_it = max(worst_it, it)
    assert worst_it <= 15


def test_kepler_vs_bracketing_root_finder():
    """An independent solver (scipy brentq on the same equation) lands on the same root."""
    rng = np.random.default_rng(5)
    for _ in range(200):
        e, M = rng.uniform(0, 0.95), rng.uniform(-math.pi, math.pi)
        want = brentq(lambda E: E - e * math.sin(E) - M, M - 1.0, M + 1.0, xtol=1e-15, rtol=1e-15)
        assert abs(oracle.kepler(M, e)[0] - want) < 5e-14


# ---- separation -----------------------------------------------------------------------------------
def _separation_by_rotation(t, t0, p, a, inc, e, w):
    """Independent construction: solve Kepler by brentq, place the planet in the orbital plane
    (pericentre on +x), rotate by w about the orbit normal, tilt by the inclination, project.
    Observer along +Z_sky... sky plane = (X, Y cos i); in front iff the line-of-sight coordinate
    Y sin i > 0.  t0 is inferior conjunction: X = 0 with the planet in front."""
    def mean_anomaly_of_true(f):
        E = 2 * math.atan2(math.sqrt(1 - e) * math.sin(f / 2), math.sqrt(1 + e) * math.cos(f / 2))
        return E - e * math.sin(E)
    M = mean_anomaly_of_true(math.pi / 2 - w) + 2 * math.pi * (t - t0) / p
    M = (M + math.pi) % (2 * math.pi) - math.pi
    E = brentq(lambda E: E - e * math.sin(E) - M, M - 1.0, M + 1.0, xtol=1e-15, rtol=1e-15)
    x, y = a * (math.cos(E) - e), a * math.sqrt(1 - e * e) * math.sin(E)
    X = x * math.cos(w) - y * math.sin(w)
    Y = x * math.sin(w) + y * math.cos(w)
    return math.hypot(X, Y * math.cos(inc)), Y * math.sin(inc) > 0


def test_separation_vs_rotation_construction():
    rng = np.random.default_rng(11)
    for _ in range(400):
        e = rng.choice([0.0, rng.uniform(0, 0.8)])
        w = rng.uniform(0, 2 * math.pi)
        p, a, t0 = rng.uniform(1, 10), rng.uniform(3, 20), rng.uniform(-0.1, 0.1)
        inc = math.acos(rng.uniform(0, 1.2) / a)
        t = rng.uniform(-6, 6)
        z, front = oracle.separation(t, t0, p, a, inc, e, w)
        z2, front2 = _separation_by_rotation(t, t0, p, a, inc, e, w)
        assert abs(z - z2) < 2e-12 * max(1.0, a), (e, w, t)
        if abs(z2 - a) > 1e-6:                      # away from quadrature the side is unambiguous
            assert front == front2


def test_eccentric_branch_at_e_zero_equals_circular():
    """e, w default to 0 = circular.  A tiny e through the Kepler branch must land on
    the circular closed form (continuity in e), for any w."""
    rng = np.random.default_rng(3)
    for _ in range(200):
        p, a, t0 = rng.uniform(1, 10), rng.uniform(3, 20), rng.uniform(-0.1, 0.1)
        inc = math.acos(rng.uniform(0, 1) / a)
        t = rng.uniform(-5, 5)
        zc, fc = oracle.separation(t, t0, p, a, inc, 0.0, 0.0)
        ze, fe = oracle.separation(t, t0, p, a, inc, 1e-300, rng.uniform(0, 2 * math.pi))
        assert abs(zc - ze) < 1e-12 * a
        if abs(zc - a) > 1e-6:
            assert fc == fe


def test_z_at_conjunction_is_impact_parameter():
    """R8: z(t0) = a cos i (1 - e^2) / (1 + e sin w), planet in front; half a period later (circular)
    it is behind the star."""
    rng = np.random.default_rng(8)
    for _ in range(200):
        e, w = rng.uniform(0, 0.8), rng.uniform(0, 2 * math.pi)
        p, a, t0 = rng.uniform(1, 10), rng.uniform(3, 20), rng.uniform(-1, 1)
        inc = math.acos(rng.uniform(0, 1) / a)
        z, front = oracle.separation(t0, t0, p, a, inc, e, w)
        assert front
        assert abs(z - a * math.cos(inc) * (1 - e * e) / (1 + e * math.sin(w))) < 1e-12 * a
    z, front = oracle.separation(1.5, 0.0, 3.0, 8.0, 1.5, 0.0, 0.0)
    assert not front


def test_z_periodic_in_p():
    for e, w in [(0.0, 0.0), (0.4, 1.0)]:
        z0, f0 = oracle.separation(0.0123, 0.001, 2.5, 9.0, 1.52, e, w)
        for n in (1, -1, 7):
            z1, f1 = oracle.separation(0.0123 + n * 2.5, 0.001, 2.5, 9.0, 1.52, e, w)
            assert abs(z0 - z1) < 1e-11 and f0 == f1


# ---- flux invariants through the whole L2 evaluation -------------------------------------------
def _small(config, npv, npt):
    return make_workload(config, npv=npv, npt=npt)


def test_flux_invariants_population():
    """Out of transit exactly 1, never above 1, >= 1 - deficit bound; secondary-eclipse phase = 1."""
    wl = _small(4, 48, 1500)
    flux, status, z = oracle.evaluate_workload(wl, want_z=True)
    assert not status.any()
    assert np.all(flux <= 1.0) and np.all(flux > 0.8)
    k = wl.pv[:, 0]
    ns = int(wl.supersampling[0])
    zz = z.reshape(wl.npv, wl.npt, ns)
    out = np.all((zz < 0) | (zz >= 1 + k[:, None, None]), axis=2)     # behind, or clear of the disc
    assert out.any() and (~out).any()
    assert np.all(flux[out] == 1.0)
    assert np.all(flux[~out] < 1.0)


def test_circular_symmetry_about_mid_transit():
    wl = _small(0, 1, 1001)                         # symmetric time grid about t0 = 0
    flux, _ = oracle.evaluate_workload(wl)
    assert np.max(np.abs(flux[0] - flux[0, ::-1])) < 1e-14
    assert flux[0].argmin() in (499, 500, 501)


def test_continuity_at_contacts_and_monotone_ingress():
    """Flux is continuous across z = 1+k and z = 1-k, and increases with z for a monotone profile."""
    wl = _small(0, 1, 10)
    m = oracle.OracleModel.from_config(wl.model)
    m.build_ld_table(wl.ldp(m.mu))
    k = 0.1
    lib = oracle.load()
    f = lambda z: lib.oracle_flux_from_table(z, k, oracle._dp(m.T[0, 0]), m.nk, m.k0, m.k1, m.ng,
                                             float(m.istar[0, 0]))
    for zc in (1 + k, 1 - k):
        assert abs(f(zc + 1e-12) - f(zc - 1e-12)) < 1e-11
    assert f(1 + k) == 1.0 and f(1 + k + 1e-9) == 1.0
    zs = np.linspace(0, 1 + k, 4001)
    fs = np.array([f(z) for z in zs])
    assert np.all(np.diff(fs) > -1e-9)              # kinks of the g-interpolation stay below 1e-9


# ---- supersampling (reading R7) ---------------------------------------------------
def test_supersampling_equals_expanded_time_array():
    wl = _small(2, 6, 300)
    ns, tau = int(wl.supersampling[0]), float(wl.exposure_time[0])
    flux, _ = oracle.evaluate_workload(wl)
    m = oracle.OracleModel.from_config(wl.model)
    m.build_ld_table(wl.ldp(m.mu))
    # every sub-sample as its own unsupersampled exposure; offsets symmetric, inside the exposure
    off = tau * ((np.arange(ns) + 0.5) / ns - 0.5)
    assert abs(off.sum()) < 1e-17 and off.min() > -tau / 2 and off.max() < tau / 2
    t_exp = (wl.times[:, None] + off[None, :]).ravel()
    one = np.ones(1, np.int32)
    f_exp, _ = m.evaluate(t_exp, np.zeros(t_exp.size, np.int32), wl.passband_index, one,
                          np.zeros(1), wl.pv)
    assert np.max(np.abs(f_exp.reshape(wl.npv, wl.npt, ns).mean(axis=2) - flux)) < 1e-15


def test_supersampling_degenerate_cases():
    wl = _small(2, 4, 200)
    m = oracle.OracleModel.from_config(wl.model)
    m.build_ld_table(wl.ldp(m.mu))
    args = (wl.times, wl.lc_index, wl.passband_index)
    base, _ = m.evaluate(*args, np.array([1], np.int32), np.array([0.0]), wl.pv)
    n1, _ = m.evaluate(*args, np.array([1], np.int32), wl.exposure_time, wl.pv)   # ns=1: offset 0
    t0, _ = m.evaluate(*args, wl.supersampling, np.array([0.0]), wl.pv)           # tau=0
    assert np.array_equal(base, n1)
    assert np.max(np.abs(base - t0)) < 1e-15


# ---- heterogeneous indexing ---------------------------------------------------
def test_paper_dummy_example_indexing():
    """times=[0..5], lcids=[0,0,1,1,1,2], pbids=[0,1,0]: points 0,1,5 see passband 0's table,
    points 2,3,4 passband 1's; the result equals evaluating each light curve on its own."""
    ex = paper_dummy_example()
    m = oracle.OracleModel(npb=2)
    ldp = np.stack([1 - 0.2 * (1 - m.mu) - 0.1 * (1 - m.mu) ** 2,
                    1 - 0.5 * (1 - m.mu) - 0.1 * (1 - m.mu) ** 2])[None]
    m.build_ld_table(ldp)
    pv = np.array([[0.10, 0.0, 1.0, 3.0, 0.5 * math.pi, 0.0, 0.0]])
    ns, et = np.array([1, 3, 2], np.int32), np.array([0.0, 0.05, 0.02])
    times = ex["times"] * 1.0 + 0.01                                          # in transit at integers
    flux, _ = m.evaluate(times, ex["lc_index"], ex["passband_index"], ns, et, pv)
    assert np.all(flux < 1.0)
    for lc in range(3):
        sel = ex["lc_index"] == lc
        pb = int(ex["passband_index"][lc])
        single = oracle.OracleModel(npb=1)
        single.build_ld_table(ldp[:, pb:pb + 1])
        f1, _ = single.evaluate(times[sel], np.zeros(sel.sum(), np.int32), np.zeros(1, np.int32),
                                ns[lc:lc + 1], et[lc:lc + 1], pv)
        assert np.array_equal(f1[0], flux[0, sel])
    # the two passbands really differ, so a swapped index would be caught
    swapped, _ = m.evaluate(times, ex["lc_index"], np.array([1, 0, 1], np.int32), ns, et, pv)
    assert np.all(np.abs(swapped - flux) > 1e-5)


def test_chromatic_radius_ratio_picks_passband_k():
    """k of shape (npv, npb) - light curves in passband 1 use the second k."""
    ex = paper_dummy_example()
    m = oracle.OracleModel(npb=2, nkpb=2)
    ldp = np.ones((1, 2, m.nz))
    m.build_ld_table(ldp)
    pv = np.array([[0.10, 0.11, 0.0, 1.0, 3.0, 0.5 * math.pi, 0.0, 0.0]])
    one, zero = np.ones(3, np.int32), np.zeros(3)
    flux, _ = m.evaluate(ex["times"], ex["lc_index"], ex["passband_index"], one, zero, pv)
    depth = 1 - flux[0]                                  # uniform disc, centred: k^2
    assert np.allclose(depth[[0, 1, 5]], 0.10 ** 2, atol=1e-15)
    assert np.allclose(depth[[2, 3, 4]], 0.11 ** 2, atol=1e-15)


def test_invalid_parameter_vectors_give_nan_rows():
    wl = _small(1, 6, 50)
    pv = wl.pv.copy()
    pv[1, 0] = 0.5            # k above k1
    pv[2, 5] = 1.0            # e = 1
    pv[3, 3] = -1.0           # a <= 0
    pv[4, 2] = 0.0            # p <= 0
    pv[5, 1] = np.nan
    m = oracle.OracleModel.from_config(wl.model)
    m.build_ld_table(wl.ldp(m.mu))
    flux, status = m.evaluate(wl.times, wl.lc_index, wl.passband_index, wl.supersampling,
                              wl.exposure_time, pv)
    assert list(status) == [0, 1, 2, 4, 8, 16]
    assert np.all(np.isfinite(flux[0])) and np.all(np.isnan(flux[1:]))


def test_config0_worked_example():
    """Config 0 geometry: b = a cos i; the count of in-transit points matches the transit duration
    formula T14 = (p/pi) asin(sqrt((1+k)^2 - b^2) / (a sin i)) (textbook, circular)."""
    wl = make_workload(0)
    flux, _, z = oracle.evaluate_workload(wl, want_z=True)
    k, t0, p, a, inc = wl.pv[0, :5]
    b = a * math.cos(inc)
    assert abs(b - 0.279195973620) < 1e-11
    assert 0 <= z[0].min() - b < 1e-4                 # the even grid straddles t0, never hits it
    # SURVEY.md section 8(c) "Config-0 worked example": values from the survey's own throw-away
    # numpy/mpmath probe of the same readings (an implementation independent of this oracle)
    assert int((z[0] < 1 + k).sum()) == 318
    assert abs(wl.times[400] - (-0.039839840)) < 1e-9 and abs(wl.times[499] - (-0.000200200)) < 1e-9
    assert abs(z[0, 400] - 0.722469824314) < 1e-11 and abs(flux[0, 400] - 0.989752454459) < 1e-11
    assert abs(z[0, 499] - 0.279216098908) < 1e-11 and abs(flux[0, 499] - 0.988209213340) < 1e-11
    t14 = p / math.pi * math.asin(math.sqrt((1 + k) ** 2 - b * b) / (a * math.sin(inc)))
    n_in = int((flux[0] < 1).sum())
    dt = wl.times[1] - wl.times[0]
    assert abs(n_in - t14 / dt) <= 1.0
    assert abs(flux[0].min() - (1 - k * k * 1.18)) < 2e-3     # depth ~ k^2 x limb-darkening boost


def test_non_finite_times_give_nan_flux():
    """Reading R15: a NaN / infinite exposure time -> NaN flux for that exposure, every pv; the other
    exposures are untouched."""
    wl = make_workload(3, npv=3, npt=6 * 20)
    ref, _ = oracle.evaluate_workload(wl)
    bad = [5, 40, 77]
    wl.times[bad] = [np.nan, np.inf, -np.inf]
    got, _ = oracle.evaluate_workload(wl)
    assert np.all(np.isnan(got[:, bad]))
    ok = np.setdiff1d(np.arange(wl.npt), bad)
    assert np.array_equal(got[:, ok], ref[:, ok])
