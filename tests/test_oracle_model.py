"""Pins for the oracle's transit model: L0 (Eq. (2) by quadrature) <- L1 (direct Eq. (5)) <- L2
(table-interpolated).  CPU only.  Citations: PAPER.md lines; readings R* in DESIGN.md section 3."""
import math
import os

import numpy as np
import pytest

import oracle
from oracle import truth


def _golden(golden_dir):
    rows = []
    for line in open(os.path.join(golden_dir, "l0_truth.txt")):
        if line.startswith("#"):
            continue
        law, kc, F = [s.strip() for s in line.split("|")]
        name, *coeffs = law.split()
        k, c = map(float, kc.split())
        rows.append((name, tuple(map(float, coeffs)), k, c, float(F)))
    return rows


def _law(name, coeffs):
    if name == "quadratic":
        return truth.quadratic(*coeffs), truth.istar_quadratic(*coeffs)
    if name == "power2":
        return truth.power2(*coeffs), truth.istar_power2(*coeffs)
    return truth.poly(coeffs), truth.istar_poly(coeffs)


# ---- L0: the two quadratures and a hand closed form agree -------------------------------------
def test_l0_centred_closed_form(golden_dir):
    """c = 0, quadratic law: occluded = 2 pi int_{mu_k}^1 mu I(mu) dmu, elementary polynomial."""
    u1, u2 = 0.4, 0.2
    for name, coeffs, k, c, F in _golden(golden_dir):
        if name != "quadratic" or c != 0.0:
            continue
        mk = math.sqrt(1 - k * k)
        prim = lambda m: (1 - u1 - u2) * m**2 / 2 + (u1 + 2 * u2) * m**3 / 3 - u2 * m**4 / 4  # noqa
        want = 1 - 2 * math.pi * (prim(1.0) - prim(mk)) / truth.istar_quadratic(u1, u2)
        assert abs(F - want) < 1e-14


def test_l0_bruteforce_vs_golden(golden_dir):
    """Brute-force 2-D polar midpoint integration of Eq. (2) vs the 30-digit radial integral:
    <= 1e-8 absolute (north-star bound)."""
    for name, coeffs, k, c, F in _golden(golden_dir):
        ld, ist = _law(name, coeffs)
        n = 3000 if abs(c - 1) > k or c < 1 - k else 6000
        got = truth.flux_polar_bruteforce(k, c, ld, ist, nrho=n, ntheta=n)
        assert abs(got - F) < 1e-8, (name, k, c, got - F)


def test_istar_closed_forms():
    assert float(truth.istar_mp(truth.quadratic(0.4, 0.2))) == pytest.approx(
        truth.istar_quadratic(0.4, 0.2), abs=1e-15)
    assert float(truth.istar_mp(truth.power2(0.6, 0.7))) == pytest.approx(
        truth.istar_power2(0.6, 0.7), abs=1e-15)
    c = (-0.4, -0.1, -0.05, -0.02)
    assert float(truth.istar_mp(truth.poly(c))) == pytest.approx(truth.istar_poly(c), abs=1e-15)


# ---- L1 direct model converges to L0 ("no asymptotic biases") ----------------------
def test_l1_direct_converges_to_l0(golden_dir):
    ze, zm, mu = oracle.z_grid(0.7, 2000, 2000)
    ze_lo, _, mu_lo = oracle.z_grid(0.7, 500, 500)
    for name, coeffs, k, c, F in _golden(golden_dir):
        ld, _ = _law(name, coeffs)
        ldp, ldp_lo = ld(mu), ld(mu_lo)
        hi = oracle.direct_flux(k, c, ze, ldp, oracle.istar(ze, ldp))
        lo = oracle.direct_flux(k, c, ze_lo, ldp_lo, oracle.istar(ze_lo, ldp_lo))
        assert abs(hi - F) < 1e-8, (name, k, c, hi - F)
        assert abs(lo - F) < 2e-7
        assert abs(hi - F) <= abs(lo - F) + 1e-10          # error shrinks with resolution


def test_default_istar_vs_analytic():
    """Reading R6: the discretised Istar is O(nz^-2) from the analytic integral."""
    for nz2, tol in [(50, 6e-5), (500, 6e-7)]:
        ze, _, mu = oracle.z_grid(0.7, nz2, nz2)
        got = oracle.istar(ze, truth.quadratic(0.4, 0.2)(mu))
        rel = abs(got / truth.istar_quadratic(0.4, 0.2) - 1)
        assert rel < tol
    ze, _, mu = oracle.z_grid(0.7, 50, 50)
    assert oracle.istar(ze, np.ones(100)) == pytest.approx(math.pi, abs=1e-15)   # uniform: exact


# ---- uniform disc: F = 1 - a(c,k)/pi exactly, through L1 and L2 ----------------
def test_uniform_disc_exact():
    m = oracle.OracleModel()
    ones = np.ones((1, 1, m.nz))
    T, ist = m.build_ld_table(ones)
    assert np.allclose(T, 1.0, rtol=0, atol=1e-14)           # every weight vector sums to 1
    assert ist[0, 0] == pytest.approx(math.pi, abs=1e-15)
    lib = oracle.load()
    rng = np.random.default_rng(5)
    for _ in range(2000):
        k = rng.uniform(0.02, 0.2)
        z = rng.uniform(0, 1.3)
        want = 1 - oracle.lens_area(1, k, z) / math.pi
        assert oracle.direct_flux(k, z, m.ze, ones[0, 0], math.pi) == pytest.approx(want, abs=1e-15)
        got = lib.oracle_flux_from_table(z, k, T.ctypes.data_as(oracle._D), m.nk, m.k0, m.k1, m.ng,
                                         math.pi)
        assert got == pytest.approx(want, abs=2e-15)


# ---- L2 against L0: the error band the paper quotes ------------------------
def test_l2_error_band_against_l0():
    m = oracle.OracleModel()                                    # nz=100, ng=100, nk=50
    lib = oracle.load()
    for ld, k in [(truth.quadratic(0.4, 0.2), 0.1), (truth.quadratic(0.4, 0.2), 0.2),
                  (truth.power2(0.6, 0.7), 0.1)]:
        T, ist = m.build_ld_table(ld(m.mu)[None, None, :])
        zs = np.linspace(0, 1 + k, 41)
        err = []
        for z in zs:
            want = float(truth.flux_radial_mp(k, z, ld, dps=20))
            got = lib.oracle_flux_from_table(z, k, T.ctypes.data_as(oracle._D), m.nk, m.k0, m.k1,
                                             m.ng, ist[0, 0])
            err.append(abs(got - want))
        err = np.array(err)
        assert err.max() < 15e-6 and err.mean() < 2e-6, (k, err.max(), err.mean())
        assert err.max() > 1e-8                                 # it IS an approximation


def test_l2_table_vs_l1_direct_same_resolution():
    """(k,g)-interpolated vs weights at the exact (c,k): 'small reduction in accuracy'."""
    m = oracle.OracleModel()
    lib = oracle.load()
    ld = truth.quadratic(0.4, 0.2)(m.mu)
    T, ist = m.build_ld_table(ld[None, None, :])
    rng = np.random.default_rng(6)
    worst = 0.0
    for _ in range(400):
        k, z = rng.uniform(0.02, 0.2), rng.uniform(0, 1.25)
        a = lib.oracle_flux_from_table(z, k, T.ctypes.data_as(oracle._D), m.nk, m.k0, m.k1, m.ng,
                                       ist[0, 0])
        b = oracle.direct_flux(k, z, m.ze, ld, ist[0, 0])
        worst = max(worst, abs(a - b))
    assert 1e-9 < worst < 2e-5


def test_l2_on_table_nodes_equals_l1():
    """On a (k,g) node both interpolation weights vanish: L2 must reproduce L1 there."""
    m = oracle.OracleModel()
    lib = oracle.load()
    ld = truth.power2(0.5, 0.8)(m.mu)
    T, ist = m.build_ld_table(ld[None, None, :])
    dk, dg = (m.k1 - m.k0) / (m.nk - 1), 1 / (m.ng - 1)
    for ik, ig in [(0, 0), (7, 13), (20, 60), (48, 97), (49, 98), (10, 99)]:
        k = m.k0 + ik * dk
        z = (1.0 if ig == m.ng - 1 else ig * dg) * (1 + k)
        a = lib.oracle_flux_from_table(z, k, T.ctypes.data_as(oracle._D), m.nk, m.k0, m.k1, m.ng,
                                       ist[0, 0])
        b = oracle.direct_flux(k, z, m.ze, ld, ist[0, 0])
        assert a == pytest.approx(b, abs=5e-13), (ik, ig)


def test_table_last_node_is_limb_sample():
    """Reading R5: T[..., ng-1] = ldp[nz-1]."""
    m = oracle.OracleModel(nzin=20, nzlimb=20, ng=30, nk=6)
    ld = truth.quadratic(0.5, 0.1)(m.mu)
    T, _ = m.build_ld_table(ld[None, None, :])
    assert np.all(T[0, 0, :, -1] == ld[-1])


def test_table_is_a_plain_matmul():
    m = oracle.OracleModel(nzin=15, nzlimb=10, ng=17, nk=4, npb=3)
    rng = np.random.default_rng(7)
    ldp = rng.uniform(0.2, 1.0, (5, 3, 25))
    T, ist = m.build_ld_table(ldp)
    assert np.allclose(T, np.einsum("kgj,vbj->vbkg", m.W, ldp), rtol=0, atol=1e-14)
    assert np.allclose(ist, math.pi * (ldp * np.diff(m.ze**2)).sum(-1), rtol=0, atol=1e-14)
    T2, ist2 = m.build_ld_table(ldp, istar_override=np.full((5, 3), 2.5))
    assert np.all(ist2 == 2.5) and np.array_equal(T, T2)
