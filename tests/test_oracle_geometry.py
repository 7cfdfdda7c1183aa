"""Pins for the oracle's geometry (grid, lens area, weights) against what the mathematics fixes.
CPU only.  Citations: PAPER.md lines; readings R* in DESIGN.md section 3."""
import math

import mpmath as mp
import numpy as np
import pytest

import oracle
from oracle import truth


# ---- grid ------------------------------------------------------------------------
@pytest.mark.parametrize("zcut,nzin,nzlimb", [(0.7, 50, 50), (0.7, 100, 100), (0.9, 7, 13)])
def test_grid_structure(zcut, nzin, nzlimb):
    ze, zm, mu = oracle.z_grid(zcut, nzin, nzlimb)
    nz = nzin + nzlimb
    assert ze.shape == (nz + 1,) and zm.shape == (nz,) and mu.shape == (nz,)
    assert ze[0] == 0.0 and ze[nz] == 1.0 and abs(ze[nzin] - zcut) < 1e-15
    assert np.all(np.diff(ze) > 0)
    # inner region: constant dz; outer region: constant dmu ("constant in mu")
    assert np.allclose(np.diff(ze[: nzin + 1]), zcut / nzin, rtol=0, atol=1e-15)
    mue = np.sqrt(np.clip(1.0 - ze[nzin:] ** 2, 0, None))
    assert np.allclose(np.diff(mue), -math.sqrt(1 - zcut**2) / nzlimb, rtol=0, atol=1e-13)
    # means and mu = sqrt(1 - zm^2)
    assert np.array_equal(zm, 0.5 * (ze[:-1] + ze[1:]))
    assert np.allclose(mu, np.sqrt(1 - zm * zm), rtol=0, atol=0)


# ---- lens area -------------------------------------------------------------------
def test_lens_limits_and_continuity():
    for k in (0.01, 0.1, 0.3, 0.7):
        assert oracle.lens_area(1, k, 0.0) == math.pi * k * k
        assert oracle.lens_area(1, k, 1 - k) == pytest.approx(math.pi * k * k, abs=1e-15)
        assert oracle.lens_area(1, k, 0.5 * (1 - k)) == math.pi * k * k
        assert oracle.lens_area(1, k, 1 + k) == 0.0
        assert oracle.lens_area(1, k, 1 + k + 1e-9) == 0.0
        # continuity across both contacts: the area changes like delta^(3/2)
        assert abs(oracle.lens_area(1, k, 1 - k + 1e-12) - math.pi * k * k) < 1e-14
        assert 0 <= oracle.lens_area(1, k, 1 + k - 1e-12) < 1e-14
    # planet larger than the star (r2 > r1): full coverage of the smaller disc
    assert oracle.lens_area(0.2, 0.5, 0.1) == pytest.approx(math.pi * 0.04, abs=1e-16)


def test_lens_symmetry_and_monotonic():
    rng = np.random.default_rng(1)
    for _ in range(200):
        r1, r2 = rng.uniform(0.05, 1.0, 2)
        d = rng.uniform(0, r1 + r2)
        a, b = oracle.lens_area(r1, r2, d), oracle.lens_area(r2, r1, d)
        assert a == pytest.approx(b, abs=1e-15)
        assert 0 <= a <= math.pi * min(r1, r2) ** 2 + 1e-15
    ds = np.linspace(0, 1.3, 400)
    a = np.array([oracle.lens_area(1, 0.3, d) for d in ds])
    assert np.all(np.diff(a) <= 1e-16)


def test_lens_equal_circles_closed_form():
    # two unit circles at distance d: 2 acos(d/2) - (d/2) sqrt(4 - d^2)   (textbook special case)
    for d in (0.1, 0.5, 1.0, 1.5, 1.99):
        want = 2 * math.acos(d / 2) - 0.5 * d * math.sqrt(4 - d * d)
        assert oracle.lens_area(1, 1, d) == pytest.approx(want, abs=2e-15)
    # orthogonal-ish known value: r1=r2=1, d=sqrt(2): pi/2 - 1
    assert oracle.lens_area(1, 1, math.sqrt(2)) == pytest.approx(math.pi / 2 - 1, abs=2e-15)


def test_lens_vs_acos_form_away_from_contacts():
    rng = np.random.default_rng(2)
    worst = 0.0
    for _ in range(20000):
        k = rng.uniform(0.01, 0.5)
        c = rng.uniform(1 - k + 1e-4, 1 + k - 1e-4)
        worst = max(worst, abs(oracle.lens_area(1, k, c) - oracle.lens_area_acos(1, k, c)))
    assert worst < 1e-13


def test_lens_vs_independent_quadrature():
    """a(c,k) = pi (1 - F_uniform): the 1-D radial arc-length integral with I = 1 (mpmath, 30
    digits) never touches the lens formula.  Includes points 1e-7 from the contacts, where the
    textbook acos form is already wrong in the 10th digit of the angle."""
    one = lambda mu: mp.mpf(1)  # noqa: E731
    for k, c in [(0.1, 0.95), (0.1, 1.05), (0.3, 1.2), (0.2, 0.8000001), (0.2, 1.1999999),
                 (0.05, 1.0), (0.5, 0.6), (0.01, 1.005)]:
        want = mp.pi * (1 - truth.flux_radial_mp(k, c, one, dps=30))
        assert abs(oracle.lens_area(1, k, c) - float(want)) < 2e-15, (k, c)


def test_lens_two_radius_general():
    """A(r; c, k) for an annulus edge r < 1 by scaling: lens(r, k, c) = r^2 lens(1, k/r, c/r)."""
    rng = np.random.default_rng(3)
    for _ in range(500):
        r = rng.uniform(0.1, 1.0)
        k = rng.uniform(0.01, 0.3)
        c = rng.uniform(0, 1.3)
        assert oracle.lens_area(r, k, c) == pytest.approx(r * r * oracle.lens_area(1, k / r, c / r),
                                                          abs=1e-15)


# ---- weights (Fig. 1) ---------------------------------------------------------------------
def test_weights_sum_support_sign():
    ze, _, _ = oracle.z_grid(0.7, 50, 50)
    rng = np.random.default_rng(4)
    for _ in range(300):
        k = rng.uniform(0.01, 0.3)
        c = rng.uniform(0, 1 + k - 1e-6)
        w = oracle.weights(c, k, ze)
        assert abs(w.sum() - 1) < 1e-13
        assert w.min() > -1e-13 / max(oracle.lens_area(1, k, c), 1e-3)
        outside = (ze[1:] <= c - k) | (ze[:-1] >= c + k)       # annuli the planet does not touch
        assert np.all(np.abs(w[outside]) < 1e-13)


def test_weights_centred_closed_form():
    """c = 0: the planet covers annulus j by pi (min(ze[j+1],k)^2 - min(ze[j],k)^2)."""
    ze, _, _ = oracle.z_grid(0.7, 50, 50)
    for k in (0.05, 0.1, 0.33):
        w = oracle.weights(0.0, k, ze)
        want = (np.minimum(ze[1:], k) ** 2 - np.minimum(ze[:-1], k) ** 2) / k**2
        assert np.allclose(w, want, rtol=0, atol=1e-15)


def test_weights_limit_at_last_contact():
    """Reading R5: at g = 1 (c = 1+k, a = 0) all the weight sits in the outermost annulus, which is
    the limit of w as c -> 1+k from below."""
    ze, _, _ = oracle.z_grid(0.7, 50, 50)
    w1 = oracle.weights(1.1, 0.1, ze)
    assert w1[-1] == 1.0 and np.all(w1[:-1] == 0)
    wlim = oracle.weights(1.1 - 1e-7, 0.1, ze)
    assert abs(wlim[-1] - 1) < 1e-6 and np.all(np.abs(wlim[:-1]) < 1e-6)


def test_weight_tensor_rows_are_weight_vectors():
    m = oracle.OracleModel(nzin=10, nzlimb=10, ng=12, nk=5, k0=0.05, k1=0.25)
    assert m.W.shape == (5, 12, 20)
    assert np.allclose(m.W.sum(axis=2), 1.0, atol=1e-13)
    dk, dg = (0.25 - 0.05) / 4, 1 / 11
    for ik, ig in [(0, 0), (2, 5), (4, 10), (3, 11)]:
        k = 0.05 + ik * dk
        g = 1.0 if ig == 11 else ig * dg
        assert np.array_equal(m.W[ik, ig], oracle.weights(g * (1 + k), k, m.ze))
