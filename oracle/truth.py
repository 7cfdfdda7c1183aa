"""L0 truth - TEST INFRASTRUCTURE.  The transit signal straight from its definition, Eq. (1)-(4)
(PAPER.md:43-55):   F = 1 - (int_{Ap} I(z) dA) / (2 pi int_0^1 z I(z) dz),
computed two independent ways, neither using the lens-area formula, the annulus weights or any
table of the model:

* ``flux_polar_bruteforce``: midpoint rule on a polar grid centred on the PLANET, integrand
  I(z) [z < 1] (numpy; the "brute-force 2-D numerical integration of Eq. (2)" of the north star);
* ``flux_radial_mp``: 1-D integral over stellar radius r of I(r) times the arc length of the circle
  of radius r inside the planet's disc, by mpmath quadrature at ``dps`` digits (Kreidberg 2015's
  reduction).

LD laws are given as callables of mu = sqrt(1 - z^2) (PAPER.md footnote 2, :71).
"""
from __future__ import annotations

import mpmath as mp
import numpy as np


# ---- limb-darkening laws and their analytic disc integrals -------------------
def quadratic(u1, u2):
    return lambda mu: 1 - u1 * (1 - mu) - u2 * (1 - mu) ** 2


def power2(c, alpha):
    return lambda mu: 1 - c * (1 - mu ** alpha)


def poly(coeffs):
    """I(mu) = 1 + sum_{n>=1} c_n (1-mu)^n, coeffs = [c_1, c_2, ...]."""
    return lambda mu: 1 + sum(cn * (1 - mu) ** (n + 1) for n, cn in enumerate(coeffs))


def istar_quadratic(u1, u2):
    """2 pi int_0^1 z I dz = 2 pi int_0^1 mu I dmu = pi (1 - u1/3 - u2/6)."""
    return np.pi * (1 - u1 / 3 - u2 / 6)


def istar_power2(c, alpha):
    return np.pi * (1 - c * alpha / (alpha + 2))


def istar_poly(coeffs):
    """int_0^1 2 mu (1-mu)^n dmu = 2/((n+1)(n+2))."""
    return np.pi * (1 + sum(2 * cn / ((n + 2) * (n + 3)) for n, cn in enumerate(coeffs)))


# The named laws of PAPER.md:143-156 (the paper lists the names and cites their sources; forms are
# the textbook ones) as callables of mu and their closed-form disc integrals, pinned against
# mpmath quadrature in tests/test_oracle_direct.py.  name -> (callable factory, Istar or None).
def law(name, c):
    c = [float(x) for x in c]
    if name == "uniform":
        return (lambda mu: 1 + 0 * mu), np.pi
    if name == "linear":
        return (lambda mu: 1 - c[0] * (1 - mu)), np.pi * (1 - c[0] / 3)
    if name == "quadratic":
        return quadratic(*c), istar_quadratic(*c)
    if name == "quadratic-tri":                       # Kipping (2013)
        u1, u2 = 2 * c[0] ** 0.5 * c[1], c[0] ** 0.5 * (1 - 2 * c[1])
        return quadratic(u1, u2), istar_quadratic(u1, u2)
    if name == "general":                             # 1 - sum_n c_n (1 - mu^n), n = 1..N
        return (lambda mu: 1 - sum(cn * (1 - mu ** (n + 1)) for n, cn in enumerate(c)),
                np.pi * (1 - sum(cn * (n + 1) / (n + 3) for n, cn in enumerate(c))))
    if name == "nonlinear":                           # Claret (2000), four coefficients
        return (lambda mu: 1 - sum(cn * (1 - mu ** ((n + 1) / 2)) for n, cn in enumerate(c)),
                np.pi * (1 - sum(cn * (n + 1) / (n + 5) for n, cn in enumerate(c))))
    if name == "logarithmic":
        def f(mu):
            if isinstance(mu, np.ndarray):
                safe = np.where(mu > 0, mu, 1.0)
                return 1 - c[0] * (1 - mu) - c[1] * np.where(mu > 0, mu * np.log(safe), 0.0)
            return 1 - c[0] * (1 - mu) - c[1] * (mu * mp.log(mu) if mu > 0 else 0)
        return f, np.pi * (1 - c[0] / 3 + 2 * c[1] / 9)
    if name == "exponential":
        def f(mu):
            e = np.exp(mu) if isinstance(mu, np.ndarray) else mp.exp(mu)
            return 1 - c[0] * (1 - mu) - c[1] / (1 - e)
        return f, None
    if name == "power-2":
        return power2(*c), istar_power2(*c)
    if name == "power-2-pm":                          # Maxted (2018)
        cc = 1 - c[0] + c[1]
        al = float(np.log2(cc / c[1]))
        return power2(cc, al), istar_power2(cc, al)
    raise ValueError(name)


def istar_mp(ld, dps=30):
    with mp.workdps(dps):
        return 2 * mp.pi * mp.quad(lambda mu: mu * ld(mu), [0, 1])


# ---- truth 1: brute force on a planet-centred polar grid ----------------------------------------
def flux_polar_bruteforce(k, c, ld, istar_value, nrho=4000, ntheta=4000):
    """Midpoint rule over rho in [0,k], theta in [0,pi] (upper half disc, doubled by symmetry)."""
    rho = (np.arange(nrho) + 0.5) * (k / nrho)
    theta = (np.arange(ntheta) + 0.5) * (np.pi / ntheta)
    total = 0.0
    ct = np.cos(theta)
    for r in rho:                                    # row by row keeps memory small
        z2 = c * c + r * r + 2.0 * c * r * ct
        inside = z2 < 1.0
        mu = np.sqrt(np.where(inside, 1.0 - z2, 0.0))
        total += r * np.sum(np.where(inside, ld(mu), 0.0))
    occluded = 2.0 * total * (k / nrho) * (np.pi / ntheta)
    return 1.0 - occluded / istar_value


# ---- truth 2: 1-D radial integral at high precision ----------------------------------------------
def flux_radial_mp(k, c, ld, dps=30):
    """occluded = int I(r) * 2 r theta(r) dr, theta(r) = half-angle of the arc of radius r (about the
    star's centre) lying inside the planet: pi if r <= k - c, acos((r^2+c^2-k^2)/(2 r c)) if
    |c-k| < r < c+k, else 0.  Limits clipped to the stellar disc r <= 1."""
    with mp.workdps(dps):
        k, c = mp.mpf(k), mp.mpf(c)
        ist = 2 * mp.pi * mp.quad(lambda mu: mu * ld(mu), [0, 1])
        if c >= 1 + k:
            return mp.mpf(1)

        def I_r(r):
            return ld(mp.sqrt(1 - r * r))

        occ = mp.mpf(0)
        if k > c:                                     # stellar centre under the planet
            hi = min(k - c, mp.mpf(1))
            occ += mp.quad(lambda r: 2 * mp.pi * r * I_r(r), [0, hi])
        lo, hi = abs(c - k), min(c + k, mp.mpf(1))
        if hi > lo and c > 0:
            def f(r):
                x = (r * r + c * c - k * k) / (2 * r * c)
                x = max(min(x, mp.mpf(1)), mp.mpf(-1))
                return 2 * r * mp.acos(x) * I_r(r)
            mid = (lo + hi) / 2
            occ += mp.quad(f, [lo, mid, hi])
        return 1 - occ / ist
