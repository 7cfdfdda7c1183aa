"""The polynomial tables of the device math (paper_2009_08500_b200/csrc/rr_math.cuh) against their
generator (tests/golden/make_device_poly.py, mpmath only) and against mpmath's atan / sin / cos in
50-digit arithmetic over the ranges the kernels use them on.  CPU only: the literals are parsed
from the source file; nothing here runs CUDA code."""
import os
import re
import sys

import mpmath as mp
import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, os.path.join(ROOT, "tests", "golden"))
import make_device_poly as gen  # noqa: E402

SRC = open(os.path.join(ROOT, "paper_2009_08500_b200", "csrc", "rr_math.cuh")).read()


def parsed(name):
    m = re.search(r"__constant__\s+(double|float)\s+" + name + r"\[(\d+)\]\s*=\s*\{(.*?)\};", SRC, re.S)
    assert m, name
    ty, n, body = m.group(1), int(m.group(2)), m.group(3)
    vals = []
    for tok in body.replace("\n", " ").split(","):
        tok = tok.strip()
        if "/" in tok:                               # "-1.0 / 6.0", "1.0f / 120.0f"
            a, b = (float(x.strip().rstrip("f")) for x in tok.split("/"))
            vals.append(np.float32(np.float32(a) / np.float32(b)) if ty == "float" else a / b)
        else:
            vals.append(np.float32(tok.rstrip("f")) if ty == "float" else float(tok))
    assert len(vals) == n
    return ty, vals


@pytest.mark.parametrize("name", sorted(gen.TABLES))
def test_tables_equal_the_generator(name):
    """Every literal equals the generator's value rounded to the table's type."""
    ty, have = parsed(name)
    want = gen.table(name)
    assert gen.TABLES[name][2] == ty and len(want) == len(have)
    for h, w in zip(have, want):
        w_r = np.float32(float(w)) if ty == "float" else float(w)
        assert h == w_r, (name, h, w_r)


def _horner(coefs, u):
    q = mp.mpf(0)
    for c in reversed(coefs):
        q = q * u + mp.mpf(float(c))
    return q


def _grid(hi, n=1501):
    return [mp.mpf(hi) * i / (n - 1) for i in range(n)]


@pytest.mark.parametrize("name,bound", [("RR_ATAN_D", 3e-18), ("RR_ATAN_F", 1e-9)])
def test_atan_polynomial_error(name, bound):
    """atan t = t + t u Q(u) on |t| <= tan(pi/8), and a little beyond (rr_atan_quadrant's T^2 is
    rounded down, so the reduced argument passes tan(pi/8) by <= 2.1e-7 relative)."""
    mp.mp.dps = 50
    _, coefs = parsed(name)
    worst = mp.mpf(0)
    for t in _grid(mp.tan(mp.pi / 8) * (1 + mp.mpf("1e-6"))):
        u = t * t
        worst = max(worst, abs(t + t * u * _horner(coefs, u) - mp.atan(t)))
    assert worst <= bound, mp.nstr(worst, 5)


@pytest.mark.parametrize("sname,cname,bs,bc", [("RR_SIN_D", "RR_COS_D", 5.2e-17, 7.1e-18),
                                               ("RR_SIN_F", "RR_COS_F", 1.3e-8, 2.9e-9)])
def test_trig_polynomial_error(sname, cname, bs, bc):
    """sin x = x + x^3 S(x^2) (relative error) and cos x - 1 = x^2 C(x^2) (relative to x^2/2) on
    |x| <= 0.5: the truncation bounds stated in rr_math.cuh."""
    mp.mp.dps = 50
    _, cs = parsed(sname)
    _, cc = parsed(cname)
    ws = wc = mp.mpf(0)
    for x in _grid(gen.TRIG_RANGE)[1:]:
        x2 = x * x
        ws = max(ws, abs(x + x * x2 * _horner(cs, x2) - mp.sin(x)) / mp.sin(x))
        wc = max(wc, abs(x2 * _horner(cc, x2) - (mp.cos(x) - 1)) / (x2 / 2))
    assert ws <= bs and wc <= bc, (mp.nstr(ws, 5), mp.nstr(wc, 5))


def test_third_order_seed_corrections():
    """rr_sqrt3 / rr_div3 (rr_math.cuh): one third-order step from a hardware seed of relative error
    |d| <= 2^-20 leaves < 3e-18 (sqrt) and < 1e-18 (reciprocal); checked on the formulas as the file
    states them, in exact arithmetic."""
    mp.mp.dps = 50
    for x in (mp.mpf("0.37"), mp.mpf(2), mp.mpf("1.7e-3"), mp.mpf(977)):
        for d in (mp.mpf(2) ** -20, -mp.mpf(2) ** -20, mp.mpf(2) ** -21, -mp.mpf(2) ** -23):
            y = (1 + d) / mp.sqrt(x)                      # rsqrt seed
            g, h = x * y, y / 2
            r = mp.mpf("0.5") - h * g
            s = g * r * (mp.mpf("1.5") * r + 1) + g
            assert abs(s / mp.sqrt(x) - 1) < 3e-18
            rc = (1 + d) / x                              # rcp seed
            e = 1 - x * rc
            rc3 = rc * (e * e + e) + rc
            assert abs(rc3 * x - 1) < 1e-18


def test_octant_threshold_literal():
    """rr_atan_quadrant's T2: tan^2(pi/8) rounded DOWN to a double with a zero low word (an
    immediate operand); the reduced argument t then passes tan(pi/8) by at most 2.1e-7."""
    mp.mp.dps = 30
    m = re.search(r"\(R\)(0\.1715728\d+)\s*:\s*\(R\)(0\.1715728\d+)f", SRC)
    assert m
    t2d = float(m.group(1))
    exact = mp.tan(mp.pi / 8) ** 2
    assert np.float64(t2d).view(np.uint64) & np.uint64(0xffffffff) == 0
    assert 0 <= mp.sqrt(exact / mp.mpf(t2d)) - 1 < 2.1e-7
    assert abs(mp.mpf(float(np.float32(m.group(2)))) / exact - 1) < 1e-7


@pytest.mark.parametrize("name", ["RR_SIN_F", "RR_COS_F", "RR_ATAN_F"])
def test_packed_tables_repeat_the_scalar_ones(name):
    """The fp32 two-exposures-per-thread path (FFMA2) reads its coefficients as (c, c) pairs from
    RR_*_F2: every pair must hold the scalar table's value twice."""
    _, scalar = parsed(name)
    m = re.search(r"__constant__\s+float2\s+" + name + r"2\[(\d+)\]\s*=\s*\{(.*?)\};", SRC, re.S)
    assert m, name
    pairs = re.findall(r"\{([^{}]+?),([^{}]+?)\}", m.group(2))
    assert len(pairs) == int(m.group(1)) == len(scalar)

    def val(tok):
        tok = tok.strip()
        if "/" in tok:
            a, b = (np.float32(x.strip().rstrip("f")) for x in tok.split("/"))
            return np.float32(a / b)
        return np.float32(tok.rstrip("f"))

    for (a, b), c in zip(pairs, scalar):
        assert val(a) == val(b) == c, (name, a, b, c)


# ---- lens area between the contacts as polynomials (csrc/rr_lens_poly.cuh) ------------------------------
LENS_SRC = open(os.path.join(ROOT, "paper_2009_08500_b200", "csrc", "rr_lens_poly.cuh")).read()


def _lens_table(name):
    m = re.search(name + r"\[(\d+)\]\s*=\s*\{(.*?)\};", LENS_SRC, re.S)
    assert m, name
    vals = [float(t) for t in m.group(2).replace("\n", " ").split(",") if t.strip()]
    assert len(vals) == int(m.group(1))
    return np.array(vals)


def test_lens_tables_equal_the_generator():
    assert LENS_SRC == gen.lens_header()          # the committed header IS the generator's output
    x, xi15, M = gen.lens_tables()
    n = gen.LENS_DEG + 1
    assert np.array_equal(_lens_table("RR_LENS_X"), [float(v) for v in x])
    assert np.array_equal(_lens_table("RR_LENS_XI15"), [float(v) for v in xi15])
    assert np.array_equal(_lens_table("RR_LENS_M").reshape(n, n),
                          [[float(M[j, i]) for i in range(n)] for j in range(n)])


def _lens_exact_mp(k, z):
    k, z = mp.mpf(k), mp.mpf(z)
    if z >= 1 + k:
        return mp.mpf(0)
    if z <= 1 - k:
        return mp.pi * k * k
    a1 = mp.acos((z * z + 1 - k * k) / (2 * z))
    a2 = mp.acos((z * z + k * k - 1) / (2 * z * k))
    return a1 + k * k * a2 - mp.sqrt((-z + 1 + k) * (z + 1 - k) * (z - 1 + k) * (z + 1 + k)) / 2


@pytest.mark.parametrize("k", [0.01, 0.05, 0.1, 0.2, 0.3, 0.32])
def test_lens_polynomial_reproduces_the_area(k):
    """The pipeline of rr_lens_fit + rr_deficit restated in float64 (exact area at the nodes
    by the half-angle form, node values -> monomial coefficients through RR_LENS_M, Horner in
    w = 4x - 1, a = pi k^2 - x^(3/2) g0 or y^(3/2) g1) against the textbook two-sector-minus-kite area
    in 40-digit arithmetic, between the contacts and right at them: <= 2.5e-13."""
    mp.mp.dps = 40
    X, XI15 = _lens_table("RR_LENS_X"), _lens_table("RR_LENS_XI15")
    n = X.size
    M = _lens_table("RR_LENS_M").reshape(n, n)
    full = np.pi * k * k

    def area64(z):                                  # float64, as the device states it
        A, B, C, D = 1 + k - z, z + 1 - k, z - 1 + k, z + 1 + k
        kite = np.sqrt(abs(A * B) * abs(C * D))
        return 2 * np.arctan2(kite, B * D) + 2 * k * k * np.arctan2(kite, abs(C * D)) - kite / 2

    g0 = np.array([(full - area64(1 - k + 2 * k * x)) for x in X]) * XI15
    g1 = np.array([area64(1 + k - 2 * k * x) for x in X]) * XI15
    a0, a1 = M @ g0, M @ g1
    xs = np.concatenate([np.linspace(0.0, 1.0, 801), 10.0 ** np.linspace(-14, -3, 40),
                         1 - 10.0 ** np.linspace(-14, -3, 40)])
    worst = 0.0
    for x in xs:
        z = 1 - k + 2 * k * x
        lo = x <= 0.5
        xx = abs(x if lo else 1 - x)
        w = 4 * xx - 1
        p = 0.0
        for c in (a0 if lo else a1)[::-1]:
            p = p * w + c
        t = xx * np.sqrt(xx)
        ap = full - t * p if lo else t * p
        worst = max(worst, abs(ap - float(_lens_exact_mp(k, z))))
    assert worst <= 2.5e-13, worst


def test_orbit_polynomial_reproduces_z2_over_a_transit_window():
    """rr_zpoly_fit's construction restated in float64 on the CPU: z^2 of an eccentric orbit over
    each half of its transit window, interpolated at the 13 Chebyshev nodes and converted to
    monomials with RR_LENS_M, against the oracle's separation (a Newton solve per point): <= 5e-12 in
    z^2 for config 4's eccentric parameter vectors whenever the kernel's tail test (|c12| + |c11| <=
    1e-12) passes, which it does for most of them."""
    import oracle
    import workloads
    X = _lens_table("RR_LENS_X")
    n = X.size
    M = _lens_table("RR_LENS_M").reshape(n, n)
    wl = workloads.make_workload(4, npv=60, npt=10)
    passed = worst = 0
    total = 0
    for row in wl.pv:
        k, t0, p, e = row[0], row[1], row[2], row[5]
        if e == 0.0:
            continue
        ts = t0 + np.linspace(-0.25 * p, 0.25 * p, 1601)
        zz = np.array([z if front else 99.0 for z, front in (oracle.separation(t, *row[1:]) for t in ts)])
        i0 = int(np.argmin(np.abs(ts - t0)))
        if not zz[i0] < 1 + k:
            continue
        ia = ib = i0
        while ia > 0 and zz[ia - 1] < 1 + k:
            ia -= 1
        while ib < ts.size - 1 and zz[ib + 1] < 1 + k:
            ib += 1
        c, h = 0.5 * (ts[ia] + ts[ib]), 0.5 * (ts[ib] - ts[ia]) * 1.03 + 1e-6
        total += 1
        tail = err = 0.0
        for sgn in (-1.0, 1.0):
            g = np.array([oracle.separation(c + sgn * h * 2 * x, *row[1:])[0] ** 2 for x in X])
            a = M @ g
            tail += abs(a[12]) / 2048 + abs(a[11]) / 1024
            for tp in np.linspace(0, 1, 33):
                w = 2 * tp - 1
                q = 0.0
                for cj in a[::-1]:
                    q = q * w + cj
                err = max(err, abs(q - oracle.separation(c + sgn * h * tp, *row[1:])[0] ** 2))
        if tail <= 1e-12:
            passed += 1
            worst = max(worst, err)
    assert total >= 20 and passed >= 0.7 * total, (passed, total)
    assert worst <= 5e-12, worst
