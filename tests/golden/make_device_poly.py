"""Generator of the polynomial coefficients in paper_2009_08500_b200/csrc/rr_math.cuh (mpmath only).

The device math of the hot path evaluates, on the reduced ranges the transit geometry guarantees
(DESIGN.md s6):
  atan t = t + t u Q(u), u = t^2, |t| <= T = tan(pi/8):  Q = the polynomial of degree n-1 that
      interpolates q(u) = (atan(sqrt u)/sqrt u - 1)/u at u_j = t_j^2, t_j the n positive roots of
      the Chebyshev polynomial of degree 2n+1 scaled to [-T, T] (the interpolation nodes of the odd
      function atan on the symmetric interval; n = 11 in fp64 -> RR_ATAN_D, n = 5 in fp32 ->
      RR_ATAN_F);
  sin x = x + x^3 (S0 + S1 x^2 + ...), cos x - 1 = x^2 (C0 + C1 x^2 + ...), |x| <= 0.5: Taylor
      coefficients (-1)^(n+1)/(2n+3)! and (-1)^(n+1)/(2n+2)!  (RR_SIN_D/F, RR_COS_D/F).

`python tests/golden/make_device_poly.py` prints the tables as C initialisers.  The CPU test
tests/test_device_poly.py regenerates them, compares them with the literals parsed from rr_math.cuh
and measures the polynomials' errors in 50-digit arithmetic.  No value comes from the CUDA path.
"""
import mpmath as mp

mp.mp.dps = 60

ATAN_RANGE = mp.tan(mp.pi / 8) ** 2          # u = t^2 in [0, tan^2(pi/8)]
TRIG_RANGE = mp.mpf("0.5")


def atan_q(u):
    """q(u) = (atan(sqrt u)/sqrt u - 1)/u, with its series at u -> 0."""
    u = mp.mpf(u)
    if u < mp.mpf("1e-20"):
        return -mp.mpf(1) / 3 + u / 5
    r = mp.sqrt(u)
    return (mp.atan(r) / r - 1) / u


def atan_coefficients(n):
    """Monomial coefficients (lowest first) of the interpolant Q of q with n coefficients."""
    T = mp.tan(mp.pi / 8)
    nodes = [(T * mp.cos((2 * j + 1) * mp.pi / (2 * (2 * n + 1)))) ** 2 for j in range(n)]
    V = mp.matrix(n, n)
    rhs = mp.matrix(n, 1)
    for i, u in enumerate(nodes):
        for j in range(n):
            V[i, j] = u ** j
        rhs[i] = atan_q(u)
    sol = mp.lu_solve(V, rhs)
    return [sol[j] for j in range(n)]


def sin_coefficients(n):
    return [(-1) ** (i + 1) / mp.factorial(2 * i + 3) for i in range(n)]


def cos_coefficients(n):
    return [(-1) ** (i + 1) / mp.factorial(2 * i + 2) for i in range(n)]


TABLES = {           # name in rr_math.cuh -> (generator, entries, float type)
    "RR_SIN_D": (sin_coefficients, 6, "double"), "RR_COS_D": (cos_coefficients, 7, "double"),
    "RR_SIN_F": (sin_coefficients, 3, "float"), "RR_COS_F": (cos_coefficients, 4, "float"),
    "RR_ATAN_D": (atan_coefficients, 11, "double"), "RR_ATAN_F": (atan_coefficients, 5, "float"),
}


def table(name):
    gen, n, _ = TABLES[name]
    with mp.workdps(60):
        return gen(n)


def literal(c, ty):
    """The shortest decimal string that rounds to the same double / float."""
    if ty == "double":
        return repr(float(c))
    import numpy as np
    return f"{float(np.float32(float(c))):.9e}f"


if __name__ == "__main__":
    for name, (_, n, ty) in TABLES.items():
        vals = ", ".join(literal(c, ty) for c in table(name))
        print(f"__constant__ {ty} {name}[{n}] = {{{vals}}};")


# ---- lens area on the ingress / egress interval as two polynomials (rr_lens_poly.cuh) -----------------
# For a planet of radius k at separation z between the contacts, x = (z - (1-k)) / (2k) in (0, 1):
#   near the second contact  a(z) = pi k^2 - x^(3/2) g0(x),      x  in [0, 1/2]
#   near the first contact   a(z) =         y^(3/2) g1(y),  y = 1 - x in [0, 1/2]
# with g0, g1 analytic (the area is an analytic function of the angle theta, x = sin^2(theta/2)), so
# they are interpolated by polynomials of degree LENS_DEG at the Chebyshev nodes of [0, 1/2].  The
# kernel evaluates the exact area at those nodes once per (parameter vector, radius ratio) and turns
# the node values into monomial coefficients in w = 4x - 1 with the matrix LENS_M below; every
# ingress / egress sub-sample then costs one square root and a Horner chain instead of two
# arctangents.  Tables: nodes x_i, x_i^(-3/2), and M = (Chebyshev -> monomial) . (values -> Chebyshev).
LENS_DEG = 12


def lens_tables(deg=LENS_DEG):
    with mp.workdps(60):                       # whatever precision the caller has set
        return _lens_tables(deg)


def _lens_tables(deg):
    n = deg + 1
    t = [mp.cos((2 * i + 1) * mp.pi / (2 * n)) for i in range(n)]          # nodes in [-1, 1]
    x = [(ti + 1) / 4 for ti in t]                                         # nodes in [0, 1/2]
    xi15 = [xi ** mp.mpf("-1.5") for xi in x]
    C = mp.matrix(n, n)                                                    # values -> Chebyshev
    for j in range(n):
        for i in range(n):
            C[j, i] = (1 if j == 0 else 2) * mp.chebyt(j, t[i]) / n
    P = mp.matrix(n, n)                                                    # P[j, m]: coefficient of w^m in T_j
    P[0, 0] = 1
    if n > 1:
        P[1, 1] = 1
    for j in range(2, n):
        for m in range(n):
            P[j, m] = (2 * P[j - 1, m - 1] if m > 0 else 0) - P[j - 2, m]
    M = P.T * C                                                            # monomial[m] = sum_i M[m, i] g_i
    for m in range(n):                                                     # entries that are exactly 0
        for i in range(n):
            if abs(M[m, i]) < mp.mpf("1e-40"):
                M[m, i] = mp.mpf(0)
    return x, xi15, M


def lens_header(deg=LENS_DEG):
    x, xi15, M = lens_tables(deg)
    n = deg + 1
    out = ["// rr_lens_poly.cuh - written by tests/golden/make_device_poly.py (mpmath); do not edit.",
           "// Tables of the polynomial form of the lens area between the contacts (see the generator).",
           "#pragma once",
           f"#define RR_LENS_DEG {deg}",
           f"#define RR_LENS_N {n}",
           f"__constant__ double RR_LENS_X[{n}] = {{" + ", ".join(repr(float(v)) for v in x) + "};",
           f"__constant__ double RR_LENS_XI15[{n}] = {{" + ", ".join(repr(float(v)) for v in xi15) + "};",
           f"__device__ const double RR_LENS_M[{n * n}] = {{"]
    for m in range(n):
        out.append("    " + ", ".join(repr(float(M[m, i])) for i in range(n)) + ",")
    out.append("};")
    return "\n".join(out) + "\n"
