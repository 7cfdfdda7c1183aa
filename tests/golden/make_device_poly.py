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
