"""Writes tests/golden/l0_truth.txt: Eq. (2) evaluated by 30-digit mpmath
quadrature (oracle/truth.py::flux_radial_mp) - calls only oracle/.  Run: python tests/golden/make_l0_truth.py
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import truth  # noqa: E402

CASES = [
    ("quadratic", (0.4, 0.2), [(0.1, 0.0), (0.1, 0.3), (0.1, 0.9), (0.1, 0.95), (0.1, 1.0),
                               (0.1, 1.05), (0.2, 1.1), (0.3, 1.0), (0.05, 0.5), (0.2, 0.8),
                               (0.2, 0.0)]),
    ("power2", (0.6, 0.7), [(0.1, 0.0), (0.1, 0.95), (0.3, 1.0), (0.15, 0.6)]),
    ("poly", (-0.4, -0.1, -0.05, -0.02), [(0.1, 0.2), (0.1, 0.97), (0.2, 1.05)]),
]

if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "l0_truth.txt")
    with open(out, "w") as f:
        f.write("# L0 truth: F = 1 - int_Ap I dA / (2 pi int_0^1 z I dz), Eq. (1)-(4), PAPER.md:43-55\n")
        f.write("# written by tests/golden/make_l0_truth.py (mpmath, 30 digits); no value from the CUDA path\n")
        f.write("# law coeffs... | k c | flux\n")
        for law, coeffs, pts in CASES:
            ld = {"quadratic": lambda: truth.quadratic(*coeffs),
                  "power2": lambda: truth.power2(*coeffs),
                  "poly": lambda: truth.poly(coeffs)}[law]()
            for k, c in pts:
                F = truth.flux_radial_mp(k, c, ld, dps=30)
                f.write(f"{law} {' '.join(repr(x) for x in coeffs)} | {k!r} {c!r} | {str(F)[:22]}\n")
    print(open(out).read())
