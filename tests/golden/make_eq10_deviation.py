"""Writes tests/golden/eq10_deviation.txt: eq.(10)/quadrature(eq.(9)) - 1 on a grid.

Calls only oracle/ (fp64 CPU) and tests/quadrature.py. Run: python tests/golden/make_eq10_deviation.py
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
sys.path.insert(0, os.path.dirname(HERE))

from oracle import ref  # noqa: E402
from quadrature import sphere_integral_of_G  # noqa: E402

GRID = [(3.0, 1.0, 0.0), (3.0, 0.0, 2.0), (1.0, 0.0, 3.0), (3.0, 1.0, 2.0), (3.0, 2.0, 5.0),
        (1.0, 0.5, 4.0), (0.5, 4.0, 6.0), (7.4, 19.0, 8.0), (55.0, 1.7, 8.0), (148.0, 0.01, 8.0)]

with open(os.path.join(HERE, "eq10_deviation.txt"), "w") as f:
    f.write("# eq.(10) as printed (PAPER.md:209-211) divided by Gauss-Legendre x trapezoid quadrature of\n"
            "# eq.(9) (PAPER.md:202-205), minus 1; phi = 0. Exact (<=1e-9) iff a = 0 or k = 0 (reading R2).\n"
            "# lambda a k deviation\n")
    for lam, a, k in GRID:
        dev = 1.0 / sphere_integral_of_G(ref, lam, a, k, 0.0, 1) - 1.0
        f.write(f"{lam:g} {a:g} {k:g} {dev:.6e}\n")
