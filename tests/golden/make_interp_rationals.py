"""Writes tests/golden/interp_weights_next.txt: the rational weights of the 6-, 9- and 10-point operators (readings
S30, S31), derived here from nothing but the definition of the Lagrange interpolant with python's exact `fractions`.
It imports neither oracle/ nor the CUDA package, so the file can pin both. Run: python tests/golden/make_interp_rationals.py"""
import os
from fractions import Fraction as Fr


def lagrange(nodes, x):
    out = []
    for m, xm in enumerate(nodes):
        v = Fr(1)
        for q, xq in enumerate(nodes):
            if q != m:
                v *= (x - xq) / (xm - xq)
        out.append(v)
    return out


ROWS = [  # name, nodes (in node spacings), target
    ("prolong9_p1", [Fr(m) for m in range(-4, 5)], Fr(1, 4)),       # cell-centred 9-point at +1/4 (parity 0: mirror)
    ("restrict10", [Fr(2 * m + 1, 2) for m in range(-5, 5)], Fr(0)),  # fine cells at -9/2..9/2, parent centre at 0
    ("vertex6_mid", [Fr(m) for m in range(-2, 4)], Fr(1, 2)),       # vertex-centred midpoint, 6 points
    ("vertex10_mid", [Fr(m) for m in range(-4, 6)], Fr(1, 2)),      # vertex-centred midpoint, 10 points
]

if __name__ == "__main__":
    here = os.path.dirname(os.path.abspath(__file__))
    with open(os.path.join(here, "interp_weights_next.txt"), "w") as f:
        f.write("# Rational Lagrange weights of the NEXT-3 operators (DESIGN.md S30, S31), written by make_interp_rationals.py\n"
                "# (python fractions; no oracle, no CUDA). name, then numerator/denominator per node, left to right.\n")
        for name, nodes, x in ROWS:
            f.write(name + " " + " ".join(f"{w.numerator}/{w.denominator}" for w in lagrange(nodes, x)) + "\n")
