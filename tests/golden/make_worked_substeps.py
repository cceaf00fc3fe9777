"""Writes tests/golden/worked_substeps.txt: the stage values of Alg. 1 for a few
hand-picked inputs, worked in 50-digit arithmetic with mpmath.  Calls neither oracle/ nor the CUDA path:
the numbers are the paper's algorithm evaluated line by line, with the drift a(x) = -V'(x) + F - lambda*zeta
of DESIGN.md R6 and V(x) = A1 sin(2 pi x) + A2 sin(4 pi x).  W1/W2 are the worked examples quoted in
SURVEY.md section 8(c); W3 adds noise and bias together.
"""
import os

import mpmath as mp

mp.mp.dps = 50
CASES = [  # A1, A2, F, D, lambda, zeta, x_n, h, g
    ("W1", 1.0, 0.25, 0.1, 0.05, 0.0, 0.0, 0.1, 1e-3, 0.5),
    ("W2", 1.0, 0.25, 0.0, 0.0, 2.0, 0.3, 0.9, 2.5e-4, 0.0),
    ("W3", 1.0, 0.25, 0.0, 0.01, 2.0, 0.3, 0.42, 7.5e-4, -1.25),
]


def drift(A1, A2, F, lam, zeta, x):
    return -(2 * mp.pi * A1 * mp.cos(2 * mp.pi * x) + 4 * mp.pi * A2 * mp.cos(4 * mp.pi * x)) + F - lam * zeta


def main():
    out = ["# Alg. 1 (PAPER.md:221-235) stage values, 50-digit mpmath; written by make_worked_substeps.py",
           "# A1 A2 F D lambda zeta x_n h g | F1 xbar1 F2 xbar2 F2' x_{n+1}"]
    for name, A1, A2, F, D, lam, zeta, x, h, g in CASES:
        a = [mp.mpf(repr(v)) for v in (A1, A2, F, D, lam, zeta, x, h, g)]
        A1m, A2m, Fm, Dm, lm, zm, xm, hm, gm = a
        dxi = mp.sqrt(2 * Dm * hm) * gm
        F1 = drift(A1m, A2m, Fm, lm, zm, xm)
        xb1 = xm + F1 * hm + dxi
        F2 = drift(A1m, A2m, Fm, lm, zm, xb1)
        xb2 = xm + (F1 + F2) * hm / 2 + dxi
        F2c = drift(A1m, A2m, Fm, lm, zm, xb2)
        xn = xm + (F1 + F2c) * hm / 2 + dxi
        out.append("  ".join(repr(v) for v in (A1, A2, F, D, lam, zeta, x, h, g)) + "  "
                   + "  ".join(mp.nstr(v, 20) for v in (F1, xb1, F2, xb2, F2c, xn)) + "  # " + name)
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "worked_substeps.txt"), "w") as f:
        f.write("\n".join(out) + "\n")


if __name__ == "__main__":
    main()
