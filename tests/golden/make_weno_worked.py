"""Writes weno_worked.json: worked WENO stencils evaluated in EXACT rational arithmetic.

This is a hand calculation, not an output of any implementation: it evaluates the classical
Jiang-Shu fifth-order / third-order WENO face value (Shu 1997, the reconstruction the paper
cites at PAPER.md:244 for its advection scheme) with python Fractions on integer
stencils, eps = 10^-6 exactly.  It imports neither oracle/ nor the CUDA package.

    python tests/golden/make_weno_worked.py
"""
import json
import os
from fractions import Fraction as F

EPS = F(1, 10 ** 6)


def worked(cells, order, vel):
    c = [F(x) for x in cells]
    # upwind-biased stencil: q0 is the upwind cell of the interface between cells[2] and cells[3]
    q = c[0:5] if vel > 0 else c[::-1][0:5]
    qm2, qm1, q0, q1, q2 = q
    if order == 3:
        p = [(2 * qm2 - 7 * qm1 + 11 * q0) / 6, (-qm1 + 5 * q0 + 2 * q1) / 6, (2 * q0 + 5 * q1 - q2) / 6]
        b = [F(13, 12) * (qm2 - 2 * qm1 + q0) ** 2 + F(1, 4) * (qm2 - 4 * qm1 + 3 * q0) ** 2,
             F(13, 12) * (qm1 - 2 * q0 + q1) ** 2 + F(1, 4) * (qm1 - q1) ** 2,
             F(13, 12) * (q0 - 2 * q1 + q2) ** 2 + F(1, 4) * (3 * q0 - 4 * q1 + q2) ** 2]
        d = [F(1, 10), F(6, 10), F(3, 10)]
    else:
        p = [(-qm1 + 3 * q0) / 2, (q0 + q1) / 2]
        b = [(q0 - qm1) ** 2, (q1 - q0) ** 2]
        d = [F(1, 3), F(2, 3)]
    a = [dd / (EPS + bb) ** 2 for dd, bb in zip(d, b)]
    return sum(aa * pp for aa, pp in zip(a, p)) / sum(a)


CASES = [([0, 0, 0, 1, 1, 1], 3, 1), ([0, 0, 0, 1, 1, 1], 3, -1), ([1, 2, 4, 8, 16, 32], 3, 1),
         ([1, 2, 4, 8, 16, 32], 3, -1), ([3, -1, 4, 1, -5, 9], 3, 1), ([3, -1, 4, 1, -5, 9], 2, -1),
         ([0, 1, 3, 4, 9, 2], 2, 1)]

if __name__ == "__main__":
    out = {"source": "exact rational evaluation of Jiang-Shu WENO (Shu 1997; PAPER.md:244, 86)", "cases": []}
    for cells, order, vel in CASES:
        v = worked(cells, order, vel)
        out["cases"].append({"cells": cells, "order": order, "vel": vel, "num": str(v.numerator),
                             "den": str(v.denominator), "approx": float(v)})
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "weno_worked.json"), "w") as fh:
        json.dump(out, fh, indent=1)
