"""Writes wenoz_worked.json: worked WENO-Z stencils evaluated in EXACT rational arithmetic.

A hand calculation, not an output of any implementation: the WENO-Z face value (Borges, Carmona, Costa & Don 2008: the
weights alpha_s = d_s (1 + (tau / (beta_s + eps))^2) with tau = |beta_0 - beta_2| on the Jiang-Shu candidates and smoothness
indicators; the same construction with tau = |beta_0 - beta_1| for the third-order member) — one member of the WENO family
the paper's "adaptive-order scheme based on WENO reconstructions" belongs to (refs at PAPER.md:244-245; the
reading is DESIGN.md §3.15) — with python Fractions on integer stencils, eps = 10^-6 exactly.  Imports neither oracle/ nor
the CUDA package.

    python tests/golden/make_wenoz_worked.py
"""
import json
import os
from fractions import Fraction as F

EPS = F(1, 10 ** 6)


def worked(cells, order, vel):
    c = [F(x) for x in cells]
    q = c[0:5] if vel > 0 else c[::-1][0:5]           # q[2] is the upwind cell of the face between cells[2] and cells[3]
    m2, m1, q0, p1, p2 = q
    if order == 3:
        cand = [(2 * m2 - 7 * m1 + 11 * q0) / 6, (-m1 + 5 * q0 + 2 * p1) / 6, (2 * q0 + 5 * p1 - p2) / 6]
        beta = [F(13, 12) * (m2 - 2 * m1 + q0) ** 2 + F(1, 4) * (m2 - 4 * m1 + 3 * q0) ** 2,
                F(13, 12) * (m1 - 2 * q0 + p1) ** 2 + F(1, 4) * (m1 - p1) ** 2,
                F(13, 12) * (q0 - 2 * p1 + p2) ** 2 + F(1, 4) * (3 * q0 - 4 * p1 + p2) ** 2]
        lin = [F(1, 10), F(6, 10), F(3, 10)]
    else:
        cand = [(3 * q0 - m1) / 2, (q0 + p1) / 2]
        beta = [(q0 - m1) ** 2, (p1 - q0) ** 2]
        lin = [F(1, 3), F(2, 3)]
    tau = abs(beta[0] - beta[-1])
    al = [d * (1 + (tau / (b + EPS)) ** 2) for d, b in zip(lin, beta)]
    return sum(a * p for a, p in zip(al, cand)) / sum(al)


CASES = [([0, 0, 0, 1, 1, 1], 3, 1), ([0, 0, 0, 1, 1, 1], 3, -1), ([1, 2, 4, 8, 16, 32], 3, 1),
         ([1, 2, 4, 8, 16, 32], 3, -1), ([3, -1, 4, 1, -5, 9], 3, 1), ([3, -1, 4, 1, -5, 9], 2, -1),
         ([0, 1, 3, 4, 9, 2], 2, 1), ([2, 7, 1, 8, 2, 8], 3, -1)]

if __name__ == "__main__":
    out = {"source": "exact rational evaluation of WENO-Z (Borges et al. 2008 weights on Jiang-Shu candidates; DESIGN.md 3.15)",
           "cases": []}
    for cells, order, vel in CASES:
        v = worked(cells, order, vel)
        out["cases"].append({"cells": cells, "order": order, "vel": vel, "num": str(v.numerator),
                             "den": str(v.denominator), "approx": float(v)})
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "wenoz_worked.json"), "w") as fh:
        json.dump(out, fh, indent=1)
