"""(v) of north_star: brute-force hand calculation at single points on a 4x4x2 grid.

An independent point-wise evaluator of DESIGN.md §3.5-§3.7 (python scalars, explicit modulo
indexing, gathers one value at a time) against the oracle's array passes.  With 4 periodic
cells the 6-cell WENO stencil wraps onto itself (halo 3 <= N = 4 is legal) and the single
interior vertical face has order 1 (SURVEY.md §8c pins).
"""
import numpy as np

import oracle
from paper_2309_06662_b200 import workloads as W
from util import box

NX = NY = 4
NZ = 2


def _weno5(q):                       # q = (q-2, q-1, q0, q+1, q+2), q0 upwind
    a, b, c, d, e = q
    p = [(2 * a - 7 * b + 11 * c) / 6, (-b + 5 * c + 2 * d) / 6, (2 * c + 5 * d - e) / 6]
    be = [13 / 12 * (a - 2 * b + c) ** 2 + (a - 4 * b + 3 * c) ** 2 / 4,
          13 / 12 * (b - 2 * c + d) ** 2 + (b - d) ** 2 / 4,
          13 / 12 * (c - 2 * d + e) ** 2 + (3 * c - 4 * d + e) ** 2 / 4]
    al = [g / (1e-6 + x) ** 2 for g, x in zip((0.1, 0.6, 0.3), be)]
    return sum(x * y for x, y in zip(al, p)) / sum(al)


def _face(cells6, vel, order):
    s = cells6[0:5] if vel > 0 else cells6[::-1][0:5]
    return _weno5(s) if order == 3 else s[2]


class Hand:
    def __init__(self, wl, fld, w, p):
        self.g, self.P = wl["grid"], wl["params"]
        self.dz = np.diff(wl["z_faces"])
        self.f = fld
        self.w_, self.p_ = w, p
        self.dx, self.dy = self.g["dx"], self.g["dy"]

    def at(self, name, k, j, i):
        return float(self.f[name][k, j % NY, i % NX])

    def w(self, k, j, i):
        return float(self.w_[k, j % NY, i % NX])

    def p(self, k, j, i):
        return float(self.p_[k, j % NY, i % NX])

    def zeta(self, k, j, i):
        return ((self.at("v", k, j, i) - self.at("v", k, j, i - 1)) / self.dx
                - (self.at("u", k, j, i) - self.at("u", k, j - 1, i)) / self.dy)

    def K(self, k, j, i):
        return 0.25 * (self.at("u", k, j, i) ** 2 + self.at("u", k, j, i + 1) ** 2
                       + self.at("v", k, j, i) ** 2 + self.at("v", k, j + 1, i) ** 2)

    def D(self, k, j, i):
        return ((self.at("u", k, j, i + 1) - self.at("u", k, j, i)) / self.dx
                + (self.at("v", k, j + 1, i) - self.at("v", k, j, i)) / self.dy)

    def Gu(self, k, j, i):
        f0, nu = self.g["f0"], self.P["nu_h"]
        vhat = 0.25 * (self.at("v", k, j, i - 1) + self.at("v", k, j, i)
                       + self.at("v", k, j + 1, i - 1) + self.at("v", k, j + 1, i))
        zt = _face([self.zeta(k, j + m, i) for m in range(-2, 4)], vhat, 3)
        out = zt * vhat + f0 * vhat
        out -= (self.K(k, j, i) - self.K(k, j, i - 1)) / self.dx
        out -= (self.p(k, j, i) - self.p(k, j, i - 1)) / self.dx
        # vertical advection: the only interior face is k = 1
        du = self.at("u", 1, j, i) - self.at("u", 0, j, i)
        wbar = 0.5 * (self.w(1, j, i - 1) + self.w(1, j, i))
        out -= 0.5 * wbar * du / self.dz[k]
        out += nu * ((self.D(k, j, i) - self.D(k, j, i - 1)) / self.dx
                     - (self.zeta(k, j + 1, i) - self.zeta(k, j, i)) / self.dy)
        if k == NZ - 1:
            out += float(self.f["tau_x"][j % NY, i % NX]) / (self.P["rho0"] * self.dz[k])
        return out

    def Gv(self, k, j, i):
        f0, nu = self.g["f0"], self.P["nu_h"]
        uhat = 0.25 * (self.at("u", k, j - 1, i) + self.at("u", k, j, i)
                       + self.at("u", k, j - 1, i + 1) + self.at("u", k, j, i + 1))
        zt = _face([self.zeta(k, j, i + m) for m in range(-2, 4)], uhat, 3)
        out = -zt * uhat - f0 * uhat
        out -= (self.K(k, j, i) - self.K(k, j - 1, i)) / self.dy
        out -= (self.p(k, j, i) - self.p(k, j - 1, i)) / self.dy
        dv = self.at("v", 1, j, i) - self.at("v", 0, j, i)
        wbar = 0.5 * (self.w(1, j - 1, i) + self.w(1, j, i))
        out -= 0.5 * wbar * dv / self.dz[k]
        out += nu * ((self.D(k, j, i) - self.D(k, j - 1, i)) / self.dy
                     + (self.zeta(k, j, i + 1) - self.zeta(k, j, i)) / self.dx)
        if k == NZ - 1:
            out += float(self.f["tau_y"][j % NY, i % NX]) / (self.P["rho0"] * self.dz[k])
        return out

    def Gc(self, name, k, j, i):
        kh = self.P["kappa_h"]

        def fx(ii):      # flux through the west face of cell ii, per unit dy*dz
            uu = self.at("u", k, j, ii)
            cf = _face([self.at(name, k, j, ii + m) for m in range(-3, 3)], uu, 3)
            return uu * cf - kh * (self.at(name, k, j, ii) - self.at(name, k, j, ii - 1)) / self.dx

        def fy(jj):
            vv = self.at("v", k, jj, i)
            cf = _face([self.at(name, k, jj + m, i) for m in range(-3, 3)], vv, 3)
            return vv * cf - kh * (self.at(name, k, jj, i) - self.at(name, k, jj - 1, i)) / self.dy

        w1 = self.w(1, j, i)
        fz1 = w1 * (self.at(name, 0, j, i) if w1 > 0 else self.at(name, 1, j, i))   # order 1 upwind
        fz_lo, fz_hi = (0.0, fz1) if k == 0 else (fz1, 0.0)
        return -((fx(i + 1) - fx(i)) / self.dx + (fy(j + 1) - fy(j)) / self.dy + (fz_hi - fz_lo) / self.dz[k])


def test_hand_calculation_4x4x2():
    rng = np.random.default_rng(42)
    wl = box(nx=NX, ny=NY, nz=NZ, depth=100.0, dx=1000.0, dy=1500.0, f0=1e-4, nu_h=20.0, kappa_h=3.0)
    fl = wl["fields"]
    fl["u"] = 0.2 * rng.standard_normal((NZ, NY, NX))
    fl["v"] = 0.2 * rng.standard_normal((NZ, NY, NX))
    fl["T"] = 10.0 + rng.standard_normal((NZ, NY, NX))
    fl["S"] = 35.0 + 0.3 * rng.standard_normal((NZ, NY, NX))
    fl["tau_x"] = 0.1 * rng.standard_normal((NY, NX))
    fl["tau_y"] = 0.1 * rng.standard_normal((NY, NX))
    m = oracle.RefModel(wl)
    masks = m.grid.masks()
    assert masks["order_x"].min() == 3 and masks["order_zeta_u"].min() == 3     # stencil wraps onto itself
    assert np.all(masks["order_z"][1] == 1) and np.all(masks["order_z"][[0, 2]] == 0)
    st, dg, G = m.get_fields(), m.diagnostics(), m.tendencies()

    # hand-computed diagnostics at every column: tiny grid, 2 levels
    P, dz = wl["params"], np.diff(wl["z_faces"])
    b = P["g"] * (P["alpha"] * (fl["T"] - P["T0"]) - P["beta_s"] * (fl["S"] - P["S0"]))
    p_hand = np.empty((NZ, NY, NX))
    p_hand[1] = -b[1] * (dz[1] / 2)
    p_hand[0] = p_hand[1] - 0.5 * (b[1] + b[0]) * (dz[0] / 2 + dz[1] / 2)
    assert np.max(np.abs(p_hand - dg["p"])) < 1e-15
    div = lambda k: ((np.roll(fl["u"][k], -1, 1) - fl["u"][k]) / 1000.0       # noqa: E731
                     + (np.roll(fl["v"][k], -1, 0) - fl["v"][k]) / 1500.0)
    w_hand = np.zeros((NZ + 1, NY, NX))
    w_hand[1] = -dz[0] * div(0)
    w_hand[2] = w_hand[1] - dz[1] * div(1)
    assert np.max(np.abs(w_hand - st["w"])) < 1e-16

    h = Hand(wl, fl, w_hand, p_hand)
    for (k, j, i) in [(0, 0, 0), (1, 2, 3), (0, 3, 1), (1, 0, 2), (1, 3, 3), (0, 1, 2)]:
        for name, fn in (("Gu", h.Gu), ("Gv", h.Gv)):
            want = fn(k, j, i)
            assert abs(G[name][k, j, i] - want) < 1e-12 * max(1e-4, abs(want)), (name, k, j, i)
        for name, c in (("GT", "T"), ("GS", "S")):
            want = h.Gc(c, k, j, i)
            assert abs(G[name][k, j, i] - want) < 1e-11 * max(1e-4, abs(want)), (name, k, j, i)
