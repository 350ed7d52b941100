"""Pins of the oracle's building blocks against what the mathematics fixes.

None of these re-types the oracle's formula: they use closed forms, exactness properties,
exact rational arithmetic on a worked stencil (tests/golden/), dense linear algebra, and
brute force on tiny inputs.
"""
import json
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
from paper_2309_06662_b200 import workloads as W
from util import box

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------ WENO ----
def _cell_averages(poly, n0, n1):
    """exact averages of a numpy poly1d over unit cells [n, n+1], n = n0..n1-1"""
    P = poly.integ()
    return np.array([P(n + 1.0) - P(n) for n in range(n0, n1)])


@pytest.mark.parametrize("vel", [1.0, -1.0])
def test_weno5_exact_for_quadratics(vel):
    # every r = 3 candidate reproduces a quadratic from its cell averages, so the nonlinear
    # weights cannot matter: the face value at x = 0 is exact (Shu 1997)
    rng = np.random.default_rng(1)
    for _ in range(20):
        poly = np.poly1d(rng.standard_normal(3))
        c = _cell_averages(poly, -3, 3)            # cells n-3..n+2, interface at x = 0
        assert abs(oracle.weno(c, 3, vel) - poly(0.0)) < 1e-12 * (1 + abs(poly(0.0)))


@pytest.mark.parametrize("vel", [1.0, -1.0])
def test_weno3_exact_for_linear(vel):
    rng = np.random.default_rng(2)
    for _ in range(20):
        poly = np.poly1d(rng.standard_normal(2))
        c = _cell_averages(poly, -3, 3)
        assert abs(oracle.weno(c, 2, vel) - poly(0.0)) < 1e-13 * (1 + abs(poly(0.0)))


def test_weno_constants_and_order1_upwind():
    c = np.full(6, 3.25)
    for order in (1, 2, 3):
        for vel in (1.0, -1.0, 0.0):
            assert oracle.weno(c, order, vel) == 3.25
    c = np.arange(6.0)
    assert oracle.weno(c, 1, +1.0) == 2.0          # upwind cell n-1
    assert oracle.weno(c, 1, -1.0) == 3.0          # upwind cell n
    assert oracle.weno(c, 1, 0.0) == 3.0           # tie -> right-biased (reading 14)
    assert oracle.weno(c, 0, 1.0) == 0.0           # closed face


def test_weno_mirror_symmetry():
    rng = np.random.default_rng(3)
    for order in (2, 3):
        for _ in range(50):
            c = rng.standard_normal(6)
            assert oracle.weno(c, order, +1.0) == oracle.weno(c[::-1].copy(), order, -1.0)


def test_weno5_fifth_order_convergence():
    # smooth profile: face-value error falls ~2^5 per grid halving
    f = lambda x: np.sin(x) + 2.0                                 # noqa: E731
    F = lambda x: -np.cos(x) + 2.0 * x                            # noqa: E731
    errs = []
    for h in (0.2, 0.1, 0.05):
        x0 = 0.3
        edges = x0 + h * np.arange(-3, 4)
        c = (F(edges[1:]) - F(edges[:-1])) / h
        errs.append(abs(oracle.weno(c, 3, 1.0) - f(x0)))
    assert errs[0] / errs[1] > 20 and errs[1] / errs[2] > 20


def test_weno5_worked_stencil_exact_rational():
    """golden/weno_worked.json: the r = 3 formula evaluated by hand in exact rationals on
    integer stencils (Jiang-Shu weights d = 1/10, 6/10, 3/10, eps = 1e-6; Shu 1997 eq. 2.58-2.63
    as cited at PAPER.md:244).  Written by tests/golden/make_weno_worked.py (Fractions only)."""
    with open(os.path.join(GOLD, "weno_worked.json")) as fh:
        gold = json.load(fh)
    for case in gold["cases"]:
        c = np.array(case["cells"], dtype=np.float64)
        want = Fraction(case["num"]) / Fraction(case["den"])
        got = oracle.weno(c, case["order"], case["vel"])
        assert abs(got - float(want)) <= 4e-16 * max(1.0, abs(float(want))), case


# ------------------------------------------------------- implicit column ----
def _dense_matrix(zf, open_faces, dtk):
    """independent dense assembly: A = I - dt*kappa * Dz^-1 * Gt * Dzc^-1 * G  (flux form)"""
    nz = len(zf) - 1
    dz = np.diff(zf)
    zc = 0.5 * (zf[:-1] + zf[1:])
    G = np.zeros((nz + 1, nz))                    # face gradient, faces 1..nz-1
    for k in range(1, nz):
        if open_faces[k]:
            G[k, k] = 1.0 / (zc[k] - zc[k - 1])
            G[k, k - 1] = -1.0 / (zc[k] - zc[k - 1])
    Dv = np.zeros((nz, nz + 1))                   # flux divergence
    for k in range(nz):
        Dv[k, k + 1] = 1.0 / dz[k]
        Dv[k, k] = -1.0 / dz[k]
    return np.eye(nz) - dtk * Dv @ G


def test_implicit_column_matches_dense_solve():
    rng = np.random.default_rng(4)
    for nz in (2, 3, 7, 12):
        zf = -np.cumsum(rng.uniform(5, 50, nz + 1))[::-1]
        zf -= zf[-1]
        open_faces = np.ones(nz + 1, np.uint8)
        open_faces[0] = open_faces[nz] = 0
        if nz > 4:
            open_faces[2] = 0                     # a closed interior face decouples the column
        phi = rng.standard_normal(nz)
        dtk = 300.0 * 1e-2
        want = np.linalg.solve(_dense_matrix(zf, open_faces, dtk), phi)
        got = oracle.implicit_column(zf, open_faces, dtk, phi)
        assert np.max(np.abs(got - want)) < 1e-13


def test_implicit_column_cosine_mode_decay_and_conservation():
    nz, dz, dtk = 16, 10.0, 60.0 * 0.05
    zf = -dz * np.arange(nz, -1, -1.0)
    open_faces = np.ones(nz + 1, np.uint8)
    k = np.arange(nz)
    for m in (1, 3, 8):
        phi = np.cos(np.pi * m * (k + 0.5) / nz)
        got = oracle.implicit_column(zf, open_faces, dtk, phi)
        decay = 1.0 / (1.0 + dtk * (4.0 / dz ** 2) * np.sin(np.pi * m / (2 * nz)) ** 2)
        assert np.max(np.abs(got - decay * phi)) < 1e-14
    rng = np.random.default_rng(5)
    zf = -np.cumsum(rng.uniform(5, 50, nz + 1))[::-1]
    zf -= zf[-1]
    phi = rng.standard_normal(nz)
    got = oracle.implicit_column(zf, open_faces, 500.0, phi)
    assert abs(np.sum(np.diff(zf) * (got - phi))) < 1e-12          # no-flux ends: integral kept


# ----------------------------------------------------------------- filter ----
def test_filter_weights():
    for M, printed in ((20, 0.07271), (30, 0.04920), (40, 0.03719)):   # SURVEY.md §8(c-9) values
        a, ratio = oracle.filter_weights(M)
        assert abs(a.sum() - 1.0) < 1e-14 and np.all(a > 0)
        assert abs(ratio * np.sum(np.arange(1, M + 1) * a) - 1.0) < 1e-14
        assert abs(ratio - printed) < 6e-6
        # power-law shape p = 2, q = 4: a_m / a_1 = (m^2 (1 - s_m^4)) / (1 - s_1^4)
        s = np.arange(1, M + 1) / (M + 1.0)
        assert np.allclose(a / a[0], (s ** 2 * (1 - s ** 4)) / (s[0] ** 2 * (1 - s[0] ** 4)), rtol=1e-13)


# ------------------------------------------------------------------ metrics ----
def test_latlon_zone_area_closed_form():
    wl = W.config2(nx=72, ny=30, nz=4, steps=1)
    g = oracle.RefGrid(wl["grid"], wl["z_faces"], wl["depth"])
    m = g.metrics()
    a = W.EARTH_RADIUS
    want = a * a * 2 * np.pi * (np.sin(np.deg2rad(75.0)) - np.sin(np.deg2rad(-75.0)))
    assert abs(72 * m["AzC"].sum() - want) < 1e-12 * want
    # dy = a*dphi; f at the equator face row is 0; dxC at 60N is half the equatorial dxF
    assert abs(m["dy"] - a * np.deg2rad(5.0)) < 1e-9
    assert abs(m["fF"][15]) < 1e-18
    assert abs(m["fF"][0] - 2 * W.EARTH_ROTATION * np.sin(np.deg2rad(-75.0))) < 1e-18
    assert abs(m["dxF"][15] - a * np.deg2rad(5.0)) < 1e-6


def test_cartesian_metrics_and_beta_plane():
    wl = box(nx=8, ny=10, nz=2, dx=2000.0, dy=3000.0, f0=1e-4, beta=2e-11)
    g = oracle.RefGrid(wl["grid"], wl["z_faces"], wl["depth"])
    m = g.metrics()
    assert np.all(m["dxC"] == 2000.0) and np.all(m["AzF"] == 6e6) and m["dy"] == 3000.0
    yf = 3000.0 * np.arange(10)
    assert np.allclose(m["fF"], 1e-4 + 2e-11 * (yf - 15000.0), rtol=0, atol=1e-20)


# -------------------------------------------------------------------- masks ----
def _brute_masks(wl):
    """independent brute force with explicit modulo / out-of-range-is-land indexing"""
    g = wl["grid"]
    nx, ny, nz = g["nx"], g["ny"], g["nz"]
    zf = wl["z_faces"]
    zc = 0.5 * (zf[:-1] + zf[1:])
    h = wl["depth"]
    wet3 = (zc[:, None, None] > -h[None]) & (h[None] > 0)
    wet3 &= (wet3.sum(axis=0) >= 2)[None]

    def wet(k, j, i):
        if k < 0 or k >= nz:
            return False
        if g["periodic_x"]:
            i %= nx
        elif i < 0 or i >= nx:
            return False
        if g["periodic_y"]:
            j %= ny
        elif j < 0 or j >= ny:
            return False
        return bool(wet3[k, j, i])

    def longest(cells_at_r):
        o = 0
        for r in (1, 2, 3):
            if all(cells_at_r(r)):
                o = r
            else:
                break
        return o

    def zvalid(k, j, i):
        return wet(k, j - 1, i - 1) and wet(k, j - 1, i) and wet(k, j, i - 1) and wet(k, j, i)

    out = {n: np.zeros((nz, ny, nx), np.uint8) for n in ("wet", "order_x", "order_y", "order_zeta_u", "order_zeta_v")}
    out["order_z"] = np.zeros((nz + 1, ny, nx), np.uint8)
    for k in range(nz + 1):
        for j in range(ny):
            for i in range(nx):
                out["order_z"][k, j, i] = longest(lambda r: [wet(m, j, i) for m in range(k - r, k + r)])
                if k == nz:
                    continue
                out["wet"][k, j, i] = wet(k, j, i)
                out["order_x"][k, j, i] = longest(lambda r: [wet(k, j, m) for m in range(i - r, i + r)])
                out["order_y"][k, j, i] = longest(lambda r: [wet(k, m, i) for m in range(j - r, j + r)])
                if wet(k, j, i) and wet(k, j, i - 1):
                    out["order_zeta_u"][k, j, i] = max(1, longest(lambda r: [zvalid(k, m, i) for m in range(j + 1 - r, j + r + 1)]))
                if wet(k, j, i) and wet(k, j - 1, i):
                    out["order_zeta_v"][k, j, i] = max(1, longest(lambda r: [zvalid(k, j, m) for m in range(i + 1 - r, i + r + 1)]))
    return out


@pytest.mark.parametrize("periodic", [(1, 1), (1, 0), (0, 0)])
def test_masks_and_orders_brute_force(periodic):
    rng = np.random.default_rng(7)
    wl = box(nx=11, ny=9, nz=6, periodic=periodic, depth=600.0)
    d = rng.uniform(0, 700.0, (9, 11))
    land = rng.uniform(size=d.shape) < 0.25
    land[:, :6] = False                            # keep an open region so that order 3 occurs
    d[land] = 0.0
    d[:, :6] = np.maximum(d[:, :6], 350.0)
    d[4, 8] = 120.0                                # one wet cell only (zc = -50) -> becomes land
    wl["depth"] = d
    g = oracle.RefGrid(wl["grid"], wl["z_faces"], wl["depth"])
    got, want = g.masks(), _brute_masks(wl)
    assert got["wet"][:, 4, 8].sum() == 0
    for n in want:
        assert np.array_equal(got[n], want[n]), n
    assert got["order_z"][0].max() == 0 and got["order_z"][-1].max() == 0
    assert got["order_x"].max() == 3 and got["order_zeta_u"].max() == 3
