"""Pins of the oracle ON THE SPHERE and ON BATHYMETRY (PAPER.md:84-86 curvilinear
finite-volume operators, PAPER.md:102 the 75S-75N latitude-longitude domain).

Everything here runs on latitude-longitude grids where dxC != dxF, AzC != AzF and f varies with the row, so that a
metric factor taken at the wrong row or of the wrong kind (the one-token mistakes a Cartesian test cannot see) fails:

 (a) a point-wise hand evaluator (`Sphere`) that works from LATITUDES, not from metric arrays: every length, area and
     Coriolis parameter is the closed form (a cos(phi) dlam, a dphi, a^2 dlam (sin phi2 - sin phi1), 2 Omega sin(phi))
     evaluated at the latitude of the point or edge it belongs to; wet cells come straight from the depth array and
     WENO orders from counting wet neighbours outward from the face.  Compared with the oracle's G_u, G_v, G_T, G_S, w,
     p and one raw barotropic sub-step on an 8 x 6 x 3 grid with two dry columns and one shallow column.
 (b) closed forms and identities of the discrete operators on the sphere: solid-body rotation (D = 0 and
     zeta = (U0/a)(sin phi_c[j] + sin phi_c[j-1]) exactly), uniform meridional flow (D and w in closed form), curl of a
     discrete gradient = 0, Stokes and Gauss sums, the energy neutrality of the Coriolis terms, volume conservation of
     the raw barotropic sub-step on a closed basin, hydrostatic pressure gradient of a zonally linear tracer.
"""
import numpy as np

import oracle
from paper_2309_06662_b200 import workloads as W

RAD = np.pi / 180.0


# =============================================================================================
# inputs
# =============================================================================================
def small_latlon(nx=8, ny=6, nz=3, periodic_x=1, lat0=40.0, dlat=5.0, dlon=5.0, seed=7, land=True, **params):
    rng = np.random.default_rng(seed)
    zf = np.array([-600.0, -300.0, -100.0, 0.0]) if nz == 3 else W.geometric_z_faces(nz, 40.0, 600.0)
    grid = dict(kind=1, nx=nx, ny=ny, nz=nz, periodic_x=periodic_x, periodic_y=0, x0=10.0, dx=dlon, y0=lat0, dy=dlat,
                radius=W.EARTH_RADIUS, rotation_rate=W.EARTH_ROTATION, f0=0.0, beta=0.0)
    depth = np.full((ny, nx), 600.0)
    if land:
        depth[2, 5] = 0.0            # two dry columns
        depth[4, 1] = 0.0
        depth[3, 3] = 250.0          # one shallow column: only the two upper cells are wet
        depth[1, 7] = 80.0           # a single wet cell: becomes land (fewer than 2 wet cells)
    p = W._params(64, 600.0, 10, 800.0, 60.0)
    p.update(params)
    f = dict(u=0.3 * rng.standard_normal((nz, ny, nx)), v=0.3 * rng.standard_normal((nz, ny, nx)),
             T=10.0 + 2.0 * rng.standard_normal((nz, ny, nx)), S=35.0 + 0.5 * rng.standard_normal((nz, ny, nx)),
             eta=0.2 * rng.standard_normal((ny, nx)), tau_x=0.1 * rng.standard_normal((ny, nx)),
             tau_y=0.1 * rng.standard_normal((ny, nx)))
    return dict(name="small_latlon", grid=grid, z_faces=zf, depth=depth, params=p, fields=f, steps=1)


# =============================================================================================
# (a) the hand evaluator
# =============================================================================================
def _w5(a, b, c, d, e):
    p = ((2 * a - 7 * b + 11 * c) / 6, (-b + 5 * c + 2 * d) / 6, (2 * c + 5 * d - e) / 6)
    be = (13 / 12 * (a - 2 * b + c) ** 2 + (a - 4 * b + 3 * c) ** 2 / 4,
          13 / 12 * (b - 2 * c + d) ** 2 + (b - d) ** 2 / 4,
          13 / 12 * (c - 2 * d + e) ** 2 + (3 * c - 4 * d + e) ** 2 / 4)
    al = [g / (1e-6 + x) ** 2 for g, x in zip((0.1, 0.6, 0.3), be)]
    return sum(x * y for x, y in zip(al, p)) / sum(al)


def _w3(b, c, d):
    p = ((3 * c - b) / 2, (c + d) / 2)
    al = ((1 / 3) / (1e-6 + (c - b) ** 2) ** 2, (2 / 3) / (1e-6 + (d - c) ** 2) ** 2)
    return (al[0] * p[0] + al[1] * p[1]) / (al[0] + al[1])


def face_value(six, vel, order):
    """six = values at n-3 .. n+2, face between six[2] and six[3]; DESIGN.md §3.4."""
    s = six if vel > 0 else six[::-1]
    if order == 3:
        return _w5(*s[0:5])
    if order == 2:
        return _w3(*s[1:4])
    return s[2] if order == 1 else 0.0


class Sphere:
    """Point-wise evaluation of DESIGN.md §3.5-§3.8 on a latitude-longitude grid from latitudes and the depth array."""

    def __init__(self, wl):
        g, self.P = wl["grid"], wl["params"]
        self.a, self.Om = g["radius"], g["rotation_rate"]
        self.nx, self.ny, self.nz = g["nx"], g["ny"], g["nz"]
        self.per = bool(g["periodic_x"])
        self.dlam, self.dphi, self.phi0 = g["dx"] * RAD, g["dy"] * RAD, g["y0"] * RAD
        self.zf = np.asarray(wl["z_faces"], float)
        self.zc = 0.5 * (self.zf[1:] + self.zf[:-1])
        self.thick = self.zf[1:] - self.zf[:-1]
        self.depth = wl["depth"]
        self.f = wl["fields"]

    # ---- geometry from latitudes -----------------------------------------------------------
    def lat_edge(self, j):                   # southern edge of row j: v points and vorticity corners
        return self.phi0 + j * self.dphi

    def lat_mid(self, j):                    # middle of row j: tracer and u points
        return self.phi0 + (j + 0.5) * self.dphi

    def arc_x(self, phi):                    # length of one cell along a parallel
        return self.a * np.cos(phi) * self.dlam

    def arc_y(self):
        return self.a * self.dphi

    def zone(self, phi_lo, phi_hi):          # area between two parallels, one cell wide
        return self.a ** 2 * self.dlam * (np.sin(phi_hi) - np.sin(phi_lo))

    def cell_area(self, j):
        return self.zone(self.lat_edge(j), self.lat_edge(j + 1))

    def corner_area(self, j):                # area around the south-west corner of row j
        return self.zone(self.lat_mid(j - 1), self.lat_mid(j))

    def coriolis(self, phi):
        return 2.0 * self.Om * np.sin(phi)

    # ---- wet cells, open faces, orders -------------------------------------------------------
    def col(self, j, i):
        if j < 0 or j >= self.ny:
            return None
        if self.per:
            return j, i % self.nx
        return (j, i) if 0 <= i < self.nx else None

    def wet(self, k, j, i):
        c = self.col(j, i)
        if c is None or k < 0 or k >= self.nz:
            return False
        h = self.depth[c]
        n_wet = int(np.sum(self.zc > -h)) if h > 0 else 0
        return n_wet >= 2 and self.zc[k] > -h

    def open_u(self, k, j, i):
        return self.wet(k, j, i) and self.wet(k, j, i - 1)

    def open_v(self, k, j, i):
        return self.wet(k, j, i) and self.wet(k, j - 1, i)

    @staticmethod
    def _run(ok, start, step):
        n = 0
        while n < 3 and ok(start + n * step):
            n += 1
        return n

    def order_x(self, k, j, i):              # face between cells i-1 and i
        ok = lambda m: self.wet(k, j, m)     # noqa: E731
        return min(self._run(ok, i - 1, -1), self._run(ok, i, +1))

    def order_y(self, k, j, i):
        ok = lambda m: self.wet(k, m, i)     # noqa: E731
        return min(self._run(ok, j - 1, -1), self._run(ok, j, +1))

    def order_z(self, k, j, i):              # face below cell k
        ok = lambda m: self.wet(m, j, i)     # noqa: E731
        return min(self._run(ok, k - 1, -1), self._run(ok, k, +1))

    def corner_ok(self, k, j, i):
        return self.wet(k, j, i) and self.wet(k, j, i - 1) and self.wet(k, j - 1, i) and self.wet(k, j - 1, i - 1)

    def order_zeta_at_u(self, k, j, i):      # between corners j and j+1 of column i
        ok = lambda m: self.corner_ok(k, m, i)     # noqa: E731
        return max(1, min(self._run(ok, j, -1), self._run(ok, j + 1, +1)))

    def order_zeta_at_v(self, k, j, i):      # between corners i and i+1 of row j
        ok = lambda m: self.corner_ok(k, j, m)     # noqa: E731
        return max(1, min(self._run(ok, i, -1), self._run(ok, i + 1, +1)))

    # ---- fields (masked as DESIGN.md §3.3 says) --------------------------------------------------
    def U(self, k, j, i):
        return float(self.f["u"][(k,) + self.col(j, i)]) if self.open_u(k, j, i) else 0.0

    def V(self, k, j, i):
        return float(self.f["v"][(k,) + self.col(j, i)]) if self.open_v(k, j, i) else 0.0

    def C(self, name, k, j, i):
        return float(self.f[name][(k,) + self.col(j, i)]) if self.wet(k, j, i) else 0.0

    def div(self, k, j, i):
        return (self.arc_y() * (self.U(k, j, i + 1) - self.U(k, j, i))
                + self.arc_x(self.lat_edge(j + 1)) * self.V(k, j + 1, i)
                - self.arc_x(self.lat_edge(j)) * self.V(k, j, i)) / self.cell_area(j)

    def w(self, k, j, i):                    # at the bottom face of cell k
        return -sum(self.thick[m] * self.div(m, j, i) for m in range(k))

    def buoy(self, k, j, i):
        P = self.P
        return P["g"] * (P["alpha"] * (self.C("T", k, j, i) - P["T0"]) - P["beta_s"] * (self.C("S", k, j, i) - P["S0"]))

    def p(self, k, j, i):
        top = self.nz - 1
        out = self.buoy(top, j, i) * self.zc[top]                   # -b (0 - zc)
        for m in range(top - 1, k - 1, -1):
            out -= 0.5 * (self.buoy(m + 1, j, i) + self.buoy(m, j, i)) * (self.zc[m + 1] - self.zc[m])
        return out

    def zeta(self, k, j, i):                 # south-west corner of cell (j, i)
        circ = (self.arc_y() * (self.V(k, j, i) - self.V(k, j, i - 1))
                - (self.arc_x(self.lat_mid(j)) * self.U(k, j, i) - self.arc_x(self.lat_mid(j - 1)) * self.U(k, j - 1, i)))
        return circ / self.corner_area(j)

    def ke(self, k, j, i):
        return 0.25 * (self.U(k, j, i) ** 2 + self.U(k, j, i + 1) ** 2 + self.V(k, j, i) ** 2 + self.V(k, j + 1, i) ** 2)

    # ---- tendencies ----------------------------------------------------------------------------
    def Gu(self, k, j, i):
        if not self.open_u(k, j, i):
            return 0.0
        here = self.arc_x(self.lat_mid(j))                                   # dx at the u point
        south, north = self.lat_edge(j), self.lat_edge(j + 1)
        vs = self.V(k, j, i - 1) + self.V(k, j, i)
        vn = self.V(k, j + 1, i - 1) + self.V(k, j + 1, i)
        vhat = 0.25 * (self.arc_x(south) * vs + self.arc_x(north) * vn) / here
        zt = face_value([self.zeta(k, j + m, i) for m in range(-2, 4)], vhat, self.order_zeta_at_u(k, j, i))
        cor = 0.25 * (self.coriolis(south) * self.arc_x(south) * vs + self.coriolis(north) * self.arc_x(north) * vn) / here
        out = zt * vhat + cor
        out -= (self.ke(k, j, i) - self.ke(k, j, i - 1)) / here
        out -= (self.p(k, j, i) - self.p(k, j, i - 1)) / here
        # vertical advection: the cell area cancels for u
        lo = (self.U(k, j, i) - self.U(k - 1, j, i)) if (k >= 1 and self.open_u(k - 1, j, i)) else 0.0
        hi = (self.U(k + 1, j, i) - self.U(k, j, i)) if (k + 1 < self.nz and self.open_u(k + 1, j, i)) else 0.0
        out -= 0.25 * ((self.w(k + 1, j, i - 1) + self.w(k + 1, j, i)) * hi + (self.w(k, j, i - 1) + self.w(k, j, i)) * lo) / self.thick[k]
        out += self.P["nu_h"] * ((self.div(k, j, i) - self.div(k, j, i - 1)) / here
                                 - (self.zeta(k, j + 1, i) - self.zeta(k, j, i)) / self.arc_y())
        if k == self.nz - 1:
            out += float(self.f["tau_x"][self.col(j, i)]) / (self.P["rho0"] * self.thick[k])
        return out

    def Gv(self, k, j, i):
        if not self.open_v(k, j, i):
            return 0.0
        here = self.arc_x(self.lat_edge(j))                                  # dx at the v point
        uhat = 0.25 * (self.U(k, j - 1, i) + self.U(k, j, i) + self.U(k, j - 1, i + 1) + self.U(k, j, i + 1))
        zt = face_value([self.zeta(k, j, i + m) for m in range(-2, 4)], uhat, self.order_zeta_at_v(k, j, i))
        out = -zt * uhat - self.coriolis(self.lat_edge(j)) * uhat
        out -= (self.ke(k, j, i) - self.ke(k, j - 1, i)) / self.arc_y()
        out -= (self.p(k, j, i) - self.p(k, j - 1, i)) / self.arc_y()
        lo = (self.V(k, j, i) - self.V(k - 1, j, i)) if (k >= 1 and self.open_v(k - 1, j, i)) else 0.0
        hi = (self.V(k + 1, j, i) - self.V(k, j, i)) if (k + 1 < self.nz and self.open_v(k + 1, j, i)) else 0.0
        As, An = self.cell_area(j - 1), self.cell_area(j)
        flux_hi = 0.5 * (As * self.w(k + 1, j - 1, i) + An * self.w(k + 1, j, i))
        flux_lo = 0.5 * (As * self.w(k, j - 1, i) + An * self.w(k, j, i))
        out -= 0.5 * (flux_hi * hi + flux_lo * lo) / (self.corner_area(j) * self.thick[k])
        out += self.P["nu_h"] * ((self.div(k, j, i) - self.div(k, j - 1, i)) / self.arc_y()
                                 + (self.zeta(k, j, i + 1) - self.zeta(k, j, i)) / here)
        if k == self.nz - 1:
            out += float(self.f["tau_y"][self.col(j, i)]) / (self.P["rho0"] * self.thick[k])
        return out

    def flux_x(self, name, k, j, i):         # through the west face of cell i
        uu, dz, kh = self.U(k, j, i), self.thick[k], self.P["kappa_h"]
        cf = face_value([self.C(name, k, j, i + m) for m in range(-3, 3)], uu, self.order_x(k, j, i))
        dif = kh * self.arc_y() * dz * (self.C(name, k, j, i) - self.C(name, k, j, i - 1)) / self.arc_x(self.lat_mid(j))
        return uu * self.arc_y() * dz * cf - (dif if self.open_u(k, j, i) else 0.0)

    def flux_y(self, name, k, j, i):         # through the south face of cell j
        vv, dz, kh = self.V(k, j, i), self.thick[k], self.P["kappa_h"]
        edge = self.arc_x(self.lat_edge(j))
        cf = face_value([self.C(name, k, j + m, i) for m in range(-3, 3)], vv, self.order_y(k, j, i))
        dif = kh * edge * dz * (self.C(name, k, j, i) - self.C(name, k, j - 1, i)) / self.arc_y()
        return vv * edge * dz * cf - (dif if self.open_v(k, j, i) else 0.0)

    def flux_z(self, name, k, j, i):         # through the bottom face of cell k
        if k <= 0 or k >= self.nz or not (self.wet(k, j, i) and self.wet(k - 1, j, i)):
            return 0.0
        ww = self.w(k, j, i)
        cf = face_value([self.C(name, k + m, j, i) for m in range(-3, 3)], ww, self.order_z(k, j, i))
        return ww * self.cell_area(j) * cf

    def Gc(self, name, k, j, i):
        if not self.wet(k, j, i):
            return 0.0
        net = (self.flux_x(name, k, j, i + 1) - self.flux_x(name, k, j, i) + self.flux_y(name, k, j + 1, i)
               - self.flux_y(name, k, j, i) + self.flux_z(name, k + 1, j, i) - self.flux_z(name, k, j, i))
        return -net / (self.cell_area(j) * self.thick[k])

    # ---- one raw barotropic sub-step (DESIGN.md §3.8 step 6, no forcing) ----------------------------
    def transport(self, which, j, i):
        if self.col(j, i) is None:
            return 0.0
        fn = self.U if which == "u" else self.V
        return sum(self.thick[k] * fn(k, j, i) for k in range(self.nz))

    def eta0(self, j, i):
        c = self.col(j, i)
        return float(self.f["eta"][c]) if (c is not None and self.wet(self.nz - 1, j, i)) else 0.0

    def eta1(self, j, i, dtau):
        if not self.wet(self.nz - 1, j, i):
            return self.eta0(j, i)
        conv = (self.arc_y() * (self.transport("u", j, i + 1) - self.transport("u", j, i))
                + self.arc_x(self.lat_edge(j + 1)) * self.transport("v", j + 1, i)
                - self.arc_x(self.lat_edge(j)) * self.transport("v", j, i))
        return self.eta0(j, i) - dtau * conv / self.cell_area(j)

    def U1(self, j, i, dtau):
        top = self.nz - 1
        if not self.open_u(top, j, i):
            return 0.0
        H = sum(self.thick[k] for k in range(self.nz) if self.open_u(k, j, i))
        slope = (self.eta1(j, i, dtau) - self.eta1(j, i - 1, dtau)) / self.arc_x(self.lat_mid(j))
        return self.transport("u", j, i) - dtau * self.P["g"] * H * slope

    def V1(self, j, i, dtau):
        top = self.nz - 1
        if not self.open_v(top, j, i):
            return 0.0
        H = sum(self.thick[k] for k in range(self.nz) if self.open_v(k, j, i))
        slope = (self.eta1(j, i, dtau) - self.eta1(j - 1, i, dtau)) / self.arc_y()
        return self.transport("v", j, i) - dtau * self.P["g"] * H * slope


def _close(got, want, rel=1e-11, floor=1e-9):
    return abs(got - want) <= rel * max(abs(want), floor)


def test_hand_evaluator_on_a_small_sphere_patch_with_land():
    wl = small_latlon()
    m = oracle.RefModel(wl)
    h = Sphere(wl)
    nz, ny, nx = 3, 6, 8
    # masks / orders first: the evaluator's outward counting against the oracle's brute force
    mk = m.grid.masks()
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                assert mk["wet"][k, j, i] == h.wet(k, j, i)
                assert mk["order_x"][k, j, i] == h.order_x(k, j, i), (k, j, i)
                assert mk["order_y"][k, j, i] == h.order_y(k, j, i), (k, j, i)
                assert mk["order_zeta_u"][k, j, i] == (h.order_zeta_at_u(k, j, i) if h.open_u(k, j, i) else 0)
                assert mk["order_zeta_v"][k, j, i] == (h.order_zeta_at_v(k, j, i) if h.open_v(k, j, i) else 0)
    assert not h.wet(2, 1, 7) and not h.wet(0, 3, 3) and h.wet(1, 3, 3)       # single-cell column is land; shallow column
    assert set(np.unique(mk["order_x"])) == {0, 1, 2, 3} and set(np.unique(mk["order_y"])) == {0, 1, 2, 3}
    st, dg, G, md = m.get_fields(), m.diagnostics(), m.tendencies(), m.momentum_diagnostics()
    # every point of the grid: 144 cells, python scalars
    n_open = {"Gu": 0, "Gv": 0}
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                assert _close(st["w"][k + 1, j, i], h.w(k + 1, j, i), floor=1e-12), ("w", k, j, i)
                if h.wet(k, j, i):
                    assert _close(dg["p"][k, j, i], h.p(k, j, i)), ("p", k, j, i)
                assert _close(md["zeta"][k, j, i], h.zeta(k, j, i), floor=1e-12), ("zeta", k, j, i)
                assert _close(md["D"][k, j, i], h.div(k, j, i), floor=1e-12), ("D", k, j, i)
                assert _close(md["K"][k, j, i], h.ke(k, j, i)), ("K", k, j, i)
                for name, fn in (("Gu", h.Gu), ("Gv", h.Gv)):
                    want = fn(k, j, i)
                    n_open[name] += want != 0.0
                    assert _close(G[name][k, j, i], want, floor=1e-8), (name, k, j, i, G[name][k, j, i], want)
                for name, c in (("GT", "T"), ("GS", "S")):
                    want = h.Gc(c, k, j, i)
                    assert _close(G[name][k, j, i], want, rel=1e-10, floor=1e-8), (name, k, j, i, G[name][k, j, i], want)
    assert n_open["Gu"] > 80 and n_open["Gv"] > 60
    # the shallow column (3, 3): its u and v faces are closed at k = 0 and open above, so the difference below the
    # k = 1 faces is masked although the velocity stored there is zero
    assert h.open_u(1, 3, 3) and not h.open_u(0, 3, 3) and h.open_u(0, 3, 2) and h.open_v(1, 3, 3) and not h.open_v(0, 3, 3)


def test_hand_evaluator_one_barotropic_substep_on_the_sphere():
    wl = small_latlon(seed=11)
    m = oracle.RefModel(wl)
    h = Sphere(wl)
    dtau = 17.0
    m.barotropic_raw(1, dtau)
    eta, dg = m.get_fields()["eta"], m.diagnostics()
    n = 0
    for j in range(6):
        for i in range(8):
            assert _close(eta[j, i], h.eta1(j, i, dtau)), ("eta", j, i)
            assert _close(dg["U"][j, i], h.U1(j, i, dtau), floor=1e-6), ("U", j, i)
            assert _close(dg["V"][j, i], h.V1(j, i, dtau), floor=1e-6), ("V", j, i)
            n += h.U1(j, i, dtau) != 0.0
    assert n > 30


def test_hand_evaluator_closed_patch_not_periodic():
    # the same evaluator on a patch with walls on all four sides (the config-4 window is run like this)
    wl = small_latlon(periodic_x=0, seed=3, lat0=-62.0, dlat=3.0, dlon=4.0)
    m = oracle.RefModel(wl)
    h = Sphere(wl)
    G = m.tendencies()
    for (k, j, i) in [(2, 0, 0), (1, 3, 4), (2, 5, 7), (1, 2, 6), (0, 3, 2), (2, 3, 3), (1, 3, 3), (2, 4, 2), (0, 1, 1)]:
        assert _close(G["Gu"][k, j, i], h.Gu(k, j, i), floor=1e-8), ("Gu", k, j, i)
        assert _close(G["Gv"][k, j, i], h.Gv(k, j, i), floor=1e-8), ("Gv", k, j, i)
        assert _close(G["GT"][k, j, i], h.Gc("T", k, j, i), rel=1e-10, floor=1e-8), ("GT", k, j, i)


# =============================================================================================
# (b) closed forms and identities on the sphere
# =============================================================================================
def _ocean(nx=12, ny=10, nz=4, lat0=-30.0, dlat=4.0, dlon=6.0, periodic_x=1, depth=600.0, **params):
    wl = small_latlon(nx=nx, ny=ny, nz=nz, periodic_x=periodic_x, lat0=lat0, dlat=dlat, dlon=dlon, land=False, **params)
    wl["depth"][:] = depth
    for n in ("u", "v", "eta", "tau_x", "tau_y"):
        wl["fields"][n][:] = 0.0
    wl["fields"]["T"][:] = 10.0
    wl["fields"]["S"][:] = 35.0
    return wl


def _lats(wl):
    g = wl["grid"]
    pf = (g["y0"] + np.arange(g["ny"] + 1) * g["dy"]) * RAD
    return pf, 0.5 * (pf[1:] + pf[:-1])


def test_solid_body_rotation_has_no_divergence_and_the_closed_form_vorticity():
    wl = _ocean(nu_h=300.0)
    a, U0 = wl["grid"]["radius"], 0.7
    pf, pc = _lats(wl)
    wl["fields"]["u"][:] = (U0 * np.cos(pc))[None, :, None]
    m = oracle.RefModel(wl)
    md, st, G = m.momentum_diagnostics(), m.get_fields(), m.tendencies()
    assert np.max(np.abs(md["D"])) < 1e-22 and np.max(np.abs(st["w"])) < 1e-18
    # zeta at the corner between rows j-1 and j: (U0/a)(sin phi_c[j] + sin phi_c[j-1]); row 0 touches the wall (u = 0 south of it)
    want = (U0 / a) * (np.sin(pc[1:]) + np.sin(pc[:-1]))
    got = md["zeta"][2, 1:, 4]
    assert np.max(np.abs(got - want)) < 1e-13 * np.max(np.abs(want))
    assert abs(want[5] - 2 * (U0 / a) * np.sin(pf[6])) < 2e-3 * abs(want[5])       # the continuum value 2 (U0/a) sin(phi)
    # the only term left in G_u away from the walls is the viscous one, -nu_h (zeta[j+1] - zeta[j]) / dy  (v = 0, K and p uniform in x)
    dy = a * wl["grid"]["dy"] * RAD
    vis = -300.0 * (want[1:] - want[:-1]) / dy                                      # rows 1 .. ny-2
    assert np.max(np.abs(G["Gu"][1, 1:-1, 7] - vis)) < 1e-12 * np.max(np.abs(vis))
    # G_v = -zeta~ u^ - f u^ - dK/dy: with the order-1 upwind value zeta~ = zeta (uniform in x) this is a closed form too
    j = 5
    uhat = 0.5 * U0 * (np.cos(pc[j - 1]) + np.cos(pc[j]))
    dK = 0.5 * U0 ** 2 * (np.cos(pc[j]) ** 2 - np.cos(pc[j - 1]) ** 2) / dy
    f = 2 * wl["grid"]["rotation_rate"] * np.sin(pf[j])
    assert abs(G["Gv"][3, j, 2] - (-(want[j - 1] + f) * uhat - dK)) < 1e-12 * abs(f * uhat)


def test_uniform_meridional_flow_divergence_and_w_closed_form():
    wl = _ocean()
    a, V0 = wl["grid"]["radius"], 0.4
    pf, pc = _lats(wl)
    wl["fields"]["v"][:] = V0
    m = oracle.RefModel(wl)
    md, st = m.momentum_diagnostics(), m.get_fields()
    Dw = V0 * (np.cos(pf[2:-1]) - np.cos(pf[1:-2])) / (a * (np.sin(pf[2:-1]) - np.sin(pf[1:-2])))     # rows 1 .. ny-2
    assert np.max(np.abs(md["D"][0, 1:-1, 3] - Dw)) < 1e-13 * np.max(np.abs(Dw))
    assert abs(Dw[4] + V0 * np.tan(pc[5]) / a) < 1e-3 * abs(Dw[4])                  # continuum: -(V0/a) tan(phi)
    assert np.max(np.abs(st["w"][-1, 1:-1, 9] + 600.0 * Dw)) < 1e-13 * 600.0 * np.max(np.abs(Dw))


def test_curl_of_a_discrete_gradient_vanishes_and_stokes_gauss_sums():
    wl = _ocean()
    g = wl["grid"]
    rng = np.random.default_rng(5)
    ny, nx, nz = g["ny"], g["nx"], g["nz"]
    ref = oracle.RefModel(wl)
    met = ref.grid.metrics()
    # u = d(chi)/dx, v = d(chi)/dy with the oracle's own face distances: zeta must vanish identically
    chi = rng.standard_normal((ny, nx)) * 1e4
    u = (chi - np.roll(chi, 1, axis=1)) / met["dxC"][:, None]
    v = np.zeros((ny, nx))
    v[1:] = (chi[1:] - chi[:-1]) / met["dy"]
    wl["fields"]["u"][:] = u[None]
    wl["fields"]["v"][:] = v[None]
    m = oracle.RefModel(wl)
    z = m.momentum_diagnostics()["zeta"]
    scale = np.max(np.abs(u)) / met["dy"]
    assert np.max(np.abs(z[:, 1:, :])) < 1e-13 * scale                       # row 0 lies on the wall
    # Stokes: sum of zeta * AzF over the corners of rows j1..j2 (all longitudes) = circulation of u along the two bounding
    # parallels; Gauss: sum of D * AzC over rows = meridional transport through the two bounding parallels
    wl2 = _ocean()
    wl2["fields"]["u"][:] = rng.standard_normal((nz, ny, nx))
    wl2["fields"]["v"][:] = rng.standard_normal((nz, ny, nx))
    m2 = oracle.RefModel(wl2)
    st2, md2 = m2.get_fields(), m2.momentum_diagnostics()
    a, dlam = g["radius"], g["dx"] * RAD
    pf, pc = _lats(wl2)
    AzF = a * a * dlam * (np.sin(pc[1:]) - np.sin(pc[:-1]))                  # corners between rows j-1 and j, j = 1..ny-1
    AzC = a * a * dlam * (np.sin(pf[1:]) - np.sin(pf[:-1]))
    k, j1, j2 = 2, 3, 7
    lhs = np.sum(md2["zeta"][k, j1:j2 + 1, :] * AzF[j1 - 1:j2, None])
    rhs = -(a * np.cos(pc[j2]) * dlam * st2["u"][k, j2].sum() - a * np.cos(pc[j1 - 1]) * dlam * st2["u"][k, j1 - 1].sum())
    assert abs(lhs - rhs) < 1e-12 * abs(rhs)
    lhs = np.sum(md2["D"][k, j1:j2 + 1, :] * AzC[j1:j2 + 1, None])
    rhs = a * np.cos(pf[j2 + 1]) * dlam * st2["v"][k, j2 + 1].sum() - a * np.cos(pf[j1]) * dlam * st2["v"][k, j1].sum()
    assert abs(lhs - rhs) < 1e-12 * abs(rhs)


def test_coriolis_terms_do_no_work_on_the_sphere_with_land():
    # C_u, C_v = G(Omega) - G(0): everything else is identical.  sum u C_u dxC dy dz - sum v C_v dxF dy dz = 0 for
    # the energy-conserving 4-point average with f at the corners (reading 5)
    wl = W.config2(nx=36, ny=24, nz=6, steps=1)
    rng = np.random.default_rng(9)
    wl["fields"]["u"] = rng.standard_normal(wl["fields"]["u"].shape)
    wl["fields"]["v"] = rng.standard_normal(wl["fields"]["v"].shape)
    m1 = oracle.RefModel(wl)
    wl0 = {**wl, "grid": {**wl["grid"], "rotation_rate": 0.0}}
    m0 = oracle.RefModel(wl0)
    G1, G0, st = m1.tendencies(), m0.tendencies(), m1.get_fields()
    Cu, mCv = G1["Gu"] - G0["Gu"], G1["Gv"] - G0["Gv"]
    g = wl["grid"]
    a, dlam, dphi = g["radius"], g["dx"] * RAD, g["dy"] * RAD
    pf, pc = _lats(wl)
    dz = np.diff(wl["z_faces"])[:, None, None]
    work_u = np.sum(st["u"] * Cu * (a * np.cos(pc) * dlam * a * dphi)[None, :, None] * dz)
    work_v = np.sum(st["v"] * mCv * (a * np.cos(pf[:-1]) * dlam * a * dphi)[None, :, None] * dz)
    assert abs(work_u) > 1e3 * abs(work_u + work_v) and abs(work_u + work_v) < 1e-11 * abs(work_u)
    # and they are what they should be at a point in the open ocean: C_v = f(phi_f[j]) u^
    wet = m1.grid.masks()["wet"]
    k = 5
    j, i = next((j, i) for j in range(3, 20) for i in range(3, 30) if wet[k, j - 1:j + 1, i - 1:i + 2].all())
    uhat = 0.25 * (st["u"][k, j - 1, i] + st["u"][k, j, i] + st["u"][k, j - 1, i + 1] + st["u"][k, j, i + 1])
    assert abs(-mCv[k, j, i] - 2 * g["rotation_rate"] * np.sin(pf[j]) * uhat) < 1e-10 * abs(mCv[k, j, i])


def test_raw_barotropic_substeps_conserve_volume_on_a_closed_latlon_basin():
    wl = W.config2(nx=40, ny=28, nz=6, steps=1)
    wl["grid"]["periodic_x"] = 0
    rng = np.random.default_rng(2)
    wl["fields"]["eta"] = 0.5 * rng.standard_normal(wl["fields"]["eta"].shape)
    wl["fields"]["u"] = 0.1 * rng.standard_normal(wl["fields"]["u"].shape)
    wl["fields"]["v"] = 0.1 * rng.standard_normal(wl["fields"]["v"].shape)
    m = oracle.RefModel(wl)
    g = wl["grid"]
    pf, _ = _lats(wl)
    area = (g["radius"] ** 2 * g["dx"] * RAD * (np.sin(pf[1:]) - np.sin(pf[:-1])))[:, None]
    e0 = m.get_fields()["eta"]
    m.barotropic_raw(25, 8.0)
    e1 = m.get_fields()["eta"]
    assert np.max(np.abs(e1 - e0)) > 1e-3
    assert abs(np.sum(area * (e1 - e0))) < 1e-13 * np.sum(area * np.abs(e1 - e0))


def test_barotropic_gravity_wave_on_the_sphere_zonal_closed_form():
    # zonally periodic channel between walls, flat bottom, eta = cos(m lambda) uniform in latitude, U = V = 0, no rotation
    # in the sub-step: after one sub-step U[j, i] = -dtau g H (eta[i] - eta[i-1]) / (a cos(phi_c[j]) dlam) exactly, and the
    # second sub-step's eta change is -dtau dy (U[i+1] - U[i]) / AzC[j] (V stays 0)
    wl = _ocean(nx=16, ny=8, nz=3, lat0=20.0, dlat=5.0, dlon=22.5)
    g = wl["grid"]
    lam = (np.arange(16) + 0.5) * g["dx"] * RAD
    wl["fields"]["eta"][:] = 0.3 * np.cos(2 * lam)[None, :]
    m = oracle.RefModel(wl)
    dtau, H, a = 30.0, 600.0, g["radius"]
    pf, pc = _lats(wl)
    m.barotropic_raw(1, dtau)
    e1, d1 = m.get_fields()["eta"], m.diagnostics()
    assert np.array_equal(e1, wl["fields"]["eta"]) and np.all(d1["V"] == 0.0)
    want_U = -dtau * W.GRAVITY * H * (e1 - np.roll(e1, 1, axis=1)) / (a * np.cos(pc) * g["dx"] * RAD)[:, None]
    assert np.max(np.abs(d1["U"] - want_U)) < 1e-13 * np.max(np.abs(want_U))
    m.barotropic_raw(1, dtau)
    e2 = m.get_fields()["eta"]
    AzC = (a * a * g["dx"] * RAD * (np.sin(pf[1:]) - np.sin(pf[:-1])))[:, None]
    want = e1 - dtau * (a * g["dy"] * RAD) * (np.roll(want_U, -1, axis=1) - want_U) / AzC
    assert np.max(np.abs(e2 - want)) < 1e-13


def test_pressure_gradient_of_a_zonally_linear_tracer_closed_form():
    # T = T0 + gam * i (closed patch), S = S0: b = g alpha gam i, p(k) = b zc(k) ... so G_u = -(p[i] - p[i-1]) / dxC[j]
    # = -g alpha gam zc[k] / (a cos(phi_c[j]) dlam) at rest, on every open u face
    wl = _ocean(periodic_x=0, nu_h=0.0, kappa_h=0.0)
    g, P = wl["grid"], wl["params"]
    gam = 0.05
    wl["fields"]["T"][:] = 10.0 + gam * np.arange(g["nx"])[None, None, :]
    m = oracle.RefModel(wl)
    G = m.tendencies()
    zc = 0.5 * (wl["z_faces"][1:] + wl["z_faces"][:-1])
    _, pc = _lats(wl)
    # trapezoid rule is exact for a buoyancy that does not vary with depth: p(k) = b * zc(k)
    want = -(P["g"] * P["alpha"] * gam) * zc[:, None] / (g["radius"] * np.cos(pc) * g["dx"] * RAD)[None, :]
    got = G["Gu"][:, :, 1:]
    assert np.max(np.abs(got - want[:, :, None])) < 1e-12 * np.max(np.abs(want))
    assert np.all(G["Gu"][:, :, 0] == 0.0) and np.max(np.abs(G["Gv"])) < 1e-18
