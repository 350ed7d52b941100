"""Pins of the scheme variants the oracle offers beyond the north_star path:
WENO-Z nonlinear weights (`advection = 1`) and the nonlinear equation of state with thermobaricity and
cabbeling (`eos = 1`).  Each is pinned by an exact hand calculation or a closed form, by the mathematical
properties of the family, and by the limit in which it reproduces the default scheme bit for bit."""
import json
import os
from fractions import Fraction

import numpy as np

import oracle
from paper_2309_06662_b200 import workloads as W
from util import box

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# =============================================================================================
# WENO-Z
# =============================================================================================
def test_wenoz_matches_exact_rational_hand_calculation():
    """golden/wenoz_worked.json, written by tests/golden/make_wenoz_worked.py with python Fractions (imports no
    implementation): Borges et al. (2008) weights on the Jiang-Shu candidates, eps = 1e-6 exactly."""
    with open(os.path.join(GOLD, "wenoz_worked.json")) as fh:
        cases = json.load(fh)["cases"]
    assert len(cases) >= 8
    for c in cases:
        exact = Fraction(int(c["num"]), int(c["den"]))
        got = oracle.weno(c["cells"], c["order"], c["vel"], scheme=1)
        assert abs(got - float(exact)) <= 4e-15 * max(1.0, abs(float(exact))), c
    # and it is a different scheme from Jiang-Shu on non-smooth data
    assert abs(oracle.weno([1, 2, 4, 8, 16, 32], 3, 1, scheme=1) - oracle.weno([1, 2, 4, 8, 16, 32], 3, 1, scheme=0)) > 1e-3


def test_wenoz_is_exact_on_quadratics_and_linears_and_mirror_symmetric():
    rng = np.random.default_rng(3)
    for _ in range(50):
        a, b, c = rng.standard_normal(3) * (1.0, 3.0, 2.0)
        F = lambda x: a * x + b * x * x / 2 + c * x ** 3 / 3          # noqa: E731  antiderivative of the quadratic
        avg = np.array([F(m + 1.0) - F(m + 0.0) for m in range(-3, 3)])   # unit cells -3..2, face at x = 0
        for vel in (1.0, -1.0):
            assert abs(oracle.weno(avg, 3, vel, 1) - a) < 1e-12 * (1 + abs(a) + abs(b) + abs(c))
        lin = np.array([a * (m + 0.5) + b for m in range(-3, 3)])
        for vel in (1.0, -1.0):
            assert abs(oracle.weno(lin, 2, vel, 1) - b) < 1e-13 * (1 + abs(a) + abs(b))
        cells = rng.standard_normal(6)
        for order in (1, 2, 3):
            assert oracle.weno(cells, order, 1.0, 1) == oracle.weno(cells[::-1].copy(), order, -1.0, 1)
        assert oracle.weno(np.full(6, 4.25), 3, 1.0, 1) == 4.25


def test_wenoz_is_closer_to_the_linear_scheme_on_smooth_data_and_fifth_order():
    """The point of the Z weights: on smooth data they stay closer to the linear fifth-order weights than Jiang-Shu's, so the
    error against the exact face value is smaller at every resolution; at a step both fall back to the smooth side."""
    A = 1000.0                              # beta >> eps at every resolution used

    def errs(N, scheme):
        h = 2 * np.pi / N
        xs = np.arange(-4, N + 4) * h
        avg = A * (np.cos(xs[:-1]) - np.cos(xs[1:])) / h
        return max(abs(oracle.weno(avg[n - 3:n + 3], 3, 1.0, scheme) - A * np.sin(xs[n])) for n in range(4, N + 3))
    prev = None
    for N in (32, 64, 128):
        ejs, ez = errs(N, 0), errs(N, 1)
        assert ez < 0.5 * ejs, (N, ejs, ez)
        if prev is not None:
            assert np.log2(prev / ez) > 4.8, (N, prev, ez)
        prev = ez
    # essentially non-oscillatory at a step, from both sides
    assert abs(oracle.weno([0, 0, 0, 1, 1, 1], 3, 1.0, 1)) < 1e-10 and abs(oracle.weno([0, 0, 0, 1, 1, 1], 3, -1.0, 1) - 1) < 1e-10


def test_wenoz_model_conserves_tracers_and_differs_from_js():
    wl = W.with_weno_z(W.config2(nx=72, ny=30, nz=12, steps=10))
    rng = np.random.default_rng(1)
    wl["fields"]["u"] = 0.2 * rng.standard_normal(wl["fields"]["u"].shape)
    wl["fields"]["v"] = 0.2 * rng.standard_normal(wl["fields"]["v"].shape)
    m = oracle.RefModel(wl)
    vol = m.grid.masks()["wet"] * np.diff(wl["z_faces"])[:, None, None] * m.grid.metrics()["AzC"][None, :, None]
    f0 = m.get_fields()
    m.step(10)
    f1 = m.get_fields()
    for n in "TS":
        assert abs(np.sum(vol * f1[n]) / np.sum(vol * f0[n]) - 1.0) < 2e-14
    wl0 = dict(wl, params=dict(wl["params"], advection=0))
    m0 = oracle.RefModel(wl0)
    m0.step(10)
    assert np.abs(m0.get_fields()["T"] - f1["T"]).max() > 1e-6


# =============================================================================================
# nonlinear equation of state
# =============================================================================================
def test_nonlinear_eos_with_zero_coefficients_is_the_linear_one_bit_for_bit():
    wl = W.config2(nx=48, ny=20, nz=10, steps=4)
    a = oracle.RefModel(wl)
    b = oracle.RefModel(W.with_nonlinear_eos(dict(wl, params=dict(wl["params"])), alpha2=0.0, gamma=0.0))
    a.step(4); b.step(4)
    fa, fb = a.get_fields(), b.get_fields()
    for n in ("u", "v", "w", "eta", "T", "S"):
        assert np.array_equal(fa[n], fb[n]), n


def test_nonlinear_eos_pressure_closed_form_thermobaric_and_cabbeling():
    """A column with a depth-independent anomaly dT: b(z) = g [alpha (1 - gamma z) dT + alpha2/2 dT^2] is linear in z, the
    trapezoid rule between centres is exact for it, and the top half cell uses b at the top centre:
        p(z_k) = b(z_t) z_t - [B(z_t) - B(z_k)],   B'(z) = b(z),  z_t = centre of the top cell."""
    nz = 7
    zf = W.geometric_z_faces(nz, 20.0, 1500.0)
    wl = W.with_nonlinear_eos(box(nx=6, ny=5, nz=nz, depth=1500.0, z_faces=zf), alpha2=1.3e-5, gamma=2.5e-4)
    dT = 3.5
    wl["fields"]["T"][:] = 10.0 + dT
    P = wl["params"]
    m = oracle.RefModel(wl)
    p = m.diagnostics()["p"][:, 2, 3]
    zc = 0.5 * (zf[1:] + zf[:-1])
    g, al, a2, ga = P["g"], P["alpha"], P["eos_alpha2"], P["eos_gamma"]
    b = lambda z: g * (al * (1 - ga * z) * dT + 0.5 * a2 * dT * dT)                    # noqa: E731
    B = lambda z: g * (al * dT * (z - ga * z * z / 2) + 0.5 * a2 * dT * dT * z)       # noqa: E731
    zt = zc[-1]
    want = b(zt) * zt - (B(zt) - B(zc))
    assert np.max(np.abs(p - want)) < 1e-13 * np.max(np.abs(want))
    # thermobaricity: the same temperature contrast pushes harder at depth.  T = T0 + s i: at rest
    # G_u = -(p[i] - p[i-1]) / dx = -(s / dT) want(z_k) / dx for the linear part, the cabbeling part grows with i
    wl2 = W.with_nonlinear_eos(box(nx=6, ny=5, nz=nz, depth=1500.0, z_faces=zf, periodic=(0, 0)), alpha2=0.0, gamma=2.5e-4)
    s = 0.25
    wl2["fields"]["T"][:] = 10.0 + s * np.arange(6)[None, None, :]
    Gu = oracle.RefModel(wl2).tendencies()["Gu"]
    lin = g * al * s * (zt * (1 - ga * zt) - ((zt - ga * zt * zt / 2) - (zc - ga * zc * zc / 2)))      # d p / d i
    assert np.max(np.abs(Gu[:, 2, 1:] + lin[:, None] / 1000.0)) < 1e-12 * np.max(np.abs(lin)) / 1000.0
    assert abs(Gu[0, 2, 3]) > 1.12 * abs(g * al * s * zc[0] / 1000.0)                 # stronger than the linear EOS at depth


def test_cabbeling_mixing_two_parcels_makes_denser_water():
    """alpha2 > 0 makes b convex in T: the mixture of two parcels is less buoyant than the mean of their buoyancies.  Seen
    through the hydrostatic pressure of three one-column states (the top-cell rule p = -b (0 - z_t))."""
    nz = 4
    zf = np.array([-400.0, -300.0, -200.0, -100.0, 0.0])

    def top_b(T):
        wl = W.with_nonlinear_eos(box(nx=4, ny=4, nz=nz, depth=400.0, z_faces=zf), alpha2=1e-5, gamma=0.0)
        wl["fields"]["T"][:] = T
        return oracle.RefModel(wl).diagnostics()["p"][-1, 0, 0] / (-50.0)              # p_top = b z_t, z_t = -50
    b1, b2, bm = top_b(2.0), top_b(22.0), top_b(12.0)
    P = W._params(64, 1, 1, 0, 0)
    assert abs((0.5 * (b1 + b2) - bm) - P["g"] * 0.5 * 1e-5 * 100.0) < 1e-12          # g alpha2/2 ((dT1^2 + dT2^2)/2 - dTm^2) = g alpha2/2 * 100


# =============================================================================================
# separate filter weights for the barotropic transports
# =============================================================================================
def _other_weights(M, p=1, q=2):
    s = np.arange(1, M + 1) / (M + 1.0)
    b = s ** p * (1.0 - s ** q)
    return b / b.sum()


def test_transport_weights_equal_to_eta_weights_change_nothing():
    wl = W.config2(nx=48, ny=20, nz=10, steps=4)
    a, _ = oracle.filter_weights(wl["params"]["substeps"])
    m0, m1 = oracle.RefModel(wl), oracle.RefModel(wl, filter_weights_uv=a)
    m0.step(4); m1.step(4)
    f0, f1 = m0.get_fields(), m1.get_fields()
    for n in ("u", "v", "w", "eta", "T", "S"):
        assert np.array_equal(f0[n], f1[n]), n


def test_transport_weights_closed_form_uniform_wind_on_a_flat_periodic_box():
    """Flat doubly periodic box at rest, f = 0, uniform wind stress: G^U = tau / rho0 everywhere, eta stays flat, so
    U^m = m dtau G^U and the filtered transport is dtau G^U sum_m m b_m (Euler first step) - it tells b from a, whose first
    moment is dt / dtau by construction; eta-bar stays exactly 0 and the corrected u has the depth mean U-bar / H."""
    M, dt, H = 12, 100.0, 400.0
    wl = box(nx=8, ny=6, nz=4, depth=H, f0=0.0, dt=dt, substeps=M, nu_z=0.0)
    wl["fields"]["tau_x"][:] = 0.2
    a, ratio = oracle.filter_weights(M)
    b = _other_weights(M)
    assert abs(np.dot(np.arange(1, M + 1), b) - np.dot(np.arange(1, M + 1), a)) > 0.3
    for weights, moment in ((None, 1.0 / ratio), (b, float(np.dot(np.arange(1, M + 1), b)))):
        m = oracle.RefModel(wl, filter_weights_uv=weights)
        m.step(1)
        U = m.diagnostics()["U"]
        want = (dt * ratio) * (0.2 / wl["params"]["rho0"]) * moment
        assert np.max(np.abs(U - want)) < 1e-14 * want, (weights is None, U[0, 0], want)
        f = m.get_fields()
        assert np.all(f["eta"] == 0.0) and np.all(f["v"] == 0.0)
        dz = np.diff(wl["z_faces"])
        assert np.max(np.abs((f["u"] * dz[:, None, None]).sum(axis=0) - want)) < 1e-13 * want


def test_user_filter_weights_set_the_sub_step_so_that_the_average_lands_on_the_new_time_level():
    """The same box with the caller's own weights a_m for everything (filter_weights): the sub-step is dt / sum_m m a_m
    (the weighted mean of the sub-step times is t^{n+1}), so the filtered transport of the uniformly forced
    ocean is exactly dt G^U whatever the weights are — with dtau = dt / sum_m a_m it would be dt G^U times their first moment."""
    M, dt, H = 12, 100.0, 400.0
    wl = box(nx=8, ny=6, nz=4, depth=H, f0=0.0, dt=dt, substeps=M, nu_z=0.0)
    wl["fields"]["tau_x"][:] = 0.2
    want = dt * 0.2 / wl["params"]["rho0"]
    for a in (_other_weights(M), np.eye(M)[M - 1], np.eye(M)[2]):       # spread out, all on the last sub-step, all on the third
        assert abs(np.dot(np.arange(1, M + 1), a) - 1.0) > 0.5
        m = oracle.RefModel(wl, filter_weights=a)
        m.step(1)
        U = m.diagnostics()["U"]
        assert np.max(np.abs(U - want)) < 1e-13 * want, (a, U[0, 0], want)


def test_transport_weights_leave_eta_filter_and_tracers_alone_but_change_the_flow():
    wl = W.config2(nx=48, ny=20, nz=10, steps=3)
    b = _other_weights(wl["params"]["substeps"])
    m0, m1 = oracle.RefModel(wl), oracle.RefModel(wl, filter_weights_uv=b)
    m0.step(1); m1.step(1)
    f0, f1 = m0.get_fields(), m1.get_fields()
    assert np.array_equal(f0["eta"], f1["eta"]) and np.array_equal(f0["T"], f1["T"])     # first step: eta-bar and T do not see U-bar
    assert np.abs(f0["u"] - f1["u"]).max() > 1e-9


# =============================================================================================
# biharmonic horizontal dissipation
# =============================================================================================
def test_biharmonic_with_zero_coefficients_changes_nothing():
    wl = W.config2(nx=48, ny=20, nz=10, steps=3)
    w0 = dict(wl, params=dict(wl["params"], nu4_h=0.0, kappa4_h=0.0))
    a, b = oracle.RefModel(wl), oracle.RefModel(w0)
    a.step(3); b.step(3)
    fa, fb = a.get_fields(), b.get_fields()
    for n in ("u", "v", "w", "eta", "T", "S"):
        assert np.array_equal(fa[n], fb[n]), n


def test_biharmonic_plane_waves_closed_form_on_a_periodic_box():
    """On a uniform doubly periodic box the discrete Laplacian of cos(k x) cos(l y) is lam * itself with
    lam = -(4/dx^2) sin^2(k dx/2) - (4/dy^2) sin^2(l dy/2); applied twice: the biharmonic tendency is -coef * lam^2 * field.
    Isolated as the difference between a model with and one without the term (everything else is identical)."""
    nx, ny, nz, dx, dy = 16, 12, 3, 2000.0, 3000.0
    x = (np.arange(nx) + 0.5) * dx; xf = np.arange(nx) * dx
    y = (np.arange(ny) + 0.5) * dy; yf = np.arange(ny) * dy
    kx, ly = 2 * np.pi * 2 / (nx * dx), 2 * np.pi * 1 / (ny * dy)
    lam = -(4 / dx ** 2) * np.sin(kx * dx / 2) ** 2 - (4 / dy ** 2) * np.sin(ly * dy / 2) ** 2
    nu4, k4 = 3.0e9, 1.5e9

    def models(**fields):
        out = []
        for on in (0, 1):
            wl = box(nx=nx, ny=ny, nz=nz, depth=300.0, dx=dx, dy=dy, f0=1e-4, nu_h=7.0, kappa_h=2.0,
                     nu4_h=on * nu4, kappa4_h=on * k4)
            for n, v in fields.items():
                wl["fields"][n] = np.broadcast_to(v, (nz, ny, nx)).copy()
            out.append(oracle.RefModel(wl).tendencies())
        return out
    c = 10.0 + 0.5 * np.cos(kx * x)[None, :] * np.cos(ly * y)[:, None]
    u = 0.3 * np.cos(kx * xf)[None, :] * np.cos(ly * y)[:, None]            # u lives on west faces, v on south faces
    v = 0.2 * np.cos(kx * x)[None, :] * np.cos(ly * yf)[:, None]
    G0, G1 = models(T=c, S=35.0 - 0.1 * (c - 10.0), u=u, v=v)
    for n, f, coef in (("GT", c - 10.0, k4), ("GS", -0.1 * (c - 10.0), k4), ("Gu", u, nu4), ("Gv", v, nu4)):
        got = (G1[n] - G0[n])[1]
        want = -coef * lam ** 2 * f
        assert np.max(np.abs(got - want)) < 2e-9 * np.max(np.abs(want)), n      # difference of two O(1e-5..1e-3) tendencies
    assert np.max(np.abs(-k4 * lam ** 2 * 0.5)) > 1e-8


def _laplacians_from_the_pinned_second_order_terms(wl):
    """L(u, v) and L(c) of a state obtained from the Laplacian viscosity / diffusion terms, which the lat-lon hand evaluator
    of tests/test_oracle_latlon.py pins: G(coefficient 1) - G(coefficient 0) with the flow frozen."""
    def G(nu_h, kappa_h):
        w = dict(wl, params=dict(wl["params"], nu_h=nu_h, kappa_h=kappa_h, nu4_h=0.0, kappa4_h=0.0))
        return oracle.RefModel(w).tendencies()
    a, b = G(1.0, 1.0), G(0.0, 0.0)
    return {n: a[n] - b[n] for n in a}


def test_biharmonic_is_the_pinned_laplacian_applied_twice_on_the_sphere_with_land():
    """<a, L b> = <L a, b> for the masked C-grid Laplacians on a lat-lon grid with land (sum by parts; areas dxC dy for u,
    dxF dy for v, AzC for tracers), so  sum u . B(u) dA = -nu4 sum |L u|^2 dA  with L taken from the ALREADY PINNED
    second-order term: a metric factor of the wrong row or a dropped mask in the second application breaks the identity."""
    wl = W.config2(nx=40, ny=28, nz=5, steps=1)
    rng = np.random.default_rng(12)
    for n, amp in (("u", 0.3), ("v", 0.3), ("T", 2.0), ("S", 0.5)):
        wl["fields"][n] = wl["fields"][n] + amp * rng.standard_normal(wl["fields"][n].shape)
    wl["params"].update(nu_h=0.0, kappa_h=0.0)
    L = _laplacians_from_the_pinned_second_order_terms(wl)
    nu4, k4 = 2.0e12, 1.0e12
    w1 = dict(wl, params=dict(wl["params"], nu4_h=nu4, kappa4_h=k4))
    m0, m1 = oracle.RefModel(wl), oracle.RefModel(w1)
    G0, G1, st = m0.tendencies(), m1.tendencies(), m0.get_fields()            # st: masked state
    B = {n: G1[n] - G0[n] for n in G0}
    g = wl["grid"]
    a, dlam, dphi = g["radius"], np.deg2rad(g["dx"]), np.deg2rad(g["dy"])
    pf = np.deg2rad(g["y0"] + np.arange(g["ny"] + 1) * g["dy"]); pc = 0.5 * (pf[1:] + pf[:-1])
    Au = (a * np.cos(pc) * dlam * a * dphi)[None, :, None]
    Av = (a * np.cos(pf[:-1]) * dlam * a * dphi)[None, :, None]
    Ac = (a * a * dlam * (np.sin(pf[1:]) - np.sin(pf[:-1])))[None, :, None]
    lhs = np.sum(st["u"] * B["Gu"] * Au + st["v"] * B["Gv"] * Av)
    rhs = -nu4 * np.sum(L["Gu"] ** 2 * Au + L["Gv"] ** 2 * Av)
    assert rhs < 0 and abs(lhs - rhs) < 1e-9 * abs(rhs), (lhs, rhs)
    wet = m0.grid.masks()["wet"]
    for n, c, c0 in (("GT", "T", 10.0), ("GS", "S", 35.0)):
        # sum B A = 0 (flux form), so the constant part of the tracer drops out: take it out before it costs digits
        lhs = np.sum((st[c] - c0) * wet * B[n] * Ac)
        rhs = -k4 * np.sum(L[n] ** 2 * Ac)
        assert abs(np.sum(B[n] * Ac)) < 1e-10 * np.sum(np.abs(B[n]) * Ac)       # B is a difference of two rounded tendencies
        assert rhs < 0 and abs(lhs - rhs) < 1e-8 * abs(rhs), (n, lhs, rhs)
    # and cross-wise with another field (symmetry, not only the quadratic form): <w, B(u)> = -nu4 <L w, L u>
    wl2 = clone_fields(wl, rng)
    L2 = _laplacians_from_the_pinned_second_order_terms(wl2)
    st2 = oracle.RefModel(wl2).get_fields()
    lhs = np.sum(st2["u"] * B["Gu"] * Au + st2["v"] * B["Gv"] * Av)
    rhs = -nu4 * np.sum(L2["Gu"] * L["Gu"] * Au + L2["Gv"] * L["Gv"] * Av)
    assert abs(lhs - rhs) < 1e-9 * abs(rhs), (lhs, rhs)
    lhs = np.sum((st2["T"] - 10.0) * wet * B["GT"] * Ac); rhs = -k4 * np.sum(L2["GT"] * L["GT"] * Ac)
    assert abs(lhs - rhs) < 1e-8 * abs(rhs)


def clone_fields(wl, rng):
    w = dict(wl, fields={k: v.copy() for k, v in wl["fields"].items()})
    for n, amp in (("u", 0.3), ("v", 0.3), ("T", 2.0)):
        w["fields"][n] = w["fields"][n] + amp * rng.standard_normal(w["fields"][n].shape)
    return w


def test_biharmonic_diffusion_conserves_tracers_and_damps_grid_noise():
    wl = W.config2(nx=48, ny=24, nz=6, steps=8)
    rng = np.random.default_rng(4)
    wl["fields"]["T"] = wl["fields"]["T"] + 0.5 * rng.standard_normal(wl["fields"]["T"].shape)
    dxmin = wl["grid"]["radius"] * np.deg2rad(wl["grid"]["dx"]) * np.cos(np.deg2rad(75.0))
    k4 = 0.01 * dxmin ** 4 / wl["params"]["dt"]                                   # well inside the explicit stability limit
    wl["params"].update(kappa_h=0.0, kappa4_h=k4, nu4_h=k4)
    m = oracle.RefModel(wl)
    vol = m.grid.masks()["wet"] * np.diff(wl["z_faces"])[:, None, None] * m.grid.metrics()["AzC"][None, :, None]
    f0 = m.get_fields()
    m.step(8)
    f1 = m.get_fields()
    for n in "TS":
        assert abs(np.sum(vol * f1[n]) / np.sum(vol * f0[n]) - 1.0) < 2e-14, n
    # grid-scale roughness along x in the polar rows (where dx is smallest and the coefficient bites), over wet triples only
    wet = m.grid.masks()["wet"].astype(bool)
    ok = (wet[:, :, 2:] & wet[:, :, 1:-1] & wet[:, :, :-2])
    rows = np.r_[0:3, 21:24]
    lap = lambda a: np.abs(a[:, :, 2:] - 2 * a[:, :, 1:-1] + a[:, :, :-2])[:, rows][ok[:, rows]].mean()      # noqa: E731
    ref = dict(wl, params=dict(wl["params"], kappa4_h=0.0, nu4_h=0.0))
    r = oracle.RefModel(ref); r.step(8)
    assert ok[:, rows].sum() > 100 and lap(f1["T"]) < 0.9 * lap(r.get_fields()["T"])
