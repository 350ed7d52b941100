"""Pins of the whole oracle step against what the physics fixes (north_star's five checks plus
closed forms of DESIGN.md §5): rest state, tracer conservation, gravity-wave speed and the
sub-step closed form, geostrophic balance, inertial oscillation under AB2, the barotropic
correction, and closed forms for w and p."""
import numpy as np
import pytest

import oracle
from paper_2309_06662_b200 import workloads as W
from util import box

G = W.GRAVITY


# ---------------------------------------------------------------- (i) rest stays at rest ------
def test_rest_state_flat_bottom_stratified_exactly_zero():
    wl = box(nx=12, ny=10, nz=8, depth=800.0, f0=1e-4, nu_h=50.0, kappa_h=5.0)
    zc = 0.5 * (wl["z_faces"][:-1] + wl["z_faces"][1:])
    wl["fields"]["T"] = np.broadcast_to((2 + 18 * np.exp(zc / 300.0))[:, None, None], (8, 10, 12)).copy()
    wl["fields"]["S"] = np.broadcast_to((35 - np.exp(zc / 200.0))[:, None, None], (8, 10, 12)).copy()
    m = oracle.RefModel(wl)
    m.step(5)
    f = m.get_fields()
    for n in ("u", "v", "w", "eta"):
        assert np.all(f[n] == 0.0), n
    # tracers only diffuse vertically: horizontally uniform still
    assert np.all(f["T"] == f["T"][:, :1, :1])


def test_rest_state_with_bathymetry_and_no_vertical_diffusion_exactly_zero():
    wl = W.config2(nx=48, ny=20, nz=10, steps=1)
    wl["params"].update(kappa_z=0.0, nu_z=0.0)
    zc = 0.5 * (wl["z_faces"][:-1] + wl["z_faces"][1:])
    wl["fields"]["T"] = np.broadcast_to((2 + 18 * np.exp(zc / 800.0))[:, None, None], (10, 20, 48)).copy()
    wl["fields"]["S"] = np.broadcast_to((35 - np.exp(zc / 500.0))[:, None, None], (10, 20, 48)).copy()
    wl["fields"]["tau_x"][:] = 0.0
    wl["fields"]["tau_y"][:] = 0.0
    m = oracle.RefModel(wl)
    assert 0.15 < 1.0 - m.grid.masks()["wet"][-1].mean() < 0.6       # there is land
    m.step(3)
    f = m.get_fields()
    for n in ("u", "v", "w", "eta"):
        assert np.all(f[n] == 0.0), n


# ------------------------------------------------------- (ii) tracer volume integrals kept ----
def _volume(wl, g):
    dz = np.diff(wl["z_faces"])
    return g.masks()["wet"] * dz[:, None, None] * g.metrics()["AzC"][None, :, None]


def test_tracer_conservation_latlon_with_land():
    wl = W.config2(nx=72, ny=30, nz=12, steps=20)
    m = oracle.RefModel(wl)
    vol = _volume(wl, m.grid)
    f0 = m.get_fields()
    I0 = {n: np.sum(vol * f0[n]) for n in "TS"}
    m.step(20)
    f1 = m.get_fields()
    assert np.abs(f1["u"]).max() > 1e-3                        # something happened
    for n in "TS":
        assert abs(np.sum(vol * f1[n]) / I0[n] - 1.0) < 2e-14, n


def test_tracer_conservation_periodic_box():
    wl = W.config0(nx=16, ny=16, nz=6)
    m = oracle.RefModel(wl)
    vol = _volume(wl, m.grid)
    I0 = np.sum(vol * m.get_fields()["T"])
    m.step(40)
    assert abs(np.sum(vol * m.get_fields()["T"]) / I0 - 1.0) < 2e-14


# ----------------------------------------------------- (iii) barotropic mode: sqrt(gH) --------
def test_barotropic_substep_plane_wave_closed_form():
    # forward-backward sub-step of a plane wave on a flat periodic box, U0 = V0 = 0, f = 0:
    #   eta^m = eta0 cos((m - 1/2) theta) / cos(theta/2),  theta = 2 asin(s/2),
    #   s^2 = g H dtau^2 [ (4/dx^2) sin^2(k dx/2) + (4/dy^2) sin^2(l dy/2) ]
    nx, ny, dx, dy, H = 16, 12, 2000.0, 3000.0, 400.0
    wl = box(nx=nx, ny=ny, nz=2, depth=H, dx=dx, dy=dy, f0=0.0)
    kx, ly = 2 * np.pi * 2 / (nx * dx), 2 * np.pi * 1 / (ny * dy)
    x = (np.arange(nx) + 0.5) * dx
    y = (np.arange(ny) + 0.5) * dy
    eta0 = 0.3 * np.cos(kx * x[None, :] + ly * y[:, None])
    wl["fields"]["eta"] = eta0
    m = oracle.RefModel(wl)
    dtau = 11.0
    s2 = G * H * dtau ** 2 * ((4 / dx ** 2) * np.sin(kx * dx / 2) ** 2 + (4 / dy ** 2) * np.sin(ly * dy / 2) ** 2)
    theta = 2 * np.arcsin(np.sqrt(s2) / 2)
    done = 0
    for mm in (1, 2, 7, 50, 200):
        m.barotropic_raw(mm - done, dtau)
        done = mm
        eta = m.get_fields()["eta"]
        want = eta0 * np.cos((mm - 0.5) * theta) / np.cos(theta / 2)
        assert np.max(np.abs(eta - want)) < 2e-14, mm
    # theta/dtau -> sqrt(gH)|k| as dx, dtau -> 0
    kk = np.hypot(kx, ly)
    assert abs(theta / dtau / (np.sqrt(G * H) * kk) - 1.0) < 0.03


def test_split_step_gravity_wave_period():
    # standing wave, L = 128 km, H = 400 m, full split-explicit step: period ~ L / sqrt(gH)
    nx, dx, H, dt = 64, 2000.0, 400.0, 20.0
    # alpha = beta_s = 0: pure barotropic mode.  (With the EOS on, the zero-top-flux reading of
    # DESIGN.md §3.10 lets eta imprint a tracer anomaly on the top cell, which shifts the speed by
    # ~ (beta_s*S0 - alpha*T0)/2 ~ 1.5 %: a property of that reading, listed in DESIGN.md §3.)
    wl = box(nx=nx, ny=4, nz=4, depth=H, dx=dx, f0=0.0, dt=dt, substeps=20, alpha=0.0, beta_s=0.0)
    L = nx * dx
    x = (np.arange(nx) + 0.5) * dx
    wl["fields"]["eta"] = np.broadcast_to(0.01 * np.cos(2 * np.pi * x / L)[None, :], (4, nx)).copy()
    m = oracle.RefModel(wl)
    period = L / np.sqrt(G * H)
    nsteps = int(2.2 * period / dt)
    a = np.empty(nsteps + 1)
    a[0] = 0.01
    amp_proj = np.cos(2 * np.pi * x / L)
    for n in range(1, nsteps + 1):
        m.step(1)
        a[n] = 2.0 * np.mean(m.get_fields()["eta"][0] * amp_proj)
    t = dt * np.arange(nsteps + 1)
    sign = np.sign(a)
    cross = np.where(sign[1:] * sign[:-1] < 0)[0]
    tc = t[cross] - a[cross] * dt / (a[cross + 1] - a[cross])          # linear interpolation
    measured = 2.0 * np.mean(np.diff(tc))
    assert abs(measured / period - 1.0) < 1e-3            # (k dx)^2/24 = 4e-4 grid dispersion
    # filter damping is mild: amplitude after two periods stays within (0.7, 1.0) of the start
    n2 = int(round(2 * measured / dt))
    assert 0.7 < abs(a[n2]) / 0.01 < 1.0


# ----------------------------------------------------- (iv) geostrophic balance is steady -----
def test_geostrophic_state_steady_to_second_order():
    L, H, f0, eta_amp, dt = 256e3, 400.0, 1e-4, 0.1, 20.0
    drift = []
    for nx in (16, 32, 64):
        dx = L / nx
        wl = box(nx=nx, ny=4, nz=2, depth=H, dx=dx, dy=dx, f0=f0, dt=dt, substeps=20)
        k = 2 * np.pi / L
        xc = (np.arange(nx) + 0.5) * dx
        wl["fields"]["eta"] = np.broadcast_to(eta_amp * np.cos(k * xc)[None, :], (4, nx)).copy()
        v0 = -G * eta_amp * k * np.sin(k * xc) / f0                      # v = g eta_x / f at x centres
        wl["fields"]["v"] = np.broadcast_to(v0[None, None, :], (2, 4, nx)).copy()
        m = oracle.RefModel(wl)
        m.step(20)
        f = m.get_fields()
        drift.append(max(np.abs(f["v"] - v0[None, None, :]).max(), np.abs(f["u"]).max()))
    assert drift[0] < 2e-4                                  # 0.05 % of max |v| = 0.24 at nx = 16
    assert 3.0 < drift[0] / drift[1] < 5.5 and 3.0 < drift[1] / drift[2] < 5.5


# ------------------------------------------- Coriolis + quasi-AB2 on a uniform flow -----------
def test_inertial_oscillation_obeys_ab2_recurrence():
    f0, dt, chi = 1.2e-4, 300.0, 0.1
    wl = box(nx=8, ny=8, nz=3, depth=300.0, f0=f0, dt=dt, substeps=10, nu_z=1e-4)
    wl["fields"]["u"][:] = 0.3
    wl["fields"]["v"][:] = -0.1
    m = oracle.RefModel(wl)
    z = -1j * f0 * dt
    q_prev, q = None, 0.3 - 0.1j
    for n in range(50):
        m.step(1)
        if q_prev is None:
            q_prev, q = q, q + z * q                                    # Euler start
        else:
            q_prev, q = q, q + z * ((1.5 + chi) * q - (0.5 + chi) * q_prev)
    f = m.get_fields()
    assert np.max(np.abs(f["u"] - q.real)) < 1e-13 and np.max(np.abs(f["v"] - q.imag)) < 1e-13
    assert np.all(f["eta"] == 0.0) or np.abs(f["eta"]).max() < 1e-15


# ---------------------------------------------------------- barotropic correction -------------
def test_correction_makes_depth_integral_equal_filtered_transport():
    wl = W.config2(nx=48, ny=24, nz=10, steps=5)
    m = oracle.RefModel(wl)
    m.step(5)
    f, d = m.get_fields(), m.diagnostics()
    dz = np.diff(wl["z_faces"])[:, None, None]
    scale = np.abs(d["U"]).max()
    assert scale > 0
    assert np.abs((f["u"] * dz).sum(0) - d["U"]).max() < 1e-13 * scale
    assert np.abs((f["v"] * dz).sum(0) - d["V"]).max() < 1e-13 * max(scale, np.abs(d["V"]).max())


# ---------------------------------------------------------- diagnostics: w and p --------------
def test_w_closed_form_linear_u_and_surface_value():
    nx, ny, nz = 12, 10, 5
    wl = box(nx=nx, ny=ny, nz=nz, depth=500.0, periodic=(0, 0), dx=1000.0)
    a = 1e-5
    xf = 1000.0 * np.arange(nx)
    wl["fields"]["u"] = np.broadcast_to((a * xf)[None, None, :], (nz, ny, nx)).copy()
    m = oracle.RefModel(wl)
    w = m.get_fields()["w"]
    zf = wl["z_faces"]
    want = -a * (zf - zf[0])
    inner = w[:, 2:-2, 2:-2]                                     # away from the walls D = a
    assert np.max(np.abs(inner - want[:, None, None])) < 1e-14 * np.abs(want).max()
    # w[Nz] * Az = -div(U, V) for arbitrary flow (periodic box)
    wl = W.config0(nx=8, ny=8, nz=4)
    m = oracle.RefModel(wl)
    d, f = m.diagnostics(), m.get_fields()
    U, V = d["U"], d["V"]
    div = 1000.0 * (np.roll(U, -1, 1) - U) + 1000.0 * (np.roll(V, -1, 0) - V)
    assert np.max(np.abs(f["w"][-1] * 1e6 + div)) < 1e-9 * np.abs(div).max()
    assert np.all(f["w"][0] == 0.0)


def test_p_exact_for_linear_buoyancy():
    nz = 9
    zf = W.geometric_z_faces(nz, 10.0, 900.0)
    wl = box(nx=4, ny=4, nz=nz, depth=900.0, z_faces=zf)
    zc = 0.5 * (zf[:-1] + zf[1:])
    c = 0.01
    wl["fields"]["T"] = np.broadcast_to((10.0 + c * zc)[:, None, None], (nz, 4, 4)).copy()
    wl["fields"]["S"] = np.full((nz, 4, 4), 35.0)
    m = oracle.RefModel(wl)
    p = m.diagnostics()["p"][:, 1, 2]
    ga = G * wl["params"]["alpha"]
    b_top = ga * c * zc[-1]
    assert abs(p[-1] - (-b_top * (0.0 - zc[-1]))) < 1e-16
    want = p[-1] - ga * c * (zc[-1] ** 2 - zc ** 2) / 2.0          # trapezoid is exact for linear b
    assert np.max(np.abs(p - want)) < 1e-13 * np.abs(want).max()
    # salinity enters with the opposite sign
    wl["fields"]["T"][:] = 10.0
    wl["fields"]["S"][:] = 36.0
    m = oracle.RefModel(wl)
    p = m.diagnostics()["p"][:, 0, 0]
    bS = -G * wl["params"]["beta_s"] * 1.0
    assert np.max(np.abs(p - bS * zc)) < 1e-12 * abs(bS * zc[0])
