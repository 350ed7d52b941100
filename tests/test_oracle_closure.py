"""Pins of the oracle's Ri-based vertical mixing closure against
closed forms, dense linear algebra and conservation — none re-types the oracle's loop."""
import numpy as np
import pytest

import oracle
from paper_2309_06662_b200 import workloads as W
from util import box, clone

G, ALPHA = W.GRAVITY, 2e-4
RI = dict(closure=1, ri_nu0=5e-3, ri_c=5.0, ri_kconv=0.1, ri_n2c=1e-6, ri_s2min=1e-10)


# ------------------------------------------------------------ variable-kappa Thomas solve ----
def _dense_matrix_var(zf, open_faces, dtk):
    """independent dense assembly A = I - Dz^-1 Gt diag(dt kappa_face) Dzc^-1 G (flux form)"""
    nz = len(zf) - 1
    dz = np.diff(zf)
    zc = 0.5 * (zf[:-1] + zf[1:])
    Gm = np.zeros((nz + 1, nz))
    for k in range(1, nz):
        if open_faces[k]:
            Gm[k, k] = 1.0 / (zc[k] - zc[k - 1])
            Gm[k, k - 1] = -1.0 / (zc[k] - zc[k - 1])
    Dv = np.zeros((nz, nz + 1))
    for k in range(nz):
        Dv[k, k + 1] = 1.0 / dz[k]
        Dv[k, k] = -1.0 / dz[k]
    return np.eye(nz) - Dv @ np.diag(dtk) @ Gm


def test_variable_kappa_column_matches_dense_solve_and_conserves():
    rng = np.random.default_rng(14)
    for nz in (2, 3, 9, 20):
        zf = -np.cumsum(rng.uniform(5, 50, nz + 1))[::-1]
        zf -= zf[-1]
        open_faces = np.ones(nz + 1, np.uint8)
        open_faces[0] = open_faces[nz] = 0
        if nz > 4:
            open_faces[3] = 0
        dtk = 300.0 * 10.0 ** rng.uniform(-5, -1, nz + 1)          # four decades of diffusivity
        phi = rng.standard_normal(nz)
        want = np.linalg.solve(_dense_matrix_var(zf, open_faces, dtk * open_faces), phi)
        got = oracle.implicit_column_var(zf, open_faces, dtk, phi)
        assert np.max(np.abs(got - want)) < 1e-13
        assert abs(np.sum(np.diff(zf) * (got - phi))) < 1e-12      # no-flux ends: integral kept


def test_variable_kappa_column_with_constant_array_is_the_constant_solve_bitwise():
    rng = np.random.default_rng(15)
    nz = 11
    zf = W.geometric_z_faces(nz, 10.0, 900.0)
    open_faces = np.ones(nz + 1, np.uint8)
    phi = rng.standard_normal(nz)
    a = oracle.implicit_column(zf, open_faces, 0.37, phi)
    b = oracle.implicit_column_var(zf, open_faces, np.full(nz + 1, 0.37), phi)
    assert np.array_equal(a, b)


# ------------------------------------------------------------ the coefficients themselves ----
def _sheared_box(gamma, shear, nz=8, dz=10.0, **kw):
    """uniform layers; T = 10 + gamma z (K/m), u = shear z (1/s), horizontally uniform"""
    wl = box(nx=6, ny=5, nz=nz, depth=nz * dz, f0=0.0, nu_z=1e-4, kappa_z=1e-5, **RI, **kw)
    zc = 0.5 * (wl["z_faces"][:-1] + wl["z_faces"][1:])
    wl["fields"]["T"] = 10.0 + gamma * zc[:, None, None] + np.zeros_like(wl["fields"]["T"])
    wl["fields"]["u"] = shear * zc[:, None, None] + np.zeros_like(wl["fields"]["u"])
    return wl


@pytest.mark.parametrize("ri_target", [0.2, 1.0, 7.0])
def test_mixing_closed_form_at_prescribed_richardson_number(ri_target):
    # uniform shear s in u only and N2 = g alpha gamma: Ri = N2 / (s^2 + S2min) by construction
    gamma = 2e-3
    N2 = G * ALPHA * gamma
    s = np.sqrt(N2 / ri_target - RI["ri_s2min"])
    mix = oracle.RefModel(_sheared_box(gamma, s)).mixing()
    f = 1.0 / (1.0 + 5.0 * ri_target)
    assert np.all(mix["nu"][0] == 0.0) and np.all(mix["kappa"][0] == 0.0)      # bottom face closed
    assert np.allclose(mix["nu"][1:], 1e-4 + 5e-3 * f ** 2, rtol=1e-9, atol=0)
    assert np.allclose(mix["kappa"][1:], 1e-5 + 5e-3 * f ** 3, rtol=1e-9, atol=0)


def test_mixing_v_shear_counts_like_u_shear():
    gamma, s = 2e-3, 3e-3
    a = _sheared_box(gamma, s)
    b = _sheared_box(gamma, 0.0)
    b["fields"]["v"] = a["fields"]["u"].copy()
    ma, mb = oracle.RefModel(a).mixing(), oracle.RefModel(b).mixing()
    assert np.allclose(ma["nu"], mb["nu"], rtol=1e-12) and np.allclose(ma["kappa"], mb["kappa"], rtol=1e-12)


def test_mixing_takes_the_shear_from_the_four_faces_of_the_column():
    """Horizontally varying u, v (random, periodic box): S2 at tracer column (j, i) averages the squared shear of ITS west and
    east u faces (i, i + 1) and ITS south and north v faces (j, j + 1) — a face of a neighbouring column must not enter.
    Expected values from array shifts in numpy."""
    rng = np.random.default_rng(31)
    wl = _sheared_box(2e-3, 0.0)
    f = wl["fields"]
    f["u"] = 0.05 * rng.standard_normal(f["u"].shape)
    f["v"] = 0.05 * rng.standard_normal(f["v"].shape)
    mix = oracle.RefModel(wl).mixing()
    zc = 0.5 * (wl["z_faces"][:-1] + wl["z_faces"][1:])
    dzc = np.diff(zc)[:, None, None]
    du, dv = np.diff(f["u"], axis=0), np.diff(f["v"], axis=0)          # level k minus level k - 1, k = 1 .. nz - 1
    S2 = (0.5 * (du ** 2 + np.roll(du, -1, axis=2) ** 2) + 0.5 * (dv ** 2 + np.roll(dv, -1, axis=1) ** 2)) / dzc ** 2
    N2 = G * ALPHA * np.diff(f["T"], axis=0) / dzc
    ff = 1.0 / (1.0 + RI["ri_c"] * np.maximum(N2, 0.0) / (S2 + RI["ri_s2min"]))
    assert np.allclose(mix["nu"][1:], 1e-4 + RI["ri_nu0"] * ff ** 2, rtol=1e-12, atol=0)
    assert np.allclose(mix["kappa"][1:], 1e-5 + RI["ri_nu0"] * ff ** 3, rtol=1e-12, atol=0)
    assert ff.min() < 0.5 and ff.max() > 0.9                             # the case spans weak and strong mixing


def test_viscosity_at_a_velocity_face_is_the_mean_of_the_two_columns_that_share_it():
    """Stronger stratification in ONE tracer column (j0, i0) changes nu there and the pressure there, nothing else of state n.
    After one step the vertical structure of u (u minus its depth mean: the barotropic correction is depth independent)
    may therefore change only at the two u faces of that column, (j0, i0) and (j0, i0 + 1), and that of v only at
    (j0, i0) and (j0 + 1, i0) — the faces whose nu is the mean over the column and its west / south neighbour
    (DESIGN.md §3.12).  An average taken over the wrong pair of columns moves other faces."""
    gamma = 2e-3
    wl = _sheared_box(gamma, 2e-3)
    zc = 0.5 * (wl["z_faces"][:-1] + wl["z_faces"][1:])
    dz = np.diff(wl["z_faces"])[:, None, None]
    wl["fields"]["v"] = 1e-3 * zc[:, None, None] + np.zeros_like(wl["fields"]["v"])
    j0, i0 = 2, 3
    pert = clone(wl)
    pert["fields"]["T"][:, j0, i0] = 10.0 + 4.0 * gamma * zc

    def structure(wl_):
        m = oracle.RefModel(wl_)
        m.step(1)
        f = m.get_fields()
        return [f[n] - (dz * f[n]).sum(axis=0) / dz.sum() for n in ("u", "v")]

    (ua, va), (ub, vb) = structure(wl), structure(pert)
    du, dv = np.abs(ub - ua).max(axis=0), np.abs(vb - va).max(axis=0)
    moved_u = {(j0, i0), (j0, (i0 + 1) % du.shape[1])}
    moved_v = {(j0, i0), ((j0 + 1) % dv.shape[0], i0)}
    for j in range(du.shape[0]):
        for i in range(du.shape[1]):
            if (j, i) in moved_u:
                assert du[j, i] > 1e-9, (j, i, du[j, i])
            else:
                assert du[j, i] < 1e-15, (j, i, du[j, i])
            if (j, i) in moved_v:
                assert dv[j, i] > 1e-9, (j, i, dv[j, i])
            else:
                assert dv[j, i] < 1e-15, (j, i, dv[j, i])


def test_mixing_neutral_and_convective_limits():
    # neutral column: Ri = 0 whatever the shear -> nu_z + nu0, kappa_z + nu0
    mix = oracle.RefModel(_sheared_box(0.0, 4e-3)).mixing()
    assert np.allclose(mix["nu"][1:], 1e-4 + 5e-3, rtol=1e-12) and np.allclose(mix["kappa"][1:], 1e-5 + 5e-3, rtol=1e-12)
    # unstable by half the ramp width: conv = kconv / 2; by ten times the width: saturated at kconv
    for frac, conv in ((0.5, 0.05), (10.0, 0.1)):
        gamma = -frac * RI["ri_n2c"] / (G * ALPHA)
        mix = oracle.RefModel(_sheared_box(gamma, 1e-3)).mixing()
        assert np.allclose(mix["nu"][1:], 1e-4 + 5e-3 + conv, rtol=1e-6)
        assert np.allclose(mix["kappa"][1:], 1e-5 + 5e-3 + conv, rtol=1e-6)


def test_mixing_salinity_enters_with_the_opposite_sign():
    # S increasing upward is unstable (b = -g beta_s S'): same N2 magnitude as a T profile of gamma_T = -beta_s/alpha gamma_S
    wl = _sheared_box(0.0, 2e-3)
    zc = 0.5 * (wl["z_faces"][:-1] + wl["z_faces"][1:])
    gS = 1e-3
    wl["fields"]["S"] = 35.0 + gS * zc[:, None, None] + np.zeros_like(wl["fields"]["S"])
    ref = _sheared_box(-8e-4 / ALPHA * gS, 2e-3)
    a, b = oracle.RefModel(wl).mixing(), oracle.RefModel(ref).mixing()
    assert np.allclose(a["kappa"], b["kappa"], rtol=1e-9) and np.allclose(a["nu"], b["nu"], rtol=1e-9)


def test_mixing_is_zero_exactly_on_closed_faces_of_a_bathymetry():
    wl = W.with_ri_closure(W.config2(nx=24, ny=16, nz=10, steps=1))
    m = oracle.RefModel(wl)
    wet = m.grid.masks()["wet"].astype(bool)
    mix = m.mixing()
    open_face = np.zeros_like(wet)
    open_face[1:] = wet[1:] & wet[:-1]
    assert np.all(mix["nu"][~open_face] == 0.0) and np.all(mix["kappa"][~open_face] == 0.0)
    assert np.all(mix["nu"][open_face] >= 1e-4) and np.all(mix["kappa"][open_face] >= 1e-5)


# ------------------------------------------------------------------------ in the time step ----
def test_closure_with_zero_amplitudes_is_the_constant_coefficient_step_bitwise():
    wl = W.config0(nx=12, ny=10, nz=6, steps=3)
    a = oracle.RefModel(wl)
    w2 = clone(wl)
    w2["params"].update(RI, ri_nu0=0.0, ri_kconv=0.0)
    b = oracle.RefModel(w2)
    a.step(3); b.step(3)
    fa, fb = a.get_fields(), b.get_fields()
    for k in fa:
        assert np.array_equal(fa[k], fb[k]), k


def test_neutral_sheared_column_decays_with_nu_for_momentum_and_kappa_for_tracers():
    # alpha = beta_s = 0: buoyancy vanishes, Ri = 0 everywhere, nu = nu_z + nu0 and kappa = kappa_z + nu0 are uniform.
    # A horizontally uniform cosine mode of u, v (zero depth integral) and of T then obeys pure backward-Euler diffusion.
    nz, dz, dt, nsteps = 16, 10.0, 600.0, 5
    wl = box(nx=5, ny=4, nz=nz, depth=nz * dz, f0=0.0, dt=dt, substeps=10, alpha=0.0, beta_s=0.0,
             nu_z=3e-3, kappa_z=1e-3, **RI)
    k = np.arange(nz)
    mode = np.cos(np.pi * 3 * (k + 0.5) / nz)[:, None, None]
    wl["fields"]["u"] = 0.2 * mode + np.zeros_like(wl["fields"]["u"])
    wl["fields"]["v"] = -0.1 * mode + np.zeros_like(wl["fields"]["u"])
    wl["fields"]["T"] = 10.0 + 0.5 * mode + np.zeros_like(wl["fields"]["u"])
    m = oracle.RefModel(wl)
    m.step(nsteps)
    f = m.get_fields()
    lam = (4.0 / dz ** 2) * np.sin(np.pi * 3 / (2 * nz)) ** 2
    dm = (1.0 / (1.0 + dt * (3e-3 + 5e-3) * lam)) ** nsteps
    dk = (1.0 / (1.0 + dt * (1e-3 + 5e-3) * lam)) ** nsteps
    assert np.max(np.abs(f["u"] - 0.2 * dm * mode)) < 1e-13
    assert np.max(np.abs(f["v"] + 0.1 * dm * mode)) < 1e-13
    assert np.max(np.abs(f["T"] - 10.0 - 0.5 * dk * mode)) < 1e-12
    assert abs(dm - dk) > 1e-2                                    # the two coefficients are told apart


def test_tracer_conservation_and_convective_mixing_with_closure_on_latlon_with_land():
    wl = W.with_ri_closure(W.config2(nx=32, ny=20, nz=10, steps=4))
    wl["fields"]["T"][-3:] -= 2.0                                  # cold water on top: statically unstable
    m = oracle.RefModel(wl)
    wet = m.grid.masks()["wet"]
    met = m.grid.metrics()
    vol = wet * np.diff(wl["z_faces"])[:, None, None] * met["AzC"][None, :, None]
    f0 = m.get_fields()

    def inversion(f):                                              # largest T drop going up across an open face
        dT = (f["T"][1:] - f["T"][:-1])[(wet[1:] * wet[:-1]).astype(bool)]
        return float(-dT.min())
    inv0 = inversion(f0)
    m.step(4)
    f1 = m.get_fields()
    for c in ("T", "S"):
        a, b = np.sum(vol * f0[c]), np.sum(vol * f1[c])
        assert abs(a - b) < 2e-13 * abs(a), c
    plain = clone(wl)
    plain["params"].update(closure=0)
    m0 = oracle.RefModel(plain)
    m0.step(4)
    assert inversion(f1) < 0.8 * inv0 < 0.8 * inversion(m0.get_fields()) / 0.95   # convective adjustment at work,
                                                                                 # the background alone barely mixes
