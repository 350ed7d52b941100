"""Pins of the oracle's surface tracer forcing against budgets and closed forms."""
import numpy as np

import oracle
from paper_2309_06662_b200 import workloads as W
from util import box, clone


def test_tracer_budget_grows_by_the_area_integrated_flux_exactly():
    # flux form + AB2 with a constant source: after n steps the volume integral has grown by n dt sum(A flux) over
    # wet columns, whatever the flow does (lat-lon grid with land, flow spun up by the wind)
    wl = W.config2(nx=32, ny=20, nz=10, steps=5)
    rng = np.random.default_rng(8)
    wl["fields"]["flux_T"] = 2e-5 * rng.standard_normal((20, 32))
    wl["fields"]["flux_S"] = 1e-6 * rng.standard_normal((20, 32))
    m = oracle.RefModel(wl)
    wet = m.grid.masks()["wet"]
    A = m.grid.metrics()["AzC"][:, None] * wet[-1]
    vol = wet * np.diff(wl["z_faces"])[:, None, None] * m.grid.metrics()["AzC"][None, :, None]
    f0 = m.get_fields()
    m.step(5)
    f1 = m.get_fields()
    dt = wl["params"]["dt"]
    for c, q in (("T", "flux_T"), ("S", "flux_S")):
        got = np.sum(vol * f1[c]) - np.sum(vol * f0[c])
        want = 5 * dt * np.sum(A * wl["fields"][q])
        assert abs(got - want) < 1e-12 * np.sum(vol * np.abs(f0[c])), (c, got, want)
        assert abs(got - want) < 1e-4 * abs(want), (c, got, want)
    land = ~wet.astype(bool)
    assert np.all(f1["T"][land] == 0.0) and np.all(f1["S"][land] == 0.0)      # a flux over land goes nowhere


def test_restoring_of_a_resting_uniform_ocean_obeys_the_ab2_recurrence():
    nz, dz, dt, gam, chi = 4, 25.0, 600.0, 5e-4, 0.1
    wl = box(nx=6, ny=5, nz=nz, depth=nz * dz, f0=1e-4, dt=dt, substeps=10, kappa_z=0.0, nu_z=0.0,
             gamma_T=gam, gamma_S=2 * gam)
    wl["fields"]["restore_T"] = np.full((5, 6), 14.0)
    wl["fields"]["restore_S"] = np.full((5, 6), 34.5)
    m = oracle.RefModel(wl)
    qT, qS, pT, pS = 10.0 - 14.0, 35.0 - 34.5, None, None
    for n in range(20):
        m.step(1)
        zT, zS = -dt * gam / dz, -dt * 2 * gam / dz
        if pT is None:
            pT, qT, pS, qS = qT, qT + zT * qT, qS, qS + zS * qS
        else:
            pT, qT = qT, qT + zT * ((1.5 + chi) * qT - (0.5 + chi) * pT)
            pS, qS = qS, qS + zS * ((1.5 + chi) * qS - (0.5 + chi) * pS)
    f = m.get_fields()
    assert np.max(np.abs(f["T"][-1] - (14.0 + qT))) < 1e-12 and np.max(np.abs(f["S"][-1] - (34.5 + qS))) < 1e-12
    assert np.all(f["T"][:-1] == 10.0) and np.all(f["S"][:-1] == 35.0)         # only the top cell is forced (kappa_z = 0)
    assert np.all(f["u"] == 0.0) and np.all(f["v"] == 0.0)                       # horizontally uniform: stays at rest


def test_uniform_heating_warms_the_top_cell_by_flux_dt_over_dz_and_zero_forcing_is_the_plain_step_bitwise():
    wl = box(nx=6, ny=5, nz=4, depth=100.0, dt=300.0, substeps=10, kappa_z=0.0, nu_z=0.0)
    wl["fields"]["flux_T"] = np.full((5, 6), 1e-5)
    m = oracle.RefModel(wl)
    m.step(3)
    f = m.get_fields()
    assert np.max(np.abs(f["T"][-1] - (10.0 + 3 * 300.0 * 1e-5 / 25.0))) < 1e-13
    assert np.all(f["S"] == 35.0)                                                # the heat flux does not touch salinity
    a = W.config0(nx=12, ny=10, nz=6, steps=3)
    b = clone(a)
    b["fields"].update(flux_T=np.zeros((10, 12)), restore_T=np.full((10, 12), 3.0))   # gamma = 0: the target is inert
    ma, mb = oracle.RefModel(a), oracle.RefModel(b)
    ma.step(3); mb.step(3)
    fa, fb = ma.get_fields(), mb.get_fields()
    assert all(np.array_equal(fa[k], fb[k]) for k in fa)


# ------------------------------------------------------------------ bottom drag ----
def test_linear_bottom_drag_obeys_the_ab2_recurrence_on_the_lowest_level_only():
    nz, dz, dt, r, chi = 4, 25.0, 600.0, 2e-3, 0.1
    wl = box(nx=6, ny=5, nz=nz, depth=nz * dz, f0=0.0, dt=dt, substeps=10, kappa_z=0.0, nu_z=0.0, drag_r=r)
    wl["fields"]["u"][:] = 0.3
    wl["fields"]["v"][:] = -0.2
    m = oracle.RefModel(wl)
    z = -dt * r / dz
    q, p = np.array([0.3, -0.2]), None
    for n in range(15):
        m.step(1)
        if p is None:
            p, q = q, q + z * q
        else:
            p, q = q, q + z * ((1.5 + chi) * q - (0.5 + chi) * p)
    f = m.get_fields()
    assert np.max(np.abs(f["u"][0] - q[0])) < 1e-13 and np.max(np.abs(f["v"][0] - q[1])) < 1e-13
    assert np.max(np.abs(f["u"][1:] - 0.3)) < 1e-13 and np.max(np.abs(f["v"][1:] + 0.2)) < 1e-13   # nu_z = 0: the rest coasts
    assert np.abs(f["eta"]).max() < 1e-12                         # uniform transport: the free surface stays flat


def test_quadratic_bottom_drag_first_step_closed_form_uses_the_speed_at_the_point():
    dz, dt, cd = 20.0, 300.0, 3e-3
    wl = box(nx=6, ny=5, nz=3, depth=3 * dz, f0=0.0, dt=dt, substeps=10, kappa_z=0.0, nu_z=0.0, drag_cd=cd)
    wl["fields"]["u"][:] = 0.4
    wl["fields"]["v"][:] = 0.3                                     # speed 0.5 at every u and v point
    m = oracle.RefModel(wl)
    m.step(1)                                                      # Euler start
    f = m.get_fields()
    assert np.max(np.abs(f["u"][0] - (0.4 - dt * cd * 0.5 * 0.4 / dz))) < 1e-14
    assert np.max(np.abs(f["v"][0] - (0.3 - dt * cd * 0.5 * 0.3 / dz))) < 1e-14


def test_drag_acts_exactly_on_the_lowest_open_u_and_v_levels_of_a_bathymetry():
    wl = W.config2(nx=32, ny=20, nz=10, steps=1)
    rng = np.random.default_rng(9)
    wl["fields"]["u"] = 0.1 * rng.standard_normal(wl["fields"]["u"].shape)
    wl["fields"]["v"] = 0.1 * rng.standard_normal(wl["fields"]["v"].shape)
    r = 1e-3
    a = oracle.RefModel(wl)
    w2 = clone(wl); w2["params"].update(drag_r=r)
    b = oracle.RefModel(w2)
    Ga, Gb, f = a.tendencies(), b.tendencies(), a.get_fields()
    masks = a.grid.masks()
    dz = np.diff(wl["z_faces"])
    for name, vel, mk in (("Gu", "u", "order_zeta_u"), ("Gv", "v", "order_zeta_v")):
        open_ = masks[mk] > 0                                      # open faces carry a vorticity order >= 1
        want = np.zeros_like(Ga[name])
        for j in range(20):                                        # brute force: first open level of each column
            for i in range(32):
                ks = np.nonzero(open_[:, j, i])[0]
                if ks.size:
                    want[ks[0], j, i] = -r * f[vel][ks[0], j, i] / dz[ks[0]]
        assert np.max(np.abs((Gb[name] - Ga[name]) - want)) < 1e-18 + 1e-12 * np.abs(want).max(), name
        assert np.abs(want).max() > 0


def test_zero_drag_coefficients_are_the_plain_step_bitwise():
    a = W.config0(nx=12, ny=10, nz=6, steps=3)
    b = clone(a); b["params"].update(drag_r=0.0, drag_cd=0.0)
    ma, mb = oracle.RefModel(a), oracle.RefModel(b)
    ma.step(3); mb.step(3)
    fa, fb = ma.get_fields(), mb.get_fields()
    assert all(np.array_equal(fa[k], fb[k]) for k in fa)


def test_forcing_only_set_fields_keeps_state_and_history_in_the_oracle():
    # re-sending the same forcing between steps must not change anything (no Euler restart, no re-derivation)
    wl = W.with_surface_forcing(W.config2(nx=24, ny=16, nz=8, steps=4))
    a, b = oracle.RefModel(wl), oracle.RefModel(wl)
    a.step(4)
    b.step(2)
    b.set_fields(**{k: wl["fields"][k] for k in ("tau_x", "tau_y", "flux_T", "flux_S", "restore_T", "restore_S")})
    b.step(2)
    fa, fb = a.get_fields(), b.get_fields()
    assert all(np.array_equal(fa[k], fb[k]) for k in fa)
