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
