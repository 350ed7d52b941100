"""Parity of the CUDA path with surface heat / salinity fluxes and restoring."""
import numpy as np
import pytest

import oracle
from paper_2309_06662_b200 import build as ocn_build
from paper_2309_06662_b200 import ocn
from paper_2309_06662_b200 import workloads as W
from util import rel_linf

pytestmark = pytest.mark.gpu
TOL = {64: 1e-11, 32: 2e-4}
FIELDS = ("u", "v", "w", "eta", "T", "S")


@pytest.fixture(scope="module", autouse=True)
def _built():
    ocn_build.build()


@pytest.mark.parametrize("prec", [64, 32])
def test_surface_forcing_latlon_reduced(prec):
    wl = W.with_surface_forcing(W.config2(nx=180, ny=75, nz=25, steps=10, precision=prec))
    ref, gpu = oracle.RefModel(wl), ocn.Model(wl)
    ref.step(10); gpu.time_step(10)
    a, b = gpu.get_fields(), ref.get_fields()
    plain = oracle.RefModel(W.config2(nx=180, ny=75, nz=25, steps=10, precision=prec))
    plain.step(10)
    assert rel_linf(plain.get_fields()["T"], b["T"]) > 1e-4                      # the forcing matters in this case
    for n in FIELDS:
        if prec == 64:
            assert np.array_equal(a[n], b[n]), (n, rel_linf(a[n], b[n]))       # bit-identical, as the rest of the fp64 path
        else:
            assert rel_linf(a[n], b[n]) <= TOL[32], (n, rel_linf(a[n], b[n]))
    gpu.close()


def test_surface_forcing_with_closure_and_periodic_box_fp64():
    wl = W.with_surface_forcing(W.with_ri_closure(W.config0()))
    ref, gpu = oracle.RefModel(wl), ocn.Model(wl)
    ref.step(6); gpu.time_step(6)
    a, b = gpu.get_fields(), ref.get_fields()
    for n in FIELDS:
        assert rel_linf(a[n], b[n]) <= TOL[64], n
    gpu.close()


def test_forcing_only_update_keeps_the_ab2_history():
    wl = W.with_surface_forcing(W.config2(nx=96, ny=40, nz=12, steps=4))
    a, b = ocn.Model(wl), ocn.Model(wl)
    a.time_step(4)
    b.time_step(2)
    b.set_fields(**{k: wl["fields"][k] for k in ("flux_T", "flux_S", "restore_T", "restore_S")})   # same forcing again
    b.time_step(2)
    fa, fb = a.get_fields(), b.get_fields()
    for n in FIELDS:
        assert np.array_equal(fa[n], fb[n]), n


@pytest.mark.parametrize("prec", [64, 32])
def test_bottom_drag_latlon_reduced(prec):
    wl = W.config2(nx=180, ny=75, nz=25, steps=10, precision=prec)
    rng = np.random.default_rng(12)
    wl["fields"]["u"] = W._round_to(prec, 0.2 * rng.standard_normal(wl["fields"]["u"].shape))   # flow at the bottom too
    wl["fields"]["v"] = W._round_to(prec, 0.2 * rng.standard_normal(wl["fields"]["v"].shape))
    wl["params"].update(drag_r=5e-4, drag_cd=2.5e-3)
    ref, gpu = oracle.RefModel(wl), ocn.Model(wl)
    ref.step(10); gpu.time_step(10)
    a, b = gpu.get_fields(), ref.get_fields()
    for n in FIELDS:
        if prec == 64:
            assert np.array_equal(a[n], b[n]), (n, rel_linf(a[n], b[n]))
        else:
            assert rel_linf(a[n], b[n]) <= TOL[32], (n, rel_linf(a[n], b[n]))
    gpu.close()


def test_bottom_drag_first_step_tendency_matches_on_ragged_basin():
    wl = W.config1(nx=45, ny=37, nz=11, steps=2)
    rng = np.random.default_rng(13)
    wl["fields"]["u"] = 0.1 * rng.standard_normal(wl["fields"]["u"].shape)
    wl["fields"]["v"] = 0.1 * rng.standard_normal(wl["fields"]["v"].shape)
    wl["params"].update(drag_r=1e-3, drag_cd=3e-3)
    ref, gpu = oracle.RefModel(wl), ocn.Model(wl)
    G = ref.tendencies()
    gpu.time_step(1)
    d = gpu.debug()
    for n in ("Gu", "Gv"):
        assert np.array_equal(d[n], G[n]), (n, rel_linf(d[n], G[n]))


def test_time_varying_forcing_updated_every_step():
    # the realistic use (forcing fields change in time): wind stress and heat flux re-sent before every
    # step on both sides; the AB2 history is kept, so this is NOT a sequence of Euler restarts
    wl = W.with_surface_forcing(W.config2(nx=96, ny=40, nz=12, steps=6))
    ref, gpu = oracle.RefModel(wl), ocn.Model(wl)
    for n in range(6):
        s = np.cos(0.7 * n)
        upd = dict(tau_x=s * wl["fields"]["tau_x"], flux_T=(1.0 - 0.3 * n) * wl["fields"]["flux_T"])
        ref.set_fields(**upd); gpu.set_fields(**upd)
        ref.step(1); gpu.time_step(1)
    a, b = gpu.get_fields(), ref.get_fields()
    for n in FIELDS:
        assert np.array_equal(a[n], b[n]), (n, rel_linf(a[n], b[n]))
    euler = oracle.RefModel(wl)                                  # what Euler restarts would have given: different
    for n in range(6):
        euler.set_fields(tau_x=np.cos(0.7 * n) * wl["fields"]["tau_x"], u=euler.get_fields()["u"])
        euler.step(1)
    assert rel_linf(euler.get_fields()["u"], b["u"]) > 1e-6
