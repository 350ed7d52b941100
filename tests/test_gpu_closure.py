"""Parity of the CUDA path with the Ri-based vertical mixing closure (closure = 1: K4 mixing coefficients, K5
per-column elimination, K3 reading the stored super-diagonals) against the oracle."""
import numpy as np
import pytest

import oracle
from paper_2309_06662_b200 import build as ocn_build
from paper_2309_06662_b200 import ocn
from paper_2309_06662_b200 import workloads as W
from util import box, clone, rel_linf

pytestmark = pytest.mark.gpu
TOL = {64: 1e-11, 32: 2e-4}
FIELDS = ("u", "v", "w", "eta", "T", "S")


@pytest.fixture(scope="module", autouse=True)
def _built():
    ocn_build.build()


def _stir(wl, seed=3, unstable_top=0):
    """a sheared flow so that Ri spans its range, and optionally cold water on top (convective ramp active)"""
    rng = np.random.default_rng(seed)
    nz = wl["grid"]["nz"]
    prof = np.linspace(0.0, 1.0, nz)[:, None, None] ** 2
    prec = wl["params"]["precision"]
    wl["fields"]["u"] = W._round_to(prec, wl["fields"]["u"] + 0.3 * prof * (1 + 0.2 * rng.standard_normal(wl["fields"]["u"].shape)))
    wl["fields"]["v"] = W._round_to(prec, wl["fields"]["v"] - 0.2 * prof * (1 + 0.2 * rng.standard_normal(wl["fields"]["v"].shape)))
    if unstable_top:
        wl["fields"]["T"][-unstable_top:] = W._round_to(prec, wl["fields"]["T"][-unstable_top:] - 1.5)
    return wl


def _run_both(wl, stops):
    ref, gpu = oracle.RefModel(wl), ocn.Model(wl)
    done, errs = 0, {}
    for stop in stops:
        ref.step(stop - done); gpu.time_step(stop - done); done = stop
        a, b = gpu.get_fields(), ref.get_fields()
        errs = {n: rel_linf(a[n], b[n]) for n in FIELDS}
        bad = {n: e for n, e in errs.items() if not e <= TOL[wl["params"]["precision"]]}
        assert not bad, (wl["name"], stop, errs)
        assert all(np.isfinite(a[n]).all() for n in FIELDS)
    gpu.close()
    return errs


def test_mixing_coefficients_match_the_oracle_fp64_bitwise_and_fp32_rounded():
    for prec in (64, 32):
        wl = _stir(W.with_ri_closure(W.config2(nx=96, ny=40, nz=12, steps=1, precision=prec)), unstable_top=2)
        ref, gpu = oracle.RefModel(wl), ocn.Model(wl)
        a, b = gpu.mixing(), ref.mixing()
        assert b["nu"].max() > 10 * b["nu"][b["nu"] > 0].min()          # the closure is active, not just the background
        for n in ("nu", "kappa"):
            if prec == 64:
                assert np.array_equal(a[n], b[n]), n
            else:
                assert np.array_equal(a[n] == 0.0, b[n] == 0.0), n      # closed faces: exact zeros at the same places
                assert rel_linf(a[n], b[n]) < 1e-5, n
        gpu.close()


def test_closure_requires_closure_model():
    gpu = ocn.Model(W.config0(nx=8, ny=8, nz=4))
    with pytest.raises(RuntimeError):
        gpu.mixing()
    bad = W.with_ri_closure(W.config0(nx=8, ny=8, nz=4), n2c=0.0)
    with pytest.raises(RuntimeError):
        ocn.Model(bad)


def test_closure_config0_periodic_fp64():
    wl = _stir(W.with_ri_closure(W.config0()))
    _run_both(wl, [1, 2, 10])


def test_closure_ragged_basin_with_walls_fp64():
    wl = _stir(W.with_ri_closure(W.config1(nx=45, ny=37, nz=11, steps=12)), unstable_top=2)
    _run_both(wl, [1, 12])


def test_closure_latlon_reduced_fp64():
    wl = _stir(W.with_ri_closure(W.config2(nx=360, ny=150, nz=50, steps=10)), unstable_top=3)
    _run_both(wl, [1, 10])


def test_closure_latlon_reduced_fp32():
    wl = _stir(W.with_ri_closure(W.config3(nx=360, ny=150, nz=50, steps=10)), unstable_top=3)
    _run_both(wl, [1, 10])


def test_closure_config4_window_fp32():
    wl = W.with_ri_closure(W.config4(window=(500, 600, 1300, 1500), steps=10))
    _run_both(wl, [1, 10])


def test_closure_with_zero_amplitudes_equals_constant_coefficient_path_on_gpu():
    # K4 + K5 + K3<RI> against the table-driven K1 / K3 of the default path: same numbers in fp64
    wl = W.config2(nx=96, ny=40, nz=12, steps=3)
    w2 = W.with_ri_closure(clone(wl), nu0=0.0, kconv=0.0)
    a, b = ocn.Model(wl), ocn.Model(w2)
    a.time_step(3); b.time_step(3)
    fa, fb = a.get_fields(), b.get_fields()
    for n in FIELDS:
        assert np.array_equal(fa[n], fb[n]), n


def test_closure_runs_inside_the_tendency_kernel():
    """The closure is evaluated inside K1: no extra launches, and the step allocates no (nu, kappa) array."""
    wl = W.with_ri_closure(W.config3(nx=96, ny=40, nz=12, steps=3))
    gpu = ocn.Model(wl)
    plain = ocn.Model(W.config3(nx=96, ny=40, nz=12, steps=3))
    gpu.time_step(1)
    gpu.profile_enable(True)
    gpu.time_step(3)
    prof = gpu.profile_read()
    assert prof["vertical_mixing"]["launches"] == 0
    assert gpu.info()["launches_per_step"] == prof["tendency"]["launches"] // 3 + prof["barotropic"]["launches"] // 3 + 1
    assert gpu.info()["launches_per_step"] == plain.info()["launches_per_step"]
    n3 = gpu.info()["device_bytes"] - plain.info()["device_bytes"]
    cells_padded = (40 + 6) * 128 * 12                      # plane layout: sy x sx x nz
    assert 3 * 4 * cells_padded <= n3 < 3.2 * 4 * cells_padded      # three more words per cell: cp of (u, v) and of (T, S)


def test_closure_fp64_is_bit_identical_to_the_oracle():
    # K4 / K5 / K3<RI> keep the association of DESIGN.md §3.12 and §3.8-4 in non-contracted IEEE operations
    for wl in (_stir(W.with_ri_closure(W.config0(nx=24, ny=20, nz=8))),
               _stir(W.with_ri_closure(W.config2(nx=96, ny=40, nz=12, steps=6)), unstable_top=2)):
        ref, gpu = oracle.RefModel(wl), ocn.Model(wl)
        ref.step(6); gpu.time_step(6)
        a, b = gpu.get_fields(), ref.get_fields()
        for n in FIELDS:
            assert np.array_equal(a[n], b[n]), (wl["name"], n, rel_linf(a[n], b[n]))
        gpu.close()


def _all_options(wl):
    """closure + surface forcing + bottom drag together"""
    W.with_surface_forcing(W.with_ri_closure(wl))
    wl["params"].update(drag_r=5e-4, drag_cd=2.5e-3)
    return wl


def test_degenerate_shapes_with_closure_forcing_and_drag():
    # the smallest grids (stencil wraps onto itself, two levels = one interior face), walls, one warp-straddling width
    for nx, ny, nz, per in ((3, 3, 2, (1, 1)), (4, 4, 2, (1, 1)), (5, 4, 3, (0, 0)), (33, 9, 2, (1, 0))):
        wl = W.config0(nx=nx, ny=ny, nz=nz)
        wl["grid"]["periodic_x"], wl["grid"]["periodic_y"] = per
        _run_both(_all_options(wl), [1, 4])


def test_all_land_and_isolated_columns_with_closure_forcing_and_drag():
    wl = _all_options(W.config1(nx=40, ny=20, nz=6, steps=3))
    wl["depth"][:] = 0.0
    gpu = ocn.Model(wl)
    gpu.time_step(3)
    f = gpu.get_fields()
    for n in FIELDS:
        assert np.all(f[n] == 0.0), n
    gpu.close()
    rng = np.random.default_rng(11)
    wl = W.config1(nx=70, ny=21, nz=9, steps=6)
    d = wl["depth"]
    d[::2, ::2] = 0.0                                   # isolated wet columns (no open faces), ragged depths
    d[10, :] = 3500.0                                   # a one-cell-wide zonal channel
    d[:, 35] = rng.uniform(200.0, 4000.0, size=d.shape[0])
    d[0, :] = d[-1, :] = 0.0; d[:, 0] = d[:, -1] = 0.0
    wl["fields"]["u"] = 0.05 * rng.standard_normal(wl["fields"]["u"].shape)
    wl["fields"]["v"] = 0.05 * rng.standard_normal(wl["fields"]["v"].shape)
    _run_both(_all_options(wl), [1, 6])


def test_many_levels_with_closure_nz_150_fp64():
    wl = W.config4(window=(600, 640, 2000, 2070), steps=3, precision=64)
    nz = 150
    zf = W.geometric_z_faces(nz, 5.0, 6000.0)
    zc_old = 0.5 * (wl["z_faces"][:-1] + wl["z_faces"][1:]); zc = 0.5 * (zf[:-1] + zf[1:])
    f = wl["fields"]
    for n in ("u", "v", "T", "S"):
        a = f[n]
        out = np.empty((nz,) + a.shape[1:])
        for j in range(a.shape[1]):
            for i in range(a.shape[2]):
                out[:, j, i] = np.interp(zc, zc_old, a[:, j, i])
        f[n] = out
    wl["z_faces"] = zf
    wl["grid"]["nz"] = nz
    _run_both(_all_options(wl), [1, 3])
