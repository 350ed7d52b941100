"""GPU parity of the scheme variants: WENO-Z weights and the nonlinear equation of
state, alone, together, and with the Ri closure; fp64 bit-identical to the oracle, fp32 within 2e-4."""
import numpy as np
import pytest

import oracle
from paper_2309_06662_b200 import build as ocn_build
from paper_2309_06662_b200 import ocn
from paper_2309_06662_b200 import workloads as W
from util import rel_linf, report_parity

pytestmark = pytest.mark.gpu
FIELDS = ("u", "v", "w", "eta", "T", "S")


@pytest.fixture(scope="module", autouse=True)
def _built():
    ocn_build.build()


def _stirred(wl, seed=21):
    rng = np.random.default_rng(seed)
    f, prec = wl["fields"], wl["params"]["precision"]
    f["u"] = W._round_to(prec, 0.3 * rng.standard_normal(f["u"].shape))
    f["v"] = W._round_to(prec, 0.3 * rng.standard_normal(f["v"].shape))
    f["T"] = W._round_to(prec, f["T"] + 0.5 * rng.standard_normal(f["T"].shape))       # non-smooth: the weights matter
    return wl


def _variant(kind, prec, closure):
    wl = _stirred(W.config2(nx=180, ny=75, nz=25, steps=8, precision=prec))
    if "z" in kind:
        W.with_weno_z(wl)
    if "e" in kind:
        W.with_nonlinear_eos(wl)
    if closure:
        W.with_ri_closure(wl)
    return wl


@pytest.mark.parametrize("kind", ["z", "e", "ze"])
@pytest.mark.parametrize("closure", [0, 1])
def test_variants_fp64_bit_identical(kind, closure):
    wl = _variant(kind, 64, closure)
    ref, gpu = oracle.RefModel(wl), ocn.Model(wl)
    ref.step(8); gpu.time_step(8)
    a, b = gpu.get_fields(), ref.get_fields()
    for n in FIELDS:
        assert np.array_equal(a[n], b[n]), (kind, closure, n, rel_linf(a[n], b[n]))
    gpu.close()


@pytest.mark.parametrize("kind", ["z", "e", "ze"])
@pytest.mark.parametrize("closure", [0, 1])
def test_variants_fp32_within_tolerance(kind, closure):
    wl = _variant(kind, 32, closure)
    ref, gpu = oracle.RefModel(wl), ocn.Model(wl)
    ref.step(8); gpu.time_step(8)
    a, b = gpu.get_fields(), ref.get_fields()
    errs = {n: rel_linf(a[n], b[n]) for n in FIELDS}
    report_parity("variants %s%s 180x75x25 fp32" % (kind, "+ri" if closure else ""), 8, errs)
    assert all(e <= 2e-4 for e in errs.values()), errs
    gpu.close()


def test_variants_change_the_answer_and_defaults_do_not():
    base = _variant("", 64, 0)
    g0 = ocn.Model(base); g0.time_step(4); f0 = g0.get_fields(); g0.close()
    for kind in ("z", "e"):
        g = ocn.Model(_variant(kind, 64, 0)); g.time_step(4); f = g.get_fields(); g.close()
        assert np.abs(f["T"] - f0["T"]).max() > 1e-7 or np.abs(f["u"] - f0["u"]).max() > 1e-7, kind
    # nonlinear EOS with zero coefficients = linear EOS, bit for bit, on the GPU too
    wl = W.with_nonlinear_eos(_variant("", 64, 0), alpha2=0.0, gamma=0.0)
    g = ocn.Model(wl); g.time_step(4); f = g.get_fields(); g.close()
    for n in FIELDS:
        assert np.array_equal(f[n], f0[n]), n


def test_wenoz_first_step_tendencies_match_on_aquaplanet_shape():
    wl = W.with_weno_z(_stirred(W.aquaplanet(nx=96, ny=40, nz=12, steps=1, precision=64)))
    ref, gpu = oracle.RefModel(wl), ocn.Model(wl)
    G = ref.tendencies()
    gpu.time_step(1)
    d = gpu.debug()
    for n in ("Gu", "Gv", "GT", "GS"):
        assert np.array_equal(d[n], G[n]), (n, rel_linf(d[n], G[n]))
    gpu.close()


def test_bad_variant_switches_are_rejected():
    wl = W.config0()
    for key, val in (("eos", 2), ("advection", 3)):
        bad = dict(wl, params=dict(wl["params"], **{key: val}))
        with pytest.raises(RuntimeError, match=key):
            ocn.Model(bad)


def _other_weights(M, p=1, q=2):
    s = np.arange(1, M + 1) / (M + 1.0)
    b = s ** p * (1.0 - s ** q)
    return b / b.sum()


@pytest.mark.parametrize("prec", [64, 32])
def test_separate_transport_filter_weights(prec):
    """filter_weights_uv: both barotropic kernels (fp64 point-wise tile, fp32 register strips; M = 30 is
    not a multiple of either kernel's sub-steps per launch) against the oracle; fp64 bit-identical."""
    wl = _stirred(W.config2(nx=180, ny=75, nz=25, steps=6, precision=prec))
    b = _other_weights(wl["params"]["substeps"])
    ref, gpu = oracle.RefModel(wl, filter_weights_uv=b), ocn.Model(wl, filter_weights_uv=b)
    plain = ocn.Model(wl)
    ref.step(6); gpu.time_step(6); plain.time_step(6)
    a, r, p0 = gpu.get_fields(), ref.get_fields(), plain.get_fields()
    assert np.abs(a["u"].astype(np.float64) - p0["u"]).max() > 1e-6             # the weights matter
    errs = {n: rel_linf(a[n], r[n]) for n in FIELDS}
    if prec == 64:
        for n in FIELDS:
            assert np.array_equal(a[n], r[n]), (n, errs[n])
    else:
        report_parity("transport weights 180x75x25 fp32", 6, errs)
        assert all(e <= 2e-4 for e in errs.values()), errs
    gpu.close(); plain.close()
    with pytest.raises(RuntimeError, match="filter_weights_uv"):
        ocn.Model(wl, filter_weights_uv=2.0 * b)


def _bih(wl, frac=0.01):
    g = wl["grid"]
    dxmin = g["radius"] * np.deg2rad(g["dx"]) * np.cos(np.deg2rad(max(abs(g["y0"]), abs(g["y0"] + g["ny"] * g["dy"])) - 0.5 * g["dy"]))
    k4 = frac * dxmin ** 4 / wl["params"]["dt"]
    wl["params"].update(nu4_h=float(k4), kappa4_h=float(0.5 * k4))
    wl["name"] = wl.get("name", "") + "+bih"
    return wl


@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("closure", [0, 1])
def test_biharmonic_dissipation(prec, closure):
    """nu4_h, kappa4_h: the pre-pass kernel pair + the add in K1 against the oracle on a lat-lon grid with
    land, periodic in x, noisy state (so that the term is large); fp64 bit-identical, fp32 within 2e-4."""
    wl = _bih(_stirred(W.config2(nx=180, ny=75, nz=25, steps=6, precision=prec)))
    if closure:
        W.with_ri_closure(wl)
    ref, gpu = oracle.RefModel(wl), ocn.Model(wl)
    off = ocn.Model(dict(wl, params=dict(wl["params"], nu4_h=0.0, kappa4_h=0.0)))
    assert gpu.info()["launches_per_step"] == off.info()["launches_per_step"] + 2
    G = ref.tendencies()
    ref.step(1); gpu.time_step(1); off.time_step(1)
    d, d0 = gpu.debug(), off.debug()
    for n in ("Gu", "Gv", "GT", "GS"):                          # first-step tendencies: the term is visible
        assert np.abs(d[n] - d0[n]).max() > 0.0, n             # the term is there (its size is pinned on the oracle side)
        if prec == 64:
            assert np.array_equal(d[n], G[n]), (n, rel_linf(d[n], G[n]))
    ref.step(5); gpu.time_step(5)
    a, r = gpu.get_fields(), ref.get_fields()
    errs = {n: rel_linf(a[n], r[n]) for n in FIELDS}
    if prec == 64:
        for n in FIELDS:
            assert np.array_equal(a[n], r[n]), (n, errs[n])
    else:
        report_parity("biharmonic%s 180x75x25 fp32" % ("+ri" if closure else ""), 6, errs)
        assert all(e <= 2e-4 for e in errs.values()), errs
    gpu.close(); off.close()


def test_biharmonic_on_small_periodic_and_walled_boxes_fp64():
    for nx, ny, per in ((5, 4, (1, 1)), (33, 9, (1, 0)), (12, 10, (0, 0))):
        wl = W.config0(nx=nx, ny=ny, nz=3)
        wl["grid"]["periodic_x"], wl["grid"]["periodic_y"] = per
        wl["params"].update(nu4_h=1.0e8, kappa4_h=5.0e7)
        ref, gpu = oracle.RefModel(wl), ocn.Model(wl)
        ref.step(4); gpu.time_step(4)
        a, r = gpu.get_fields(), ref.get_fields()
        for n in FIELDS:
            assert np.array_equal(a[n], r[n]), (nx, ny, per, n, rel_linf(a[n], r[n]))
        gpu.close()
