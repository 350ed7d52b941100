"""Every BASELINE.json config at its STATED size and step count against the oracle (north_star: "every config matches the
oracle within the stated tolerances"), in the launch configuration bench.py times (CUDA-graph replay of the AB2 step):

    config 1  256 x 256 x 32, fp64, 100 steps   bit-identical
    config 2  1440 x 600 x 50, fp64, 50 steps    bit-identical
    config 3  1440 x 600 x 50, fp32, 50 steps    <= 2e-4, checked after 10, 25 and 50 steps
    config 4  2880 x 1200 x 100, fp32, 6 steps   <= 2e-4 against the oracle on a 700 x 560 x 100 window (interior only)

The oracle (OpenMP over rows, bit-identical to serial) needs about 100 s per full quarter-degree run on 16 cores.  The
per-field errors are printed in pytest's terminal summary (tests/conftest.py)."""
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


def _compare(wl, checkpoints, tol, exact):
    ref, gpu = oracle.RefModel(wl), ocn.Model(wl)
    done = 0
    for stop in checkpoints:
        ref.step(stop - done); gpu.time_step(stop - done)
        done = stop
        a, b = gpu.get_fields(), ref.get_fields()
        errs = {n: rel_linf(a[n], b[n]) for n in FIELDS}
        report_parity(wl["name"] + " FULL %dx%dx%d fp%d" % (wl["grid"]["nx"], wl["grid"]["ny"], wl["grid"]["nz"],
                                                              wl["params"]["precision"]), stop, errs)
        assert all(np.isfinite(a[n]).all() for n in FIELDS)
        assert np.abs(b["u"]).max() > 1e-4                      # the run is not trivial
        if exact:
            for n in FIELDS:
                assert np.array_equal(a[n], b[n]), (wl["name"], stop, n, errs[n])
        else:
            assert all(e <= tol for e in errs.values()), (wl["name"], stop, errs)
    gpu.close()


def test_config1_full_size_100_steps_fp64_bit_identical():
    _compare(W.config1(), [50, 100], 1e-11, exact=True)


def test_config2_full_size_50_steps_fp64_bit_identical():
    _compare(W.config2(), [50], 1e-11, exact=True)


def test_config3_full_size_50_steps_fp32():
    _compare(W.config3(), [10, 25, 50], 2e-4, exact=False)


@pytest.mark.parametrize("closure", [0, 1])
def test_config4_full_size_6_steps_against_a_larger_oracle_window(closure):
    """One step has a finite domain of dependence (3 cells of stencil + one cell per barotropic sub-step = 43 cells), so
    after 6 steps every point further than 6 x 43 cells from the walls of a window run by the oracle as a closed box must
    agree with the full-size GPU run."""
    j0, j1, i0, i1 = 320, 880, 1150, 1850
    steps = 6
    margin = steps * (40 + 3) + 2
    full = W.config4()
    if closure:
        W.with_ri_closure(full)
    gpu = ocn.Model(full)
    gpu.time_step(steps)
    a = gpu.get_fields()
    gpu.close()
    del full
    win = W.config4(window=(j0, j1, i0, i1))
    if closure:
        W.with_ri_closure(win)
    ref = oracle.RefModel(win)
    ref.step(steps)
    b = ref.get_fields()
    js, je, is_, ie = margin, (j1 - j0) - margin, margin, (i1 - i0) - margin
    assert je - js >= 30 and ie - is_ >= 150
    errs = {}
    for n in FIELDS:
        fa = a[n][..., j0 + js:j0 + je, i0 + is_:i0 + ie].astype(np.float64)
        fb = b[n][..., js:je, is_:ie]
        errs[n] = float(np.abs(fa - fb).max() / max(np.abs(b[n]).max(), 1e-300))
    report_parity("cfg4 FULL 2880x1200x100 fp32 vs oracle window%s" % (" +ri" if closure else ""), steps, errs)
    assert all(e <= 2e-4 for e in errs.values()), errs


def test_statically_unstable_recipe_with_the_closure_reduced_size():
    """SURVEY 8(d)'s original T/S proposal (S = 35 - cos(2 phi) e^{z/500}, T = 2 + 25 cos^2(phi) e^{z/800}) is statically
    unstable poleward of 45 degrees; DESIGN.md §4 replaced it for the timed configs because an overturning state amplifies
    round-off.  It stays alive here: reduced size, closure on (the convective ramp is what such a state needs), fp64
    bit-identical for 10 steps and fp32 inside the tolerance for the first steps."""
    def unstable(precision):
        wl = W.config2(nx=180, ny=75, nz=25, steps=10, precision=precision)
        g = wl["grid"]
        zc = 0.5 * (wl["z_faces"][:-1] + wl["z_faces"][1:])
        lat = np.deg2rad(g["y0"] + (np.arange(g["ny"]) + 0.5) * g["dy"])
        rng = np.random.default_rng(W.SEED_BASE + 77)
        T = 2.0 + 25.0 * (np.cos(lat) ** 2)[None, :, None] * np.exp(zc / 800.0)[:, None, None] + 0.01 * rng.standard_normal((g["nz"], g["ny"], g["nx"]))
        S = 35.0 - np.cos(2 * lat)[None, :, None] * np.exp(zc / 500.0)[:, None, None] + 0.001 * rng.standard_normal((g["nz"], g["ny"], g["nx"]))
        wl["fields"]["T"] = W._round_to(precision, T)
        wl["fields"]["S"] = W._round_to(precision, S)
        wl["name"] = "cfg2_unstable_recipe"
        return W.with_ri_closure(wl)
    wl = unstable(64)
    # there ARE statically unstable columns: N2 < 0 somewhere poleward of 45 degrees
    P = wl["params"]
    b = P["g"] * (P["alpha"] * (wl["fields"]["T"] - P["T0"]) - P["beta_s"] * (wl["fields"]["S"] - P["S0"]))
    assert (np.diff(b, axis=0)[:, :8, :] < 0).mean() > 0.2
    ref, gpu = oracle.RefModel(wl), ocn.Model(wl)
    kap = ref.mixing()["kappa"]
    assert kap.max() > 0.05                                      # the convective term is active
    ref.step(10); gpu.time_step(10)
    a, r = gpu.get_fields(), ref.get_fields()
    for n in FIELDS:
        assert np.array_equal(a[n], r[n]), (n, rel_linf(a[n], r[n]))
    gpu.close()
    wl32 = unstable(32)
    ref, gpu = oracle.RefModel(wl32), ocn.Model(wl32)
    ref.step(3); gpu.time_step(3)
    a, r = gpu.get_fields(), ref.get_fields()
    errs = {n: rel_linf(a[n], r[n]) for n in FIELDS}
    report_parity("cfg3 unstable recipe + ri 180x75x25 fp32", 3, errs)
    assert all(e <= 2e-4 for e in errs.values()), errs
    gpu.close()
