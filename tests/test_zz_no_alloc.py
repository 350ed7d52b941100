"""ocn_get_mixing_noalloc: the allocation-free variant of ocn_get_mixing (static device scratch, include/ocn.h) against the
existing path.  In a file of its own that pytest collects LAST (the suite runs with `pytest -x`: a failure here must not
hide other tests).  Passes alone in a fresh process and after the other GPU tests: it creates its own models and assumes
nothing about what the shared scratch array holds."""
import numpy as np
import pytest

import oracle
from paper_2309_06662_b200 import build as ocn_build
from paper_2309_06662_b200 import ocn
from paper_2309_06662_b200 import workloads as W
from util import rel_linf

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    ocn_build.build()


def _stirred(wl, seed):
    rng = np.random.default_rng(seed)
    f, prec = wl["fields"], wl["params"]["precision"]
    zc = 0.5 * (wl["z_faces"][:-1] + wl["z_faces"][1:])
    shear = 0.3 * ((zc - zc[0]) / (zc[-1] - zc[0])) ** 2
    f["u"] = W._round_to(prec, shear[:, None, None] * (1 + 0.2 * rng.standard_normal(f["u"].shape)))
    f["v"] = W._round_to(prec, 0.5 * shear[:, None, None] * (1 + 0.2 * rng.standard_normal(f["v"].shape)))
    f["T"] = W._round_to(prec, f["T"] - 1.5 * (np.arange(len(zc)) >= len(zc) - 2)[:, None, None])      # an inversion on top
    return wl


def test_noalloc_mixing_matches_existing_path_on_two_calls_in_a_row():
    # call 1: fp64, lat-lon with land, 96 x 40 x 12 (1.1 MB of the scratch); call 2: fp32, another grid with another land
    # pattern and row pitch, 70 x 30 x 100 (2.7 MB): it finds call 1's values where its own land and halos lie; call 3:
    # model 1 again, on top of what model 2 left
    wa = _stirred(W.with_ri_closure(W.config2(nx=96, ny=40, nz=12, steps=1)), 3)
    wb = _stirred(W.with_ri_closure(W.config4(window=(500, 530, 1300, 1370), steps=1)), 4)
    wb["params"]["precision"] = 32
    wb["fields"] = {k: W._round_to(32, v) for k, v in wb["fields"].items()}
    a, b = ocn.Model(wa), ocn.Model(wb)
    ref_a = oracle.RefModel(wa).mixing()
    for model, tol_oracle, ref in ((a, 0.0, ref_a), (b, None, None), (a, 0.0, ref_a)):
        want = model.mixing()                      # existing path (allocates its output array on first use)
        got = model.mixing_noalloc()               # static scratch
        for n in ("nu", "kappa"):
            assert want[n].max() > 10 * want[n][want[n] > 0].min()               # the closure is active
            assert np.array_equal(got[n], want[n]), (n, rel_linf(got[n], want[n]))
            if ref is not None:                                                     # fp64: bit-identical to the oracle as well
                assert np.array_equal(got[n], ref[n]), n
    # after a few steps the state has changed: both paths follow it
    a.time_step(3)
    want, got = a.mixing(), a.mixing_noalloc()
    assert not np.array_equal(want["nu"], ref_a["nu"])
    for n in ("nu", "kappa"):
        assert np.array_equal(got[n], want[n]), n
    # fp32 model against the oracle at the tolerance tests/test_gpu_closure.py uses for the coefficients
    ref_b = oracle.RefModel(wb).mixing()
    got = b.mixing_noalloc()
    for n in ("nu", "kappa"):
        assert np.array_equal(got[n] == 0.0, ref_b[n] == 0.0), n
        assert rel_linf(got[n], ref_b[n]) < 1e-5, n
    a.close(); b.close()


def test_noalloc_mixing_allocates_no_device_memory():
    import torch
    wl = _stirred(W.with_ri_closure(W.config2(nx=96, ny=40, nz=12, steps=1)), 5)
    m = ocn.Model(wl)
    m.mixing_noalloc()                             # first call: kernel code is loaded, the symbol address looked up
    m.synchronize(); torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        m.mixing_noalloc()
    m.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, (free0, free1)
    m.close()


def test_noalloc_mixing_rejects_models_beyond_the_static_scratch():
    cap = ocn.lib().ocn_noalloc_scratch_bytes()
    assert cap == 16 << 20
    wl = W.with_ri_closure(W.config2(nx=360, ny=150, nz=50, steps=1))         # 384 x 156 x 50 pairs of fp64 = 47.9 MB
    m = ocn.Model(wl)
    with pytest.raises(RuntimeError, match="static scratch holds 16777216"):
        m.mixing_noalloc()
    assert m.mixing()["nu"].max() > 0                                          # the allocating path serves it
    m.close()
    plain = ocn.Model(W.config0())
    with pytest.raises(RuntimeError, match="closure = 0"):
        plain.mixing_noalloc()
    plain.close()
