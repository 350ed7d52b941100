"""GPU tests of checkpoint / resume and the finite check (include/ocn.h): a model that loads a checkpoint
continues bit for bit where the saved one stood — which a restart through ocn_get_fields / ocn_set_fields does not (it takes an
Euler step: the quasi-AB2 history is not part of the field set)."""
import numpy as np
import pytest

from paper_2309_06662_b200 import build as ocn_build
from paper_2309_06662_b200 import ocn
from paper_2309_06662_b200 import workloads as W

pytestmark = pytest.mark.gpu
FIELDS = ("u", "v", "w", "eta", "T", "S")


@pytest.fixture(scope="module", autouse=True)
def _built():
    ocn_build.build()


def _workload(prec, kind=""):
    wl = W.config2(nx=96, ny=48, nz=12, steps=6, precision=prec)
    rng = np.random.default_rng(44)
    f = wl["fields"]
    f["u"] = W._round_to(prec, 0.3 * rng.standard_normal(f["u"].shape))
    f["v"] = W._round_to(prec, 0.3 * rng.standard_normal(f["v"].shape))
    f["T"] = W._round_to(prec, f["T"] + 0.5 * rng.standard_normal(f["T"].shape))
    if "r" in kind:
        W.with_ri_closure(wl)
    if "d" in kind:
        wl["params"].update(drag_r=2e-4, drag_cd=2e-3)
    if "b" in kind:
        wl["params"].update(nu4_h=1e9, kappa4_h=5e8)
    return wl


@pytest.mark.parametrize("prec,kind", [(32, ""), (32, "r"), (64, "db"), (64, "r")])
def test_resume_is_bit_exact(prec, kind):
    wl = _workload(prec, kind)
    a = ocn.Model(wl)
    a.time_step(3)
    blob = a.checkpoint()
    a.time_step(4)
    fa = a.get_fields()
    b = ocn.Model(wl)                       # same grid and parameters, its own (initial) state
    b.time_step(1)
    b.restore(blob)
    b.time_step(4)
    fb = b.get_fields()
    for k in FIELDS:
        assert np.array_equal(fa[k], fb[k]), (prec, kind, k)
    # the saved model can go back too
    a.restore(blob)
    a.time_step(4)
    fa2 = a.get_fields()
    for k in FIELDS:
        assert np.array_equal(fa[k], fa2[k]), k
    a.close(); b.close()


def test_a_restart_through_the_field_set_is_not_a_resume():
    wl = _workload(64)
    a = ocn.Model(wl)
    a.time_step(3)
    f3 = a.get_fields(("u", "v", "T", "S", "eta"))
    a.time_step(4)
    fa = a.get_fields()
    b = ocn.Model(wl)
    b.set_fields(**f3)                      # state only: the next step is an Euler step
    b.time_step(4)
    fb = b.get_fields()
    assert not np.array_equal(fa["u"], fb["u"])
    assert np.abs(fa["u"] - fb["u"]).max() < 0.5 * np.abs(fa["u"]).max()       # the same flow, not the same bits (rough initial state)
    a.close(); b.close()


def test_checkpoints_are_checked():
    a, b = ocn.Model(_workload(32)), ocn.Model(_workload(64))
    blob = a.checkpoint()
    assert blob.size == a.checkpoint().size and bytes(blob[:8]) == b"OCNCKPT1"
    with pytest.raises(RuntimeError, match="another size or precision"):
        b.restore(blob)
    with pytest.raises(RuntimeError, match="size mismatch"):
        a.restore(blob[:-16])
    bad = blob.copy(); bad[0] = ord("X")
    with pytest.raises(RuntimeError, match="bad magic"):
        a.restore(bad)
    with pytest.raises(RuntimeError, match="too short"):
        a.restore(blob[:8])
    a.step_part(0)
    with pytest.raises(RuntimeError, match="split step is in progress"):
        a.checkpoint()
    a.close(); b.close()


def test_finite_check_counts_poisoned_words():
    wl = _workload(32)
    m = ocn.Model(wl)
    m.time_step(2)
    assert m.nonfinite() == 0
    T = np.array(wl["fields"]["T"], dtype=np.float32)
    wet = np.argwhere(np.isfinite(T[-1]) & (wl["depth"] > 0))
    j, i = wet[len(wet) // 2]
    T[-1, j, i] = np.nan
    m.set_fields(T=T)
    assert m.nonfinite() >= 1
    m.time_step(1)
    assert m.nonfinite() > 1               # it spreads
    m.close()
