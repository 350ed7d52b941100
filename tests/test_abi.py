"""CPU-side checks of the boundary: libocn.so loads, exports every symbol include/ocn.h declares,
and the host-only calls (grid creation, masks) agree bit-exactly with the oracle."""
import os
import re

import numpy as np
import pytest

import oracle
from paper_2309_06662_b200 import build as ocn_build
from paper_2309_06662_b200 import ocn
from paper_2309_06662_b200 import workloads as W
from util import box

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    ocn_build.build()


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "ocn.h")).read()
    declared = set(re.findall(r"\b(ocn_[a-z_]+)\s*\(", hdr))
    assert declared == set(ocn.EXPORTS)
    L = ocn.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert b"sm_100a" in L.ocn_version()


def test_bad_arguments_return_status_not_crash():
    wl = box(nx=8, ny=8, nz=4)
    g = dict(wl["grid"], nz=300)
    with pytest.raises(RuntimeError, match="nz > 250"):
        ocn.Grid(g, np.linspace(-300, 0, 301), np.ones((8, 8)))
    with pytest.raises(RuntimeError, match="increasing"):
        ocn.Grid(wl["grid"], wl["z_faces"][::-1].copy(), wl["depth"])
    with pytest.raises(RuntimeError, match="resting surface"):
        ocn.Grid(wl["grid"], wl["z_faces"] - 1.0, wl["depth"])
    zf = wl["z_faces"].copy(); zf[1] = np.nan
    with pytest.raises(RuntimeError, match="finite"):
        ocn.Grid(wl["grid"], zf, wl["depth"])
    g = dict(wl["grid"], kind=1, periodic_y=1)
    with pytest.raises(RuntimeError, match="periodic in latitude"):
        ocn.Grid(g, wl["z_faces"], wl["depth"])


def _mask_cases():
    rng = np.random.default_rng(11)
    for periodic in ((1, 1), (1, 0), (0, 0)):
        wl = box(nx=13, ny=10, nz=7, periodic=periodic, depth=700.0)
        d = rng.uniform(0, 800.0, (10, 13))
        d[rng.uniform(size=d.shape) < 0.2] = 0.0
        d[:, :6] = np.maximum(d[:, :6], 350.0)
        wl["depth"] = d
        yield wl
    yield W.config0(nx=4, ny=4, nz=2)                 # stencil wraps onto itself
    yield W.config1(nx=24, ny=20, nz=8)
    yield W.config2(nx=96, ny=40, nz=20)
    yield W.config4(nx=120, ny=48, nz=30, window=(4, 44, 10, 90))


@pytest.mark.parametrize("wl", list(_mask_cases()), ids=lambda w: f"{w['name']}_{w['grid']['nx']}x{w['grid']['ny']}")
def test_masks_bit_exact_against_oracle(wl):
    got = ocn.Grid(wl["grid"], wl["z_faces"], wl["depth"]).masks()
    want = oracle.RefGrid(wl["grid"], wl["z_faces"], wl["depth"]).masks()
    for n in want:
        assert np.array_equal(got[n], want[n]), n


def test_workspace_bytes_is_a_host_only_dry_run():
    """ocn_model_workspace_bytes sizes a model without touching a device (this test runs on the CPU box)."""
    import ctypes as C
    from paper_2309_06662_b200 import workloads as W
    wl = W.make(3, nx=96, ny=48, nz=12)
    g = ocn.Grid(wl["grid"], wl["z_faces"], wl["depth"])

    def size(**over):
        p = dict(wl["params"]); p.update(over)
        d = ocn.ocn_model_desc(device=0, **p)
        n = C.c_ulonglong()
        rc = ocn.lib().ocn_model_workspace_bytes(g.h, C.byref(d), C.byref(n))
        return rc, n.value

    rc, base = size()
    assert rc == 0
    sx, sy, nz = 128, 48 + 6, 12
    assert base > 7 * 8 * sx * sy * nz                     # at least the seven 3-D pair / fp64 arrays
    rc, ri = size(closure=1, ri_nu0=5e-3, ri_c=5.0, ri_kconv=0.1, ri_n2c=1e-7, ri_s2min=1e-10)
    assert rc == 0 and ri >= base + (8 + 4) * sx * sy * nz  # + the two super-diagonal arrays
    rc, bih = size(nu4_h=1e9)
    assert rc == 0 and bih >= base + 4 * 8 * sx * sy * nz
    rc, f64 = size(precision=64)
    assert rc == 0 and f64 > 1.5 * base
    rc, _ = size(dt=-1.0)
    assert rc != 0 and b"dt must be > 0" in ocn.lib().ocn_last_error()
    g.close()
