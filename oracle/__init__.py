"""ctypes front end of the CPU oracle (oracle/ocn_ref.cpp).

TEST INFRASTRUCTURE ONLY: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package.  It shares no code with the CUDA library and
does not import paper_2309_06662_b200.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libocn_ref.so")
_SRC = [os.path.join(_HERE, "ocn_ref.cpp"), os.path.join(_HERE, "ocn_ref.h")]
# tests/test_oracle_mutations.py points this at a deliberately broken copy of ocn_ref.cpp (built into its own .so next
# to that copy) to prove that the pins of tests/ notice the mistake; unset everywhere else
if os.environ.get("OCN_REF_MUTANT_SRC"):
    _SRC = [os.environ["OCN_REF_MUTANT_SRC"], _SRC[1]]
    _SO = os.environ["OCN_REF_MUTANT_SRC"] + ".so"
_lib = None


def build(force=False):
    """Compile the oracle with g++ (plain -O2, OpenMP over rows; no fast-math)."""
    if not force and os.path.exists(_SO) and all(os.path.getmtime(_SO) >= os.path.getmtime(s) for s in _SRC):
        return _SO
    cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", "-I", _HERE,
           "-o", _SO, _SRC[0]]
    subprocess.check_call(cmd)
    return _SO


class GridDesc(C.Structure):
    _fields_ = [("kind", C.c_int), ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("periodic_x", C.c_int), ("periodic_y", C.c_int),
                ("x0", C.c_double), ("dx", C.c_double), ("y0", C.c_double), ("dy", C.c_double),
                ("radius", C.c_double), ("rotation_rate", C.c_double),
                ("f0", C.c_double), ("beta", C.c_double)]


class ModelDesc(C.Structure):
    _fields_ = [("dt", C.c_double), ("substeps", C.c_int), ("chi", C.c_double),
                ("g", C.c_double), ("alpha", C.c_double), ("beta_s", C.c_double),
                ("T0", C.c_double), ("S0", C.c_double), ("rho0", C.c_double),
                ("nu_h", C.c_double), ("kappa_h", C.c_double), ("nu_z", C.c_double),
                ("kappa_z", C.c_double), ("filter_weights", C.POINTER(C.c_double)),
                ("closure", C.c_int), ("ri_nu0", C.c_double), ("ri_c", C.c_double), ("ri_kconv", C.c_double),
                ("ri_n2c", C.c_double), ("ri_s2min", C.c_double), ("gamma_T", C.c_double), ("gamma_S", C.c_double),
                ("drag_r", C.c_double), ("drag_cd", C.c_double),
                ("eos", C.c_int), ("eos_alpha2", C.c_double), ("eos_gamma", C.c_double), ("advection", C.c_int),
                ("filter_weights_uv", C.POINTER(C.c_double)), ("nu4_h", C.c_double), ("kappa4_h", C.c_double)]


class Fields(C.Structure):
    _fields_ = [(n, C.POINTER(C.c_double)) for n in ("u", "v", "T", "S", "w", "eta", "tau_x", "tau_y",
                                                       "flux_T", "flux_S", "restore_T", "restore_S")]


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_SO)
        _lib.ocn_ref_last_error.restype = C.c_char_p
        _lib.ocn_ref_weno.restype = C.c_double
        _lib.ocn_ref_weno.argtypes = [C.POINTER(C.c_double), C.c_int, C.c_double]
        _lib.ocn_ref_weno_scheme.restype = C.c_double
        _lib.ocn_ref_weno_scheme.argtypes = [C.POINTER(C.c_double), C.c_int, C.c_double, C.c_int]
        _lib.ocn_ref_barotropic_raw.argtypes = [C.c_void_p, C.c_int, C.c_double]
        _lib.ocn_ref_implicit_column.argtypes = [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_ubyte),
                                                 C.c_double, C.POINTER(C.c_double)]
        _lib.ocn_ref_implicit_column_var.argtypes = [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_ubyte),
                                                     C.POINTER(C.c_double), C.POINTER(C.c_double)]
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _bp(a):
    return a.ctypes.data_as(C.POINTER(C.c_ubyte)) if a is not None else None


def _check(rc):
    if rc != 0:
        raise RuntimeError("oracle: " + lib().ocn_ref_last_error().decode())


def num_threads():
    return int(lib().ocn_ref_num_threads())


def set_num_threads(n):
    lib().ocn_ref_set_num_threads(int(n))


def weno(c6, order, vel, scheme=0):
    c = np.ascontiguousarray(c6, dtype=np.float64)
    assert c.size == 6
    if scheme == 0:
        return float(lib().ocn_ref_weno(_dp(c), int(order), float(vel)))
    return float(lib().ocn_ref_weno_scheme(_dp(c), int(order), float(vel), int(scheme)))


def implicit_column(z_faces, open_faces, dt_kappa, phi):
    zf = np.ascontiguousarray(z_faces, dtype=np.float64)
    op = np.ascontiguousarray(open_faces, dtype=np.uint8)
    x = np.array(phi, dtype=np.float64)
    _check(lib().ocn_ref_implicit_column(len(x), _dp(zf), _bp(op), float(dt_kappa), _dp(x)))
    return x


def implicit_column_var(z_faces, open_faces, dt_kappa_faces, phi):
    zf = np.ascontiguousarray(z_faces, dtype=np.float64)
    op = np.ascontiguousarray(open_faces, dtype=np.uint8)
    dk = np.ascontiguousarray(dt_kappa_faces, dtype=np.float64)
    x = np.array(phi, dtype=np.float64)
    assert op.size == len(x) + 1 and dk.size == len(x) + 1
    _check(lib().ocn_ref_implicit_column_var(len(x), _dp(zf), _bp(op), _dp(dk), _dp(x)))
    return x


def filter_weights(M):
    a = np.zeros(M)
    r = C.c_double()
    _check(lib().ocn_ref_filter_weights(int(M), _dp(a), C.byref(r)))
    return a, r.value


class RefGrid:
    def __init__(self, grid, z_faces, depth):
        self.desc = GridDesc(**{k: grid[k] for k, _ in GridDesc._fields_})
        self.nx, self.ny, self.nz = grid["nx"], grid["ny"], grid["nz"]
        zf = np.ascontiguousarray(z_faces, dtype=np.float64)
        h = np.ascontiguousarray(depth, dtype=np.float64)
        assert zf.size == self.nz + 1 and h.shape == (self.ny, self.nx)
        self.h = C.c_void_p()
        _check(lib().ocn_ref_grid_create(C.byref(self.desc), _dp(zf), _dp(h), C.byref(self.h)))

    def masks(self):
        nz, ny, nx = self.nz, self.ny, self.nx
        out = {n: np.zeros((nz, ny, nx), np.uint8) for n in ("wet", "order_x", "order_y", "order_zeta_u", "order_zeta_v")}
        out["order_z"] = np.zeros((nz + 1, ny, nx), np.uint8)
        _check(lib().ocn_ref_get_masks(self.h, _bp(out["wet"]), _bp(out["order_x"]), _bp(out["order_y"]),
                                       _bp(out["order_z"]), _bp(out["order_zeta_u"]), _bp(out["order_zeta_v"])))
        return out

    def metrics(self):
        m = {n: np.zeros(self.ny) for n in ("dxC", "dxF", "AzC", "AzF", "fF")}
        dy = C.c_double()
        _check(lib().ocn_ref_get_metrics(self.h, _dp(m["dxC"]), _dp(m["dxF"]), _dp(m["AzC"]), _dp(m["AzF"]),
                                         _dp(m["fF"]), C.byref(dy)))
        m["dy"] = dy.value
        return m

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.ocn_ref_grid_destroy(self.h)
            self.h = None


class RefModel:
    """Oracle model.  `workload` is a dict from paper_2309_06662_b200.workloads (passed in by the
    caller; this module does not import it)."""

    def __init__(self, workload, filter_weights=None, filter_weights_uv=None):
        self.grid = RefGrid(workload["grid"], workload["z_faces"], workload["depth"])
        p = dict(workload["params"])
        p.pop("precision", None)
        self._fw = None if filter_weights is None else np.ascontiguousarray(filter_weights, dtype=np.float64)
        self._fwuv = None if filter_weights_uv is None else np.ascontiguousarray(filter_weights_uv, dtype=np.float64)
        self.desc = ModelDesc(filter_weights=_dp(self._fw) if self._fw is not None else None,
                              filter_weights_uv=_dp(self._fwuv) if self._fwuv is not None else None, **p)
        self.nx, self.ny, self.nz = self.grid.nx, self.grid.ny, self.grid.nz
        self.h = C.c_void_p()
        _check(lib().ocn_ref_model_create(self.grid.h, C.byref(self.desc), C.byref(self.h)))
        if "fields" in workload:
            self.set_fields(**workload["fields"])

    def set_fields(self, **kw):
        keep = {k: np.ascontiguousarray(v, dtype=np.float64) for k, v in kw.items() if v is not None}
        f = Fields(**{k: _dp(v) for k, v in keep.items()})
        _check(lib().ocn_ref_set_fields(self.h, C.byref(f)))

    def step(self, n=1):
        _check(lib().ocn_ref_time_step(self.h, int(n)))

    def get_fields(self):
        nz, ny, nx = self.nz, self.ny, self.nx
        out = {k: np.zeros((nz, ny, nx)) for k in ("u", "v", "T", "S")}
        out["w"] = np.zeros((nz + 1, ny, nx))
        out["eta"] = np.zeros((ny, nx))
        f = Fields(**{k: _dp(v) for k, v in out.items()})
        _check(lib().ocn_ref_get_fields(self.h, C.byref(f)))
        return out

    def tendencies(self):
        nz, ny, nx = self.nz, self.ny, self.nx
        G = {k: np.zeros((nz, ny, nx)) for k in ("Gu", "Gv", "GT", "GS")}
        _check(lib().ocn_ref_get_tendencies(self.h, _dp(G["Gu"]), _dp(G["Gv"]), _dp(G["GT"]), _dp(G["GS"])))
        return G

    def diagnostics(self):
        nz, ny, nx = self.nz, self.ny, self.nx
        d = dict(p=np.zeros((nz, ny, nx)), U=np.zeros((ny, nx)), V=np.zeros((ny, nx)))
        _check(lib().ocn_ref_get_diagnostics(self.h, _dp(d["p"]), _dp(d["U"]), _dp(d["V"])))
        return d

    def momentum_diagnostics(self):
        nz, ny, nx = self.nz, self.ny, self.nx
        d = dict(zeta=np.zeros((nz, ny, nx)), K=np.zeros((nz, ny, nx)), D=np.zeros((nz, ny, nx)))
        _check(lib().ocn_ref_get_momentum_diagnostics(self.h, _dp(d["zeta"]), _dp(d["K"]), _dp(d["D"])))
        return d

    def mixing(self):
        nz, ny, nx = self.nz, self.ny, self.nx
        d = dict(nu=np.zeros((nz, ny, nx)), kappa=np.zeros((nz, ny, nx)))
        _check(lib().ocn_ref_get_mixing(self.h, _dp(d["nu"]), _dp(d["kappa"])))
        return d

    def barotropic_raw(self, m, dtau):
        _check(lib().ocn_ref_barotropic_raw(self.h, int(m), float(dtau)))

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.ocn_ref_model_destroy(self.h)
            self.h = None
