"""Thin ctypes binding over the C ABI of libocn.so (include/ocn.h): argument marshalling only.

Function names mirror the C entry points (ocn_grid_create, ocn_model_create, ocn_set_fields,
ocn_time_step, ocn_get_fields, ocn_get_masks, ...); `Model` is a convenience wrapper that owns the
handles.  torch is used only for pinned host buffers / streams by callers; this module needs
numpy + ctypes.  There is no CPU fallback: a missing library or GPU raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libocn.so")
_lib = None

OCN_OK = 0


class ocn_grid_desc(C.Structure):
    _fields_ = [("kind", C.c_int), ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("periodic_x", C.c_int), ("periodic_y", C.c_int),
                ("x0", C.c_double), ("dx", C.c_double), ("y0", C.c_double), ("dy", C.c_double),
                ("radius", C.c_double), ("rotation_rate", C.c_double), ("f0", C.c_double), ("beta", C.c_double),
                ("j_offset", C.c_int), ("ny_global", C.c_int)]


class ocn_model_desc(C.Structure):
    _fields_ = [("precision", C.c_int), ("dt", C.c_double), ("substeps", C.c_int), ("chi", C.c_double),
                ("g", C.c_double), ("alpha", C.c_double), ("beta_s", C.c_double), ("T0", C.c_double),
                ("S0", C.c_double), ("rho0", C.c_double), ("nu_h", C.c_double), ("kappa_h", C.c_double),
                ("nu_z", C.c_double), ("kappa_z", C.c_double), ("filter_weights", C.POINTER(C.c_double)),
                ("device", C.c_int), ("stream", C.c_void_p),
                ("closure", C.c_int), ("ri_nu0", C.c_double), ("ri_c", C.c_double), ("ri_kconv", C.c_double),
                ("ri_n2c", C.c_double), ("ri_s2min", C.c_double), ("gamma_T", C.c_double), ("gamma_S", C.c_double),
                ("drag_r", C.c_double), ("drag_cd", C.c_double),
                ("eos", C.c_int), ("eos_alpha2", C.c_double), ("eos_gamma", C.c_double), ("advection", C.c_int),
                ("filter_weights_uv", C.POINTER(C.c_double)), ("nu4_h", C.c_double), ("kappa4_h", C.c_double),
                ("workspace", C.c_void_p), ("workspace_bytes", C.c_ulonglong)]


class ocn_fields(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("u", "v", "T", "S", "w", "eta", "tau_x", "tau_y",
                                          "flux_T", "flux_S", "restore_T", "restore_S")] + [("on_device", C.c_int)]


class ocn_peer(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("precision", C.c_int), ("sx", C.c_int), ("sy", C.c_int),
                ("device", C.c_int), ("ptr", C.c_void_p * 3), ("ipc", (C.c_ubyte * 64) * 3), ("ipc_offset", C.c_ulonglong * 3)]


EXPORTS = ["ocn_grid_create", "ocn_grid_destroy", "ocn_model_create", "ocn_model_destroy", "ocn_set_fields",
           "ocn_time_step", "ocn_get_fields", "ocn_synchronize", "ocn_get_masks", "ocn_model_info",
           "ocn_get_debug", "ocn_last_error", "ocn_version", "ocn_profile_enable", "ocn_profile_read",
           "ocn_stage_name", "ocn_get_mixing", "ocn_get_fields_async", "ocn_wait", "ocn_tune", "ocn_selftest_division", "ocn_get_timeline",
           "ocn_get_mixing_noalloc", "ocn_noalloc_scratch_bytes",
           "ocn_step_parts", "ocn_step_part", "ocn_rows_bytes", "ocn_pack_rows", "ocn_unpack_rows", "ocn_band_overlap",
           "ocn_peer_export", "ocn_peer_attach",
           "ocn_checkpoint_bytes", "ocn_checkpoint_save", "ocn_checkpoint_load", "ocn_check_finite", "ocn_model_workspace_bytes"]
ROWS_STATE, ROWS_FORCING, ROWS_BAROTROPIC_0, ROWS_BAROTROPIC_1, ROWS_STATE_2D = 0, 1, 2, 3, 4
NSTAGES = 4


def lib():
    """Loads libocn.so (built in-tree by paper_2309_06662_b200.build); fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise RuntimeError(f"{_SO} is missing: run `python -m paper_2309_06662_b200.build` (no CPU fallback)")
        L = C.CDLL(_SO)
        L.ocn_last_error.restype = C.c_char_p
        L.ocn_version.restype = C.c_char_p
        vp = C.c_void_p
        L.ocn_grid_create.argtypes = [C.POINTER(ocn_grid_desc), vp, vp, C.POINTER(vp)]
        L.ocn_grid_destroy.argtypes = [vp]
        L.ocn_model_create.argtypes = [vp, C.POINTER(ocn_model_desc), C.POINTER(vp)]
        L.ocn_model_destroy.argtypes = [vp]
        L.ocn_model_workspace_bytes.argtypes = [vp, C.POINTER(ocn_model_desc), C.POINTER(C.c_ulonglong)]
        L.ocn_set_fields.argtypes = [vp, C.POINTER(ocn_fields)]
        L.ocn_time_step.argtypes = [vp, C.c_int]
        L.ocn_get_fields.argtypes = [vp, C.POINTER(ocn_fields)]
        L.ocn_synchronize.argtypes = [vp]
        L.ocn_get_fields_async.argtypes = [vp, C.POINTER(ocn_fields), C.POINTER(C.c_ulonglong)]
        L.ocn_wait.argtypes = [vp, C.c_ulonglong]
        L.ocn_tune.argtypes = [vp, C.c_char_p, C.c_double]
        L.ocn_get_timeline.argtypes = [vp, C.POINTER(C.c_double), C.c_int]
        L.ocn_selftest_division.argtypes = [C.c_int, C.c_ulonglong, C.c_ulonglong, C.POINTER(C.c_ulonglong)]
        L.ocn_get_masks.argtypes = [vp] + [vp] * 6
        L.ocn_model_info.argtypes = [vp, C.POINTER(C.c_int), C.POINTER(C.c_ulonglong)]
        L.ocn_get_debug.argtypes = [vp] + [vp] * 6
        L.ocn_get_mixing.argtypes = [vp, vp, vp]
        L.ocn_get_mixing_noalloc.argtypes = [vp, vp, vp]
        L.ocn_noalloc_scratch_bytes.restype = C.c_ulonglong
        L.ocn_profile_enable.argtypes = [vp, C.c_int]
        L.ocn_profile_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong), C.c_int]
        L.ocn_step_parts.argtypes = [vp, C.POINTER(C.c_int)]
        L.ocn_step_part.argtypes = [vp, C.c_int]
        L.ocn_rows_bytes.argtypes = [vp, C.c_int, C.c_int, C.POINTER(C.c_ulonglong)]
        L.ocn_pack_rows.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp]
        L.ocn_unpack_rows.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp]
        L.ocn_band_overlap.argtypes = [C.c_int, C.c_int]
        L.ocn_checkpoint_bytes.argtypes = [vp, C.POINTER(C.c_ulonglong)]
        L.ocn_checkpoint_save.argtypes = [vp, vp]
        L.ocn_checkpoint_load.argtypes = [vp, vp, C.c_ulonglong]
        L.ocn_check_finite.argtypes = [vp, C.POINTER(C.c_ulonglong)]
        L.ocn_peer_export.argtypes = [vp, C.POINTER(ocn_peer)]
        L.ocn_peer_attach.argtypes = [vp, C.c_int, C.POINTER(ocn_peer), C.c_int, C.c_int, C.c_int, C.c_int]
        L.ocn_stage_name.restype = C.c_char_p
        L.ocn_stage_name.argtypes = [C.c_int]
        _lib = L
    return _lib


def selftest_division(n, seed=1, device=0):
    """ocn_selftest_division: number of operand pairs (of n) on which the fast fp64 quotient differs from __ddiv_rn."""
    bad = C.c_ulonglong()
    _check(lib().ocn_selftest_division(int(device), int(n), int(seed), C.byref(bad)))
    return bad.value


def band_overlap(precision, substeps):
    """ocn_band_overlap: overlap rows a latitude band needs on each inner side."""
    h = int(lib().ocn_band_overlap(int(precision), int(substeps)))
    if h < 0:
        raise ValueError("band_overlap: precision must be 32 or 64 and substeps >= 1")
    return h


def _check(rc):
    if rc != OCN_OK:
        raise RuntimeError(f"libocn status {rc}: {lib().ocn_last_error().decode()}")


def _ptr(a):
    return None if a is None else C.c_void_p(a.ctypes.data)


class Grid:
    def __init__(self, grid, z_faces, depth):
        self.desc = ocn_grid_desc(**{k: grid.get(k, 0) if k in ("j_offset", "ny_global") else grid[k] for k, _ in ocn_grid_desc._fields_})
        self.nx, self.ny, self.nz = int(grid["nx"]), int(grid["ny"]), int(grid["nz"])
        zf = np.ascontiguousarray(z_faces, dtype=np.float64)
        h = np.ascontiguousarray(depth, dtype=np.float64)
        if zf.size != self.nz + 1 or h.shape != (self.ny, self.nx):
            raise ValueError("z_faces / depth shape mismatch")
        self.h = C.c_void_p()
        _check(lib().ocn_grid_create(C.byref(self.desc), _ptr(zf), _ptr(h), C.byref(self.h)))

    def masks(self):
        nz, ny, nx = self.nz, self.ny, self.nx
        names = ("wet", "order_x", "order_y", "order_z", "order_zeta_u", "order_zeta_v")
        out = {n: np.zeros((nz + 1 if n == "order_z" else nz, ny, nx), np.uint8) for n in names}
        _check(lib().ocn_get_masks(self.h, *[_ptr(out[n]) for n in names]))
        return out

    def close(self):
        if getattr(self, "h", None):
            lib().ocn_grid_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Model:
    """ocn_model_create + ocn_set_fields on a workload dict (paper_2309_06662_b200.workloads)."""

    def __init__(self, workload, device=0, stream=None, filter_weights=None, set_fields=True, filter_weights_uv=None,
                 workspace=None):
        """workspace: None (the library allocates), or a callable nbytes -> (handle, device pointer) that provides the model's
        device memory (e.g. a torch uint8 tensor and its data_ptr()); the handle is kept alive with the model."""
        self.grid = Grid(workload["grid"], workload["z_faces"], workload["depth"])
        p = dict(workload["params"])
        self.precision = int(p["precision"])
        self.dtype = np.float32 if self.precision == 32 else np.float64
        self._fw = None if filter_weights is None else np.ascontiguousarray(filter_weights, dtype=np.float64)
        fw = self._fw.ctypes.data_as(C.POINTER(C.c_double)) if self._fw is not None else None
        self._fwuv = None if filter_weights_uv is None else np.ascontiguousarray(filter_weights_uv, dtype=np.float64)
        fwuv = self._fwuv.ctypes.data_as(C.POINTER(C.c_double)) if self._fwuv is not None else None
        self.desc = ocn_model_desc(filter_weights=fw, filter_weights_uv=fwuv, device=int(device), stream=stream, **p)
        self.nx, self.ny, self.nz = self.grid.nx, self.grid.ny, self.grid.nz
        self._workspace = None
        if workspace is not None:
            need = self.workspace_bytes()
            got = workspace(need)                          # (handle, pointer) or (handle, pointer, bytes actually provided)
            self._workspace, ptr = got[0], got[1]
            self.desc.workspace, self.desc.workspace_bytes = int(ptr), int(got[2]) if len(got) > 2 else need
        self.h = C.c_void_p()
        _check(lib().ocn_model_create(self.grid.h, C.byref(self.desc), C.byref(self.h)))
        if set_fields and "fields" in workload:
            self.set_fields(**workload["fields"])

    def workspace_bytes(self):
        """ocn_model_workspace_bytes for this grid and these parameters (host-only)."""
        n = C.c_ulonglong()
        _check(lib().ocn_model_workspace_bytes(self.grid.h, C.byref(self.desc), C.byref(n)))
        return n.value

    # -- host numpy arrays ---------------------------------------------------------------
    def set_fields(self, **kw):
        keep = {k: np.ascontiguousarray(v, dtype=self.dtype) for k, v in kw.items() if v is not None}
        f = ocn_fields(on_device=0, **{k: v.ctypes.data for k, v in keep.items()})
        _check(lib().ocn_set_fields(self.h, C.byref(f)))

    def get_fields(self, names=("u", "v", "T", "S", "w", "eta")):
        nz, ny, nx = self.nz, self.ny, self.nx
        shp = {"w": (nz + 1, ny, nx), "eta": (ny, nx), "tau_x": (ny, nx), "tau_y": (ny, nx)}
        out = {k: np.zeros(shp.get(k, (nz, ny, nx)), self.dtype) for k in names}
        f = ocn_fields(on_device=0, **{k: v.ctypes.data for k, v in out.items()})
        _check(lib().ocn_get_fields(self.h, C.byref(f)))
        return out

    # -- raw pointers (pinned host or device memory owned by the caller, e.g. torch tensors) ----
    def set_fields_ptr(self, on_device=False, **ptrs):
        f = ocn_fields(on_device=int(on_device), **{k: int(v) for k, v in ptrs.items()})
        _check(lib().ocn_set_fields(self.h, C.byref(f)))

    def get_fields_ptr(self, on_device=False, **ptrs):
        f = ocn_fields(on_device=int(on_device), **{k: int(v) for k, v in ptrs.items()})
        _check(lib().ocn_get_fields(self.h, C.byref(f)))

    def get_fields_async_ptr(self, on_device=False, **ptrs):
        """ocn_get_fields_async: returns a ticket; the buffers are valid after wait(ticket)."""
        f = ocn_fields(on_device=int(on_device), **{k: int(v) for k, v in ptrs.items()})
        t = C.c_ulonglong()
        _check(lib().ocn_get_fields_async(self.h, C.byref(f), C.byref(t)))
        return t.value

    def wait(self, ticket):
        _check(lib().ocn_wait(self.h, int(ticket)))

    def tune(self, key, value):
        _check(lib().ocn_tune(self.h, key.encode(), float(value)))

    def timeline(self, reset=True):
        """ocn_get_timeline (diagnostic builds): {phase: cycles per iteration, per warp}."""
        buf = (C.c_double * 64)()
        _check(lib().ocn_get_timeline(self.h, buf, int(bool(reset))))
        names = ("prologue+barrier_wait", "tma_wait", "phase1", "faces", "partB", "barrier_issue")
        return [{n: buf[w * 8 + q] / max(buf[w * 8 + 6], 1.0) for q, n in enumerate(names)} for w in range(8)]

    def time_step(self, n=1):
        _check(lib().ocn_time_step(self.h, int(n)))

    def synchronize(self):
        _check(lib().ocn_synchronize(self.h))

    # -- the step in parts and the rows a neighbouring band needs (include/ocn.h, "Latitude bands") ----
    def step_parts(self):
        n = C.c_int()
        _check(lib().ocn_step_parts(self.h, C.byref(n)))
        return n.value

    def step_part(self, part):
        _check(lib().ocn_step_part(self.h, int(part)))

    def rows_bytes(self, group, nrows):
        b = C.c_ulonglong()
        _check(lib().ocn_rows_bytes(self.h, int(group), int(nrows), C.byref(b)))
        return b.value

    def pack_rows(self, group, j_begin, nrows, dst_device_ptr):
        _check(lib().ocn_pack_rows(self.h, int(group), int(j_begin), int(nrows), C.c_void_p(int(dst_device_ptr))))

    # -- checkpoint / resume, finite check ----
    def checkpoint(self):
        """ocn_checkpoint_save into a new numpy uint8 array (everything a bit-exact resume needs)."""
        n = C.c_ulonglong()
        _check(lib().ocn_checkpoint_bytes(self.h, C.byref(n)))
        buf = np.empty(n.value, np.uint8)
        _check(lib().ocn_checkpoint_save(self.h, _ptr(buf)))
        return buf

    def restore(self, blob):
        buf = np.ascontiguousarray(blob, dtype=np.uint8)
        _check(lib().ocn_checkpoint_load(self.h, _ptr(buf), buf.size))

    def nonfinite(self):
        """ocn_check_finite: number of NaN / infinite words in u, v, T, S, eta."""
        n = C.c_ulonglong()
        _check(lib().ocn_check_finite(self.h, C.byref(n)))
        return n.value

    def peer_export(self):
        """ocn_peer_export as bytes (plain data: addresses for this process, CUDA IPC handles for another)."""
        p = ocn_peer()
        _check(lib().ocn_peer_export(self.h, C.byref(p)))
        return bytes(p)

    def peer_attach(self, side, peer_bytes, my_first_row, peer_first_row, rows, same_process):
        p = ocn_peer.from_buffer_copy(peer_bytes)
        _check(lib().ocn_peer_attach(self.h, int(side), C.byref(p), int(my_first_row), int(peer_first_row), int(rows),
                                     int(bool(same_process))))

    def unpack_rows(self, group, j_begin, nrows, src_device_ptr):
        _check(lib().ocn_unpack_rows(self.h, int(group), int(j_begin), int(nrows), C.c_void_p(int(src_device_ptr))))

    def info(self):
        n, b = C.c_int(), C.c_ulonglong()
        _check(lib().ocn_model_info(self.h, C.byref(n), C.byref(b)))
        return dict(launches_per_step=n.value, device_bytes=b.value)

    def profile_enable(self, on=True):
        _check(lib().ocn_profile_enable(self.h, int(bool(on))))

    def profile_read(self, reset=True):
        ms = (C.c_double * NSTAGES)()
        n = (C.c_longlong * NSTAGES)()
        _check(lib().ocn_profile_read(self.h, ms, n, int(bool(reset))))
        return {lib().ocn_stage_name(q).decode(): dict(ms=ms[q], launches=n[q]) for q in range(NSTAGES)}

    def debug(self):
        nz, ny, nx = self.nz, self.ny, self.nx
        d = {k: np.zeros((nz, ny, nx)) for k in ("Gu", "Gv", "GT", "GS")}
        d["U"] = np.zeros((ny, nx)); d["V"] = np.zeros((ny, nx))
        _check(lib().ocn_get_debug(self.h, *[_ptr(d[k]) for k in ("Gu", "Gv", "GT", "GS", "U", "V")]))
        return d

    def mixing(self):
        nz, ny, nx = self.nz, self.ny, self.nx
        d = dict(nu=np.zeros((nz, ny, nx)), kappa=np.zeros((nz, ny, nx)))
        _check(lib().ocn_get_mixing(self.h, _ptr(d["nu"]), _ptr(d["kappa"])))
        return d

    def mixing_noalloc(self):
        """ocn_get_mixing_noalloc: the same diagnostic through the static scratch array (no device allocation)."""
        nz, ny, nx = self.nz, self.ny, self.nx
        d = dict(nu=np.zeros((nz, ny, nx)), kappa=np.zeros((nz, ny, nx)))
        _check(lib().ocn_get_mixing_noalloc(self.h, _ptr(d["nu"]), _ptr(d["kappa"])))
        return d

    def close(self):
        if getattr(self, "h", None):
            lib().ocn_model_destroy(self.h)
            self.h = None
        self.grid.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
