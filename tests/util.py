"""Helpers shared by the tests: small workload builders (inputs only) and the error metric."""
import copy

import numpy as np

from paper_2309_06662_b200 import workloads as W


def box(nx=16, ny=16, nz=4, *, depth=400.0, dx=1000.0, dy=None, periodic=(1, 1), f0=1e-4, beta=0.0,
        dt=60.0, substeps=20, z_faces=None, **params):
    """Cartesian box at rest with uniform T, S; tests overwrite what they need."""
    dy = dx if dy is None else dy
    zf = W.geometric_z_faces(nz, depth / nz, depth) if z_faces is None else np.asarray(z_faces, float)
    grid = dict(kind=0, nx=nx, ny=ny, nz=nz, periodic_x=periodic[0], periodic_y=periodic[1], x0=0.0, dx=dx,
                y0=0.0, dy=dy, radius=W.EARTH_RADIUS, rotation_rate=W.EARTH_ROTATION, f0=f0, beta=beta)
    p = W._params(64, dt, substeps, 0.0, 0.0)
    p.update(params)
    z3 = np.zeros((nz, ny, nx))
    z2 = np.zeros((ny, nx))
    fields = dict(u=z3.copy(), v=z3.copy(), T=z3 + 10.0, S=z3 + 35.0, eta=z2.copy(), tau_x=z2.copy(), tau_y=z2.copy())
    return dict(name="box", grid=grid, z_faces=zf, depth=np.full((ny, nx), depth), params=p, fields=fields, steps=1)


def rel_linf(a, ref, mask=None):
    """relative L-infinity error normalised by max |ref| (north_star's metric)."""
    a = np.asarray(a, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    d = np.abs(a - ref)
    if mask is not None:
        d = d[mask]
    scale = np.max(np.abs(ref))
    if scale == 0.0:
        return float(d.max()) if d.size else 0.0
    return float(d.max() / scale) if d.size else 0.0


def clone(wl):
    return copy.deepcopy(wl)


# per-field parity margins of the full-size GPU tests; tests/conftest.py prints them in the terminal summary so that the
# driver's log of `pytest -m gpu` shows how far inside the tolerance each case is
PARITY_REPORT = []


def report_parity(case, steps, errs):
    PARITY_REPORT.append("%-58s steps %3d  " % (case, steps) + "  ".join("%s %.2e" % (n, e) for n, e in errs.items()))
