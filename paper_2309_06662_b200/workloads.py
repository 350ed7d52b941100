"""Seeded synthetic workloads (inputs only) for the hydrostatic free-surface time step.

This module is the ONE piece shared by the CUDA path and the CPU oracle: it draws the
seeded inputs (grids, bathymetry, initial fields, wind stress) for the five configurations
of BASELINE.json and holds none of the method's arithmetic (no stencils, no scans, no
solves, no masks).  It imports numpy only.

The shapes stand in for the paper's workloads (§6: near-global
75S-75N latitude-longitude domains, periodic in longitude, 48-100 stretched levels,
realistic bathymetry) whose data (ECCO2 forcing, real bathymetry) are not
available here.  Recipes follow SURVEY.md §8(d) and are restated in DESIGN.md §4.

Every workload is a plain dict:

    grid   : dict(kind, nx, ny, nz, periodic_x, periodic_y, x0, dx, y0, dy, radius,
                  rotation_rate, f0, beta)
    z_faces: float64[nz+1], increasing, z_faces[nz] == 0
    depth  : float64[ny, nx]  bottom depth in metres (>= 0, 0 = land)
    params : dict(precision, dt, substeps, chi, g, alpha, beta_s, T0, S0, rho0,
                  nu_h, kappa_h, nu_z, kappa_z [, closure, ri_nu0, ri_c, ri_kconv, ri_n2c, ri_s2min])
    fields : dict(u, v, T, S [nz,ny,nx]; eta, tau_x, tau_y [ny,nx])  float64, already
             rounded to the run precision (the fp64 oracle receives the rounded values)
    steps  : number of baroclinic steps the configuration asks for
    name   : label
"""
from __future__ import annotations

import numpy as np

SEED_BASE = 6662

EARTH_RADIUS = 6371000.0
EARTH_ROTATION = 7.292115e-5
GRAVITY = 9.80665


def _params(precision, dt, substeps, nu_h, kappa_h, beta_s=8e-4):
    return dict(precision=int(precision), dt=float(dt), substeps=int(substeps), chi=0.1,
                g=GRAVITY, alpha=2e-4, beta_s=float(beta_s), T0=10.0, S0=35.0, rho0=1025.0,
                nu_h=float(nu_h), kappa_h=float(kappa_h), nu_z=1e-4, kappa_z=1e-5)


def with_ri_closure(wl, nu0=5e-3, c=5.0, kconv=0.1, n2c=1e-5, s2min=1e-10):
    """Switches a workload to the Richardson-number-based vertical mixing closure (the one used in
    all of the paper's runs; parameters of the reading in DESIGN.md §3.12): only the
    parameter dict changes, nu_z / kappa_z become the background values."""
    wl["params"].update(closure=1, ri_nu0=float(nu0), ri_c=float(c), ri_kconv=float(kconv), ri_n2c=float(n2c),
                        ri_s2min=float(s2min))
    wl["name"] = wl.get("name", "") + "+ri"
    return wl


def with_nonlinear_eos(wl, alpha2=1e-5, gamma=2e-4):
    """Switches a workload to the nonlinear equation of state of DESIGN.md §3.16: thermobaric
    (alpha grows with depth at rate gamma [1/m]) and cabbeling (alpha2 [1/K^2]) terms; parameters only."""
    wl["params"].update(eos=1, eos_alpha2=float(alpha2), eos_gamma=float(gamma))
    wl["name"] = wl.get("name", "") + "+eos"
    return wl


def with_weno_z(wl):
    """Switches a workload to WENO-Z nonlinear weights; parameters only."""
    wl["params"].update(advection=1)
    wl["name"] = wl.get("name", "") + "+wenoz"
    return wl


def with_surface_forcing(wl, seed=SEED_BASE + 40, heat=2e-5, salt=2e-6, piston=1e-5):
    """Adds seeded surface tracer forcing to a workload (the realistic runs are "forced by realistic
    surface momentum, heat, and salinity fluxes"; ECCO2 data are not available, these stand in for their shape):
    smooth kinematic fluxes flux_T [K m/s] (|.| <= heat, about 80 W/m^2), flux_S [psu m/s], and restoring of the top
    cell toward the initial surface T, S shifted by a smooth anomaly, with piston velocity `piston` [m/s] (about 1 m/day).
    Inputs only: no method arithmetic."""
    rng = np.random.default_rng(seed)
    g, prec = wl["grid"], wl["params"]["precision"]
    ny, nx = g["ny"], g["nx"]
    per = bool(g["periodic_x"])
    f = wl["fields"]
    f["flux_T"] = _round_to(prec, heat * _low_mode_field(rng, ny, nx, 3, periodic=per))
    f["flux_S"] = _round_to(prec, salt * _low_mode_field(rng, ny, nx, 3, periodic=per))
    f["restore_T"] = _round_to(prec, f["T"][-1] + 0.5 * _low_mode_field(rng, ny, nx, 2, periodic=per))
    f["restore_S"] = _round_to(prec, f["S"][-1] + 0.05 * _low_mode_field(rng, ny, nx, 2, periodic=per))
    wl["params"].update(gamma_T=float(piston), gamma_S=float(piston))
    wl["name"] = wl.get("name", "") + "+sfc"
    return wl


def _round_to(precision, a):
    a = np.asarray(a, dtype=np.float64)
    if precision == 32:
        return a.astype(np.float32).astype(np.float64)
    return a


def geometric_z_faces(nz, top_dz, total_depth):
    """nz layers whose thickness grows geometrically downward from top_dz at the surface and
    sums to total_depth (the ratio is solved for, so the sum is exact)."""
    if abs(nz * top_dz - total_depth) < 1e-9 * total_depth:
        dz = np.full(nz, top_dz)
    else:
        lo, hi = 1.0 + 1e-12, 4.0
        for _ in range(200):
            r = 0.5 * (lo + hi)
            s = top_dz * (r ** nz - 1.0) / (r - 1.0)
            if s < total_depth:
                lo = r
            else:
                hi = r
        r = 0.5 * (lo + hi)
        dz = top_dz * r ** np.arange(nz)          # index 0 = surface layer
    zf = np.zeros(nz + 1)
    zf[:nz] = -np.cumsum(dz)[::-1]                # zf[0] = -total, zf[nz] = 0
    zf[0] = -float(total_depth)
    zf[nz] = 0.0
    return zf


def _z_centres(zf):
    return 0.5 * (zf[:-1] + zf[1:])


def _low_mode_field(rng, ny, nx, nmodes, periodic=True):
    """Smooth random 2-D field: sum over wavenumbers 1..nmodes per axis of cosines with seeded
    amplitude and phase.  Returns values on cell centres, normalised to max |.| = 1."""
    y = (np.arange(ny) + 0.5) / ny
    x = (np.arange(nx) + 0.5) / nx
    f = np.zeros((ny, nx))
    for ky in range(1, nmodes + 1):
        for kx in range(1, nmodes + 1):
            a = rng.standard_normal()
            px, py = rng.uniform(0, 2 * np.pi, size=2)
            f += a * np.cos(2 * np.pi * kx * x[None, :] + px) * np.cos(2 * np.pi * ky * y[:, None] + py)
    return f / np.max(np.abs(f))


def fractal_field(rng, ny, nx, slope=-2.0):
    """Seeded Gaussian noise filtered in Fourier space to a power spectrum ~ K^slope
    (K = horizontal wavenumber magnitude in index space; doubly periodic FFT)."""
    noise = rng.standard_normal((ny, nx))
    fk = np.fft.rfft2(noise)
    ky = np.fft.fftfreq(ny)[:, None] * ny
    kx = np.fft.rfftfreq(nx)[None, :] * nx
    K = np.sqrt(kx * kx + ky * ky)
    K[0, 0] = 1.0
    fk *= K ** (0.5 * slope)
    fk[0, 0] = 0.0
    out = np.fft.irfft2(fk, s=(ny, nx))
    return out / out.std()


# ------------------------------------------------------------------------------------------
# config 0: doubly periodic f-plane box
# ------------------------------------------------------------------------------------------
def config0(nx=32, ny=32, nz=8, steps=10, seed=SEED_BASE + 0):
    rng = np.random.default_rng(np.random.PCG64(seed))
    Hd = 400.0
    zf = geometric_z_faces(nz, Hd / nz, Hd)
    zc = _z_centres(zf)
    grid = dict(kind=0, nx=nx, ny=ny, nz=nz, periodic_x=1, periodic_y=1, x0=0.0, dx=1000.0,
                y0=0.0, dy=1000.0, radius=EARTH_RADIUS, rotation_rate=EARTH_ROTATION,
                f0=1e-4, beta=0.0)
    depth = np.full((ny, nx), Hd)
    T = 10.0 + 0.02 * (zc[:, None, None] + Hd) + 0.01 * rng.standard_normal((nz, ny, nx))
    S = np.full((nz, ny, nx), 35.0)
    prof = 0.5 * (1.0 + np.cos(np.pi * zc / Hd))
    u2 = _low_mode_field(rng, ny, nx, 4)
    v2 = _low_mode_field(rng, ny, nx, 4)
    u = 0.1 * u2[None] * prof[:, None, None]
    v = 0.1 * v2[None] * prof[:, None, None]
    z2 = np.zeros((ny, nx))
    fields = dict(u=u, v=v, T=T, S=S, eta=z2.copy(), tau_x=z2.copy(), tau_y=z2.copy())
    params = _params(64, 60.0, 20, 10.0, 1.0, beta_s=0.0)
    return dict(name="cfg0_fplane_box", grid=grid, z_faces=zf, depth=depth, params=params,
                fields={k: _round_to(64, a) for k, a in fields.items()}, steps=steps)


# ------------------------------------------------------------------------------------------
# config 1: closed beta-plane basin with smooth bathymetry and zonal wind
# ------------------------------------------------------------------------------------------
def config1(nx=256, ny=256, nz=32, steps=100, seed=SEED_BASE + 1):
    rng = np.random.default_rng(np.random.PCG64(seed))
    Hd = 4000.0
    zf = geometric_z_faces(nz, 10.0, Hd)
    zc = _z_centres(zf)
    dx = 5000.0 * 256.0 / nx
    grid = dict(kind=0, nx=nx, ny=ny, nz=nz, periodic_x=0, periodic_y=0, x0=0.0, dx=dx,
                y0=0.0, dy=dx, radius=EARTH_RADIUS, rotation_rate=EARTH_ROTATION,
                f0=1e-4, beta=2e-11)
    bump = _low_mode_field(rng, ny, nx, 2)                    # 4 low seeded modes
    depth = 3000.0 + 1000.0 * bump                            # 2-4 km
    depth[0, :] = depth[-1, :] = 0.0                          # outer ring of land cells
    depth[:, 0] = depth[:, -1] = 0.0
    T = np.broadcast_to((2.0 + 18.0 * np.exp(zc / 800.0))[:, None, None], (nz, ny, nx)).copy()
    S = np.broadcast_to((35.0 - np.exp(zc / 500.0))[:, None, None], (nz, ny, nx)).copy()
    yc = (np.arange(ny) + 0.5) / ny
    tau_x = np.broadcast_to((0.1 * np.cos(np.pi * yc))[:, None], (ny, nx)).copy()
    z3 = np.zeros((nz, ny, nx))
    z2 = np.zeros((ny, nx))
    fields = dict(u=z3.copy(), v=z3.copy(), T=T, S=S, eta=z2.copy(), tau_x=tau_x, tau_y=z2.copy())
    params = _params(64, 300.0, 30, 100.0, 10.0)
    return dict(name="cfg1_double_gyre", grid=grid, z_faces=zf, depth=depth, params=params,
                fields={k: _round_to(64, a) for k, a in fields.items()}, steps=steps)


# ------------------------------------------------------------------------------------------
# configs 2-4: near-global latitude-longitude grids with fractal immersed bathymetry
# ------------------------------------------------------------------------------------------
def latlon_bathymetry(rng, ny, nx, max_depth=6000.0, land_fraction=0.30):
    F = fractal_field(rng, ny, nx, slope=-2.0)
    q_land = np.quantile(F, land_fraction)
    q_hi = np.quantile(F, 0.99)
    depth = np.clip(max_depth * (F - q_land) / (q_hi - q_land), 50.0, max_depth)
    depth[F < q_land] = 0.0
    return depth


def aquaplanet_bathymetry(ny, nx, max_depth=6000.0, ridge_height=4000.0, ridge_width_deg=8.0):
    """Idealised bathymetry of the paper's aqua-planet suite: a flat 6 km floor with two
    meridional (pole-to-pole) Gaussian ridges, 180 degrees apart; no land."""
    lon = (np.arange(nx) + 0.5) * 360.0 / nx
    def ridge(l0):
        d = np.minimum(np.abs(lon - l0), 360.0 - np.abs(lon - l0))
        return np.exp(-0.5 * (d / ridge_width_deg) ** 2)
    h = max_depth - ridge_height * np.maximum(ridge(90.0), ridge(270.0))
    return np.broadcast_to(h[None, :], (ny, nx)).copy()


def latlon(nx, ny, nz, *, dt, substeps, steps, nu_h, kappa_h, precision, seed, name,
           noise=True, lat0=-75.0, lat1=75.0, window=None, bathymetry="fractal"):
    """Near-global lat-lon workload.  `window=(j0, j1, i0, i1)` cuts a sub-window out of the
    full-size fields (identical values) and turns it into a closed box: not periodic, and the
    bathymetry is used as is (the library treats non-periodic edges as land)."""
    rng = np.random.default_rng(np.random.PCG64(seed))
    dlat = (lat1 - lat0) / ny
    dlon = 360.0 / nx
    zf = geometric_z_faces(nz, 10.0, 6000.0)
    zc = _z_centres(zf)
    depth = latlon_bathymetry(rng, ny, nx) if bathymetry == "fractal" else aquaplanet_bathymetry(ny, nx)
    latc = np.deg2rad(lat0 + (np.arange(ny) + 0.5) * dlat)
    # wind stress: zonal 0.1*cos(3*lat) plus seeded low modes (periodic in longitude)
    tx_modes = _low_mode_field(rng, ny, nx, 3)
    ty_modes = _low_mode_field(rng, ny, nx, 3)
    tau_x = 0.1 * np.cos(3.0 * latc)[:, None] + 0.02 * tx_modes
    tau_y = 0.02 * ty_modes

    if window is None:
        j0, j1, i0, i1 = 0, ny, 0, nx
    else:
        j0, j1, i0, i1 = window
    wny, wnx = j1 - j0, i1 - i0
    cos2 = (np.cos(latc[j0:j1]) ** 2)[:, None]
    T = np.empty((nz, wny, wnx))
    S = np.empty((nz, wny, wnx))
    for k in range(nz):                       # level by level: full-size noise, keep the window
        # statically stable everywhere: warm and fresh at the surface (dT/dz > 0, dS/dz < 0 at every
        # latitude), 5 K of stratification left at the poleward walls; the noise decays with depth so
        # that it never overturns the weak abyssal stratification
        Tk = 2.0 + (5.0 + 20.0 * cos2) * np.exp(zc[k] / 800.0)
        Sk = 35.0 - cos2 * np.exp(zc[k] / 500.0)
        damp = np.exp(zc[k] / 2000.0)
        if noise:
            nT = rng.standard_normal((ny, nx), dtype=np.float32)[j0:j1, i0:i1]
            nS = rng.standard_normal((ny, nx), dtype=np.float32)[j0:j1, i0:i1]
            T[k] = Tk + 0.01 * damp * nT
            S[k] = Sk + 0.001 * damp * nS
        else:
            T[k] = Tk
            S[k] = Sk
    grid = dict(kind=1, nx=wnx, ny=wny, nz=nz, periodic_x=1 if window is None else 0,
                periodic_y=0, x0=i0 * dlon, dx=dlon, y0=lat0 + j0 * dlat, dy=dlat,
                radius=EARTH_RADIUS, rotation_rate=EARTH_ROTATION, f0=0.0, beta=0.0)
    z3 = np.zeros((nz, wny, wnx))
    fields = dict(u=z3, v=z3.copy(), T=T, S=S, eta=np.zeros((wny, wnx)),
                  tau_x=tau_x[j0:j1, i0:i1].copy(), tau_y=tau_y[j0:j1, i0:i1].copy())
    params = _params(precision, dt, substeps, nu_h, kappa_h)
    return dict(name=name, grid=grid, z_faces=zf, depth=depth[j0:j1, i0:i1].copy(), params=params,
                fields={k: _round_to(precision, a) for k, a in fields.items()}, steps=steps)


def config2(nx=1440, ny=600, nz=50, steps=50, precision=64, seed=SEED_BASE + 2, window=None):
    scale = 1440.0 / nx       # reduced-resolution analogues: dt ~ resolution, capped at 1200 s (f dt < 0.2)
    return latlon(nx, ny, nz, dt=min(540.0 * scale, 1200.0), substeps=30, steps=steps, nu_h=1000.0 * scale,
                  kappa_h=100.0 * scale, precision=precision, seed=seed,
                  name="cfg2_latlon_quarter_deg" if precision == 64 else "cfg3_latlon_quarter_deg_fp32",
                  window=window)


def config3(nx=1440, ny=600, nz=50, steps=50, window=None):
    # "same grid and seeded fields as config 2" -> config 2's seed, values rounded to fp32
    return config2(nx, ny, nz, steps, precision=32, seed=SEED_BASE + 2, window=window)


def config4(nx=2880, ny=1200, nz=100, steps=20, seed=SEED_BASE + 4, window=None, precision=32):
    scale = 2880.0 / nx
    return latlon(nx, ny, nz, dt=min(270.0 * scale, 1200.0), substeps=40, steps=steps, nu_h=500.0 * scale,
                  kappa_h=50.0 * scale, precision=precision, seed=seed,
                  name="cfg4_latlon_eighth_deg_fp32", window=window)


def aquaplanet(nx=2160, ny=900, nz=100, steps=20, precision=32, seed=SEED_BASE + 5, window=None):
    """the aqua-planet workload of the paper's weak-scaling suite at
    its per-GPU resolution of 1/6 degree x 100 levels: two meridional ridges, no land, the same seeded T/S profiles
    and wind stress as the realistic-shape configurations.  Not a BASELINE.json config; used as a second bench workload
    (every cell is wet) and a parity case."""
    scale = 2160.0 / nx
    return latlon(nx, ny, nz, dt=min(360.0 * scale, 1200.0), substeps=40, steps=steps, nu_h=700.0 * scale,
                  kappa_h=70.0 * scale, precision=precision, seed=seed, name="ap_aquaplanet_sixth_deg",
                  window=window, bathymetry="aquaplanet")


def tile_patch_planet(w=16, h=4, nx=1440, ny=600, nz=100, tile=(32, 8), steps=10, precision=32, seed=SEED_BASE + 6):
    """A synthetic mask for kernel analysis (profiles/: the floor / slope model of the tendency kernel): the aqua-planet
    fields at nx x ny x nz on a flat 6 km floor where only a w x h patch of every tile[0] x tile[1] block of columns is ocean
    (all nz levels wet there), the rest land - every tile-level of the tendency kernel then holds exactly w * h wet cells.
    Not a BASELINE.json config; inputs only."""
    wl = aquaplanet(nx=nx, ny=ny, nz=nz, steps=steps, precision=precision, seed=seed)
    jj, ii = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    ocean = (ii % tile[0] < w) & (jj % tile[1] < h)
    wl["depth"] = np.where(ocean, 6000.0, 0.0)
    wl["name"] = "patch_%dx%d_of_%dx%d" % (w, h, tile[0], tile[1])
    return wl


CONFIGS = {0: config0, 1: config1, 2: config2, 3: config3, 4: config4, 5: aquaplanet, 6: tile_patch_planet}


def make(config, **kw):
    return CONFIGS[int(config)](**kw)
