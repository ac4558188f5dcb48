"""Seeded synthetic CT / CBCT phantoms and displacement fields (inputs only).

This module serves BOTH the CPU oracle (`oracle/`) and the CUDA path
(`paper_1204_6295_b200/`) and therefore holds none of the method's arithmetic:
no patch moments, no demons force, no regularisation, no pyramid.  It only
draws volumes.  The recipe is DESIGN.md "Input recipe" (taken from
BASELINE.json `configs` and SURVEY.md section 8(d)).

The paper measures on one Monte-Carlo simulated and six clinical head-and-neck
CT/CBCT pairs (sections 2.4.1-2.4.2).  None of that data is
public; these phantoms stand in for it.  They take their shapes (H&N volumes of
256x256x~68-128 voxels in HU), their artefact kinds (scatter cupping, streaks,
bow-tie crescent, noise: PAPER.md:41) and the deformation magnitudes from the
paper and BASELINE.json.

Array layout everywhere: C-order ``[nz, ny, nx]`` float32, x fastest, i.e.
``idx = (z*ny + y)*nx + x``.  Displacement fields are planar ``[3, nz, ny, nx]``
with component 0,1,2 = x,y,z in voxel units.  The CBCT is generated as
``cbct(x) = gain * ct(x + u(x)) + artefacts + noise`` so that the pull-back
field recovered by the registration is ``r ~ u``.
"""
from __future__ import annotations

import numpy as np
from scipy import ndimage

BASE_SEED = 12046295  # + config index

# BASELINE.json `configs` 1..4: schedule and phantom parameters.
CONFIGS = {
    1: dict(dims=(64, 64, 32), patch_radius=3, sigma=1.5, levels=1, iters=50,
            kind="ellipsoid", max_disp=3.0, gain=0.9, cupping=150.0, noise=20.0),
    2: dict(dims=(128, 128, 64), patch_radius=4, sigma=1.5, levels=2, iters=100,
            kind="hn", max_disp=5.0, gain=0.9, cupping=200.0, noise=30.0,
            streaks=True, crescent=False),
    3: dict(dims=(256, 256, 128), patch_radius=5, sigma=2.0, levels=3, iters=100,
            kind="hn", max_disp=8.0, gain=0.9, cupping=200.0, noise=40.0,
            streaks=True, crescent=True),
    4: dict(dims=(512, 512, 128), patch_radius=7, sigma=2.0, levels=4, iters=100,
            kind="hn", max_disp=12.0, gain=0.9, cupping=250.0, noise=50.0,
            streaks=True, crescent=True),
}


def _grid(dims, dtype=np.float32):
    nx, ny, nz = dims
    z = np.arange(nz, dtype=dtype)[:, None, None]
    y = np.arange(ny, dtype=dtype)[None, :, None]
    x = np.arange(nx, dtype=dtype)[None, None, :]
    return x, y, z


def _blur(vol, sigma):
    return ndimage.gaussian_filter(vol, sigma=sigma, mode="nearest").astype(np.float32)


# --------------------------------------------------------------------------
# CT phantoms
# --------------------------------------------------------------------------
def ct_ellipsoid(dims, rng):
    """Config 1 CT: ellipsoid body (40 HU) in air (-1000 HU) with 3 spheres."""
    nx, ny, nz = dims
    x, y, z = _grid(dims)
    cx, cy, cz = (nx - 1) / 2.0, (ny - 1) / 2.0, (nz - 1) / 2.0
    ax, ay, az = 0.42 * nx, 0.36 * ny, 0.45 * nz
    vol = np.full((nz, ny, nx), -1000.0, dtype=np.float32)
    body = ((x - cx) / ax) ** 2 + ((y - cy) / ay) ** 2 + ((z - cz) / az) ** 2 <= 1.0
    vol[body] = 40.0
    for hu in (700.0, -100.0, -800.0):
        rad = float(rng.uniform(4.0, 8.0))
        # centre drawn inside the body, shrunk so the sphere stays inside
        while True:
            c = np.array([rng.uniform(-1, 1), rng.uniform(-1, 1), rng.uniform(-1, 1)])
            if np.sum(c ** 2) <= 1.0:
                break
        sx = cx + c[0] * max(ax - rad - 1, 1.0)
        sy = cy + c[1] * max(ay - rad - 1, 1.0)
        sz = cz + c[2] * max(az - rad - 1, 1.0)
        sph = (x - sx) ** 2 + (y - sy) ** 2 + (z - sz) ** 2 <= rad * rad
        vol[sph] = hu
    return _blur(vol, 1.0)


def ct_head_neck(dims, rng):
    """Configs 2-4 CT: elliptic-cylinder neck with spine, mandible arc, airway."""
    nx, ny, nz = dims
    x, y, z = _grid(dims)
    vol = np.full((nz, ny, nx), -1000.0, dtype=np.float32)
    # soft tissue 40 + 40*T, T = smoothed white noise scaled to [-1, 1]
    tex = ndimage.gaussian_filter(rng.standard_normal((nz, ny, nx)).astype(np.float32),
                                  sigma=nx / 32.0, mode="nearest")
    tex /= max(float(np.abs(tex).max()), 1e-12)
    cx, cy = 0.5 * nx, 0.5 * ny
    body = ((x - cx) / (0.40 * nx)) ** 2 + ((y - cy) / (0.33 * ny)) ** 2 <= 1.0
    body = np.broadcast_to(body, vol.shape)
    vol[body] = (40.0 + 40.0 * tex)[body]
    # spine: annulus centred (0.5nx, 0.68ny), outer radius 0.06nx, 800-1200 HU radial ramp
    sx, sy, ro = 0.5 * nx, 0.68 * ny, 0.06 * nx
    rs = np.sqrt((x - sx) ** 2 + (y - sy) ** 2)
    ri = 0.5 * ro
    spine = np.broadcast_to((rs <= ro) & (rs >= ri), vol.shape)
    ramp = np.broadcast_to(800.0 + 400.0 * (rs - ri) / (ro - ri), vol.shape)
    vol[spine] = ramp[spine].astype(np.float32)
    # mandible: 200-degree arc, centre (0.5nx, 0.45ny), radius 0.22nx, thickness 0.035nx, lower half of slices
    mx, my, rm, th = 0.5 * nx, 0.45 * ny, 0.22 * nx, 0.035 * nx
    rr = np.sqrt((x - mx) ** 2 + (y - my) ** 2)
    ang = np.degrees(np.arctan2(-(y - my), x - mx))  # arc opens toward the spine (+y)
    arc = (np.abs(rr - rm) <= th / 2) & (np.abs(ang - 90.0) <= 100.0)
    arc3 = np.broadcast_to(arc, vol.shape) & np.broadcast_to(z < nz / 2.0, vol.shape)
    mramp = np.broadcast_to(800.0 + 400.0 * np.clip((rr - (rm - th / 2)) / th, 0, 1), vol.shape)
    vol[arc3] = mramp[arc3].astype(np.float32)
    # airway tube radius 0.035nx at (0.5nx, 0.52ny)
    air = (x - 0.5 * nx) ** 2 + (y - 0.52 * ny) ** 2 <= (0.035 * nx) ** 2
    vol[np.broadcast_to(air, vol.shape)] = -900.0
    return _blur(vol, 1.0)


# --------------------------------------------------------------------------
# displacement fields
# --------------------------------------------------------------------------
def disp_sinusoid(dims, amplitude=3.0, period=32.0):
    """u_c = amplitude * sin(2*pi*x_c/period): each component varies along its own axis."""
    nx, ny, nz = dims
    x, y, z = _grid(dims, np.float64)
    u = np.empty((3, nz, ny, nx), dtype=np.float32)
    u[0] = np.broadcast_to(amplitude * np.sin(2 * np.pi * x / period), (nz, ny, nx))
    u[1] = np.broadcast_to(amplitude * np.sin(2 * np.pi * y / period), (nz, ny, nx))
    u[2] = np.broadcast_to(amplitude * np.sin(2 * np.pi * z / period), (nz, ny, nx))
    return u


def _bspline_basis(n, spacing):
    """Dense [n, ncoef] matrix of uniform cubic B-spline weights."""
    ncoef = int(np.ceil((n - 1) / spacing)) + 3
    t = np.arange(n, dtype=np.float64) / spacing
    i0 = np.floor(t).astype(int)
    f = t - i0
    w = np.stack([(1 - f) ** 3 / 6.0,
                  (3 * f ** 3 - 6 * f ** 2 + 4) / 6.0,
                  (-3 * f ** 3 + 3 * f ** 2 + 3 * f + 1) / 6.0,
                  f ** 3 / 6.0], axis=1)
    B = np.zeros((n, ncoef), dtype=np.float64)
    for k in range(4):
        B[np.arange(n), i0 + k] += w[:, k]
    return B


def disp_bspline(dims, rng, max_disp, spacing=None):
    """Random smooth field: cubic B-spline, control spacing nx/8, coefficients U(-1,1), max|u_c| = max_disp."""
    nx, ny, nz = dims
    spacing = spacing or nx / 8.0
    Bx, By, Bz = _bspline_basis(nx, spacing), _bspline_basis(ny, spacing), _bspline_basis(nz, spacing)
    u = np.empty((3, nz, ny, nx), dtype=np.float32)
    for c in range(3):
        coef = rng.uniform(-1.0, 1.0, size=(Bz.shape[1], By.shape[1], Bx.shape[1]))
        f = np.tensordot(Bz, coef, axes=(1, 0))            # [nz, cy, cx]
        f = np.tensordot(f, By, axes=(1, 1))               # [nz, cx, ny]
        f = np.tensordot(f, Bx, axes=(1, 1))               # [nz, ny, nx]
        f *= max_disp / max(float(np.abs(f).max()), 1e-12)
        u[c] = f.astype(np.float32)
    return u


def disp_smooth_random(dims, rng, max_disp=5.0, smooth=4.0):
    """Config 5 field: U(-1,1) noise smoothed with sigma 4, scaled to max|u_c| = max_disp."""
    nx, ny, nz = dims
    u = np.empty((3, nz, ny, nx), dtype=np.float32)
    for c in range(3):
        f = ndimage.gaussian_filter(rng.uniform(-1, 1, size=(nz, ny, nx)).astype(np.float32),
                                    sigma=smooth, mode="nearest")
        f *= max_disp / max(float(np.abs(f).max()), 1e-12)
        u[c] = f
    return u


def volume_smooth_random(dims, rng, smooth=2.0):
    """Config 5 volume: U(-1000,1500) HU white noise smoothed with a Gaussian of sigma 2."""
    nx, ny, nz = dims
    v = rng.uniform(-1000.0, 1500.0, size=(nz, ny, nx)).astype(np.float32)
    return ndimage.gaussian_filter(v, sigma=smooth, mode="nearest").astype(np.float32)


# --------------------------------------------------------------------------
# CBCT synthesis
# --------------------------------------------------------------------------
def pullback(vol, u):
    """vol(x + u(x)), trilinear, coordinates clamped (input synthesis only)."""
    nz, ny, nx = vol.shape
    zz, yy, xx = np.meshgrid(np.arange(nz, dtype=np.float32), np.arange(ny, dtype=np.float32),
                             np.arange(nx, dtype=np.float32), indexing="ij")
    coords = np.stack([np.clip(zz + u[2], 0, nz - 1), np.clip(yy + u[1], 0, ny - 1),
                       np.clip(xx + u[0], 0, nx - 1)])
    return ndimage.map_coordinates(vol, coords, order=1, mode="nearest").astype(np.float32)


def make_cbct(ct, u, rng, gain=0.9, cupping=150.0, noise=20.0, streaks=False, crescent=False):
    nz, ny, nx = ct.shape
    x, y, z = _grid((nx, ny, nz))
    cbct = gain * pullback(ct, u)
    cx, cy = (nx - 1) / 2.0, (ny - 1) / 2.0
    rho2 = ((x - cx) ** 2 + (y - cy) ** 2) / (nx / 2.0) ** 2
    cbct = cbct - cupping * np.maximum(0.0, 1.0 - rho2)          # radial cupping, deepest at centre
    if streaks:
        sx, sy = 0.5 * nx, 0.68 * ny                               # through the spine centre
        for amp in (100.0, -100.0, 100.0, -100.0):
            ang = rng.uniform(0.0, np.pi)
            d = (x - sx) * np.sin(ang) - (y - sy) * np.cos(ang)    # distance to the line
            cbct = cbct + amp * np.exp(-0.5 * (d / 1.5) ** 2)
    if crescent:
        rc = np.sqrt((x - (cx + 30.0)) ** 2 + (y - cy) ** 2)
        fov = np.sqrt((x - cx) ** 2 + (y - cy) ** 2) <= 0.48 * nx
        band = (np.abs(rc - 0.42 * nx) <= 3.0) & fov
        cbct = cbct + 150.0 * band
    cbct = cbct + rng.normal(0.0, noise, size=(nz, ny, nx))
    return np.ascontiguousarray(cbct, dtype=np.float32)


def make_pair(config, dims=None):
    """Return (ct, cbct, u_true, params) for BASELINE.json config 1..4 (optionally at other dims)."""
    p = dict(CONFIGS[config])
    if dims is not None:
        p["dims"] = tuple(dims)
    rng = np.random.default_rng(BASE_SEED + config)
    d = p["dims"]
    if p["kind"] == "ellipsoid":
        ct = ct_ellipsoid(d, rng)
        u = disp_sinusoid(d, amplitude=p["max_disp"], period=32.0)
    else:
        ct = ct_head_neck(d, rng)
        u = disp_bspline(d, rng, p["max_disp"])
    cbct = make_cbct(ct, u, rng, gain=p["gain"], cupping=p["cupping"], noise=p["noise"],
                     streaks=p.get("streaks", False), crescent=p.get("crescent", False))
    return np.ascontiguousarray(ct), cbct, u, p


def make_sweep_inputs(dims, seed_offset=5):
    """Config 5: (volume, second volume, displacement field) for the per-kernel sweep."""
    rng = np.random.default_rng(BASE_SEED + seed_offset)
    a = volume_smooth_random(dims, rng)
    b = volume_smooth_random(dims, rng)
    u = disp_smooth_random(dims, rng, max_disp=5.0)
    return a, b, u
