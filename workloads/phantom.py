"""Analytic thorax phantom (stands in for the NCAT phantom of PAPER.md:L115).

Structures are given in config-0 millimetres (BASELINE.json configs[0]); a
configuration with a different field of view multiplies every coordinate and
semi-axis, per axis, by ``cfg.scale``.  Later structures overwrite earlier:

  1. body ellipsoid, centre 0, semi-axes (60, 40, 60), mu = 0.02 /mm
  2. lungs, centres (+-28, 0, 0), semi-axes (20, 25, 45), mu = 0.004
  3. heart (C1-C4), centre (6, 8, -15), semi-axes (10, 12, 14), mu = 0.021
  4. rib shells (C1-C4), mu = 0.04: points whose in-plane body-ellipse radius
     relative to the body cross-section at that height,
     rho = sqrt((x/60)^2 + (y/40)^2) / sqrt(1 - (z/60)^2), lies in [0.86, 0.93],
     with |z| < 50 and (z mod 16) < 6
  5. tumour sphere r = 8, centre (-28, 0, 0) (right lung = -x), mu = 0.02

A voxel value is the mean of mu over a 4x4x4 sub-sample of the voxel (partial
volume; keeps the objective smooth).  Sub-sampling is applied to every voxel
whose 3x3x3 neighbourhood of centre samples is not uniform; the others take
their centre sample (identical result there, because the voxel is interior to
one structure up to features thinner than a voxel).
"""
from __future__ import annotations

import numpy as np
from scipy import ndimage

from .configs import Config

MU_BODY, MU_LUNG, MU_HEART, MU_RIB, MU_TUMOUR = 0.02, 0.004, 0.021, 0.04, 0.02
TUMOUR_CENTRE_C0 = (-28.0, 0.0, 0.0)
TUMOUR_RADIUS_C0 = 8.0


def mu_c0(x, y, z, heart_and_ribs: bool):
    """Attenuation at points given in config-0 millimetres (arrays broadcast)."""
    x = np.asarray(x, dtype=np.float64)
    y = np.asarray(y, dtype=np.float64)
    z = np.asarray(z, dtype=np.float64)
    mu = np.zeros(np.broadcast(x, y, z).shape, dtype=np.float64)
    body = (x / 60.0) ** 2 + (y / 40.0) ** 2 + (z / 60.0) ** 2 <= 1.0
    mu[body] = MU_BODY
    for cx in (28.0, -28.0):
        lung = ((x - cx) / 20.0) ** 2 + (y / 25.0) ** 2 + (z / 45.0) ** 2 <= 1.0
        mu[lung] = MU_LUNG
    if heart_and_ribs:
        heart = ((x - 6.0) / 10.0) ** 2 + ((y - 8.0) / 12.0) ** 2 + ((z + 15.0) / 14.0) ** 2 <= 1.0
        mu[heart] = MU_HEART
        zc = np.clip(1.0 - (z / 60.0) ** 2, 1e-12, None)
        rho = np.sqrt(((x / 60.0) ** 2 + (y / 40.0) ** 2) / zc)
        rib = (rho >= 0.86) & (rho <= 0.93) & (np.abs(z) < 50.0) & (np.mod(z, 16.0) < 6.0)
        mu[rib] = MU_RIB
    tx, ty, tz = TUMOUR_CENTRE_C0
    tumour = (x - tx) ** 2 + (y - ty) ** 2 + (z - tz) ** 2 <= TUMOUR_RADIUS_C0 ** 2
    mu[tumour] = MU_TUMOUR
    return mu


def grid_axes(cfg: Config):
    """World coordinates (mm) of voxel centres along x, y, z (isocentre = volume centre)."""
    xs = (np.arange(cfg.nx) - (cfg.nx - 1) / 2.0) * cfg.hx
    ys = (np.arange(cfg.ny) - (cfg.ny - 1) / 2.0) * cfg.hy
    zs = (np.arange(cfg.nz) - (cfg.nz - 1) / 2.0) * cfg.hz
    return xs, ys, zs


def tumour_centre_mm(cfg: Config) -> np.ndarray:
    return np.array(TUMOUR_CENTRE_C0) * np.array(cfg.scale)


def voxelise(cfg: Config, dvf_mm: np.ndarray | None = None, sub: int = 4) -> np.ndarray:
    """Phantom sampled on the grid, float64 [nz][ny][nx].

    With ``dvf_mm`` ([3][nz][ny][nx], pull-back, mm) the phantom is evaluated at
    r + x(r): the ground-truth deformed volume (not a trilinear warp of f0).
    The displacement of a voxel's centre is used for all its sub-samples.
    """
    xs, ys, zs = grid_axes(cfg)
    sx, sy, sz = cfg.scale
    Z, Y, X = np.meshgrid(zs, ys, xs, indexing="ij")
    if dvf_mm is not None:
        X = X + dvf_mm[0]
        Y = Y + dvf_mm[1]
        Z = Z + dvf_mm[2]
    centre = mu_c0(X / sx, Y / sy, Z / sz, cfg.heart_and_ribs)
    if sub <= 1:
        return centre
    hi = ndimage.maximum_filter(centre, size=3, mode="nearest")
    lo = ndimage.minimum_filter(centre, size=3, mode="nearest")
    bz, by, bx = np.nonzero(hi != lo)
    out = centre.copy()
    if bz.size == 0:
        return out
    offs = (np.arange(sub) + 0.5) / sub - 0.5
    chunk = 1 << 16
    for s in range(0, bz.size, chunk):
        iz, iy, ix = bz[s:s + chunk], by[s:s + chunk], bx[s:s + chunk]
        px, py, pz = X[iz, iy, ix], Y[iz, iy, ix], Z[iz, iy, ix]
        acc = np.zeros(px.shape, dtype=np.float64)
        for oz in offs:
            for oy in offs:
                qx = (px[:, None] + offs[None, :] * cfg.hx) / sx
                qy = ((py + oy * cfg.hy) / sy)[:, None]
                qz = ((pz + oz * cfg.hz) / sz)[:, None]
                acc += mu_c0(qx, qy, qz, cfg.heart_and_ribs).sum(axis=1)
        out[iz, iy, ix] = acc / float(sub ** 3)
    return out
