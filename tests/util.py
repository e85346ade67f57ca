"""Test helpers: small geometries, independent brute-force ray/box intersection, smooth inputs.

Nothing here is imported by the product.  The brute-force routines are written
separately from oracle.cpp (numpy, slab method on one box at a time) so that
they pin it rather than repeat it.
"""
from __future__ import annotations

import numpy as np

import oracle
from workloads import planted


def geom(nx=8, ny=7, nz=6, h=(2.0, 2.5, 3.0), K=2, nu=12, nv=9, pitch=(1.5, 2.0), sad=1000.0, sdd=1500.0,
         centre=(0.0, 0.0, 0.0), off=(0.0, 0.0)) -> oracle.Geometry:
    return oracle.Geometry(nx, ny, nz, h[0], h[1], h[2], K, nu, nv, pitch[0], pitch[1], sad, sdd,
                           off[0], off[1], centre[0], centre[1], centre[2])


def geom_from_config(cfg, centre=(0.0, 0.0, 0.0)) -> oracle.Geometry:
    return oracle.Geometry(cfg.nx, cfg.ny, cfg.nz, cfg.hx, cfg.hy, cfg.hz, cfg.K, cfg.nu, cfg.nv, cfg.pu, cfg.pv,
                           cfg.sad, cfg.sdd, 0.0, 0.0, centre[0], centre[1], centre[2])


def f32r(v):
    """Round through float32 the way the C-ABI does."""
    return float(np.float32(v))


def ray_endpoints(g: oracle.Geometry, theta, iu, iv):
    """Source and pixel centre in world mm (SURVEY 8(a) geometry), float64."""
    th = f32r(theta)
    c, s = np.cos(th), np.sin(th)
    sad, sdd = f32r(g.sad), f32r(g.sdd)
    S = np.array([sad * c, sad * s, 0.0])
    Cc = -(sdd - sad) * np.array([c, s, 0.0])
    uu = (iu - (g.nu - 1) / 2.0 + f32r(g.off_u)) * f32r(g.pu)
    vv = (iv - (g.nv - 1) / 2.0 + f32r(g.off_v)) * f32r(g.pv)
    D = Cc + uu * np.array([-s, c, 0.0]) + vv * np.array([0.0, 0.0, 1.0])
    return S, D


def box_chord(S, D, lo, hi):
    """Length of the part of segment S->D inside the axis-aligned box [lo, hi] (slab method)."""
    d = D - S
    t0, t1 = 0.0, 1.0
    for c in range(3):
        if d[c] == 0.0:
            if S[c] < lo[c] or S[c] >= hi[c]:
                return 0.0
            continue
        a, b = (lo[c] - S[c]) / d[c], (hi[c] - S[c]) / d[c]
        t0, t1 = max(t0, min(a, b)), min(t1, max(a, b))
    return max(0.0, t1 - t0) * float(np.linalg.norm(d))


def volume_box(g: oracle.Geometry):
    h = np.array([f32r(g.hx), f32r(g.hy), f32r(g.hz)])
    n = np.array([g.nx, g.ny, g.nz])
    c = np.array([f32r(g.cx), f32r(g.cy), f32r(g.cz)])
    return c - n * h / 2.0, c + n * h / 2.0, h


def dense_system_matrix(g: oracle.Geometry, theta):
    """Brute force l_ij for every (pixel, voxel) pair: [nv*nu][nz*ny*nx].  Tiny inputs only."""
    lo, _, h = volume_box(g)
    A = np.zeros((g.nu * g.nv, g.V))
    for iv in range(g.nv):
        for iu in range(g.nu):
            S, D = ray_endpoints(g, theta, iu, iv)
            for k in range(g.nz):
                for j in range(g.ny):
                    for i in range(g.nx):
                        blo = lo + np.array([i, j, k]) * h
                        A[iv * g.nu + iu, (k * g.ny + j) * g.nx + i] = box_chord(S, D, blo, blo + h)
    return A


def smooth_model(g: oracle.Geometry, seed=7, disp_vox=1.5, with_mean=True):
    """Smooth f0 (zero border) plus an orthonormal smooth basis: float32 arrays for a planted test.

    Returns f0, xbar, u (unit-norm) and a coefficient scale such that |w| ~ scale moves voxels by
    about `disp_vox` voxels rms.
    """
    shape = g.vshape
    f0 = planted.blob_volume(shape, seed=seed).astype(np.float32)
    U = planted.orthonormal_basis(shape, g.K + 1, seed=seed)
    hmin = min(g.hx, g.hy, g.hz)
    scale = disp_vox * hmin * np.sqrt(g.V)
    xbar = (0.3 * scale * U[g.K]).astype(np.float32) if with_mean else np.zeros((3,) + shape, np.float32)
    u = U[:g.K].astype(np.float32)
    return f0, xbar, u, scale
