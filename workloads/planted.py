"""Purpose-built inputs for planted-coefficient and closed-form tests.

Smooth analytic vector fields (separable low-order cosines) QR-orthonormalised
into a known basis U*, and smooth test volumes that vanish at the border.  Used
where a test needs a known answer (planted w*, known PCA basis) rather than the
anatomy of the phantom.
"""
from __future__ import annotations

import numpy as np


def cosine_fields(shape_zyx, n: int, seed: int = 7) -> np.ndarray:
    """n smooth vector fields [n][3][nz][ny][nx], float64, linearly independent."""
    nz, ny, nx = shape_zyx
    z = (np.arange(nz) + 0.5) / nz
    y = (np.arange(ny) + 0.5) / ny
    x = (np.arange(nx) + 0.5) / nx
    rng = np.random.default_rng(seed)
    out = np.zeros((n, 3, nz, ny, nx))
    for k in range(n):
        for c in range(3):
            for _ in range(3):
                fz, fy, fx = rng.integers(0, 3, size=3)
                amp = rng.uniform(-1.0, 1.0)
                ph = rng.uniform(0, np.pi, size=3)
                out[k, c] += amp * (np.cos(np.pi * fz * z + ph[0])[:, None, None]
                                    * np.cos(np.pi * fy * y + ph[1])[None, :, None]
                                    * np.cos(np.pi * fx * x + ph[2])[None, None, :])
    return out


def orthonormal_basis(shape_zyx, K: int, seed: int = 7) -> np.ndarray:
    """K orthonormal smooth vector fields, float64 [K][3][nz][ny][nx]."""
    F = cosine_fields(shape_zyx, K, seed).reshape(K, -1)
    Q, R = np.linalg.qr(F.T)
    Q = Q * np.sign(np.diag(R))[None, :]
    return Q.T.reshape((K, 3) + tuple(shape_zyx))


def blob_volume(shape_zyx, n_blobs: int = 6, seed: int = 3) -> np.ndarray:
    """Smooth positive volume, float64, exactly zero on the outer two voxel layers."""
    nz, ny, nx = shape_zyx
    rng = np.random.default_rng(seed)
    z = np.arange(nz)[:, None, None] / (nz - 1.0)
    y = np.arange(ny)[None, :, None] / (ny - 1.0)
    x = np.arange(nx)[None, None, :] / (nx - 1.0)
    vol = np.zeros((nz, ny, nx))
    for _ in range(n_blobs):
        c = rng.uniform(0.3, 0.7, size=3)
        s = rng.uniform(0.08, 0.2, size=3)
        a = rng.uniform(0.005, 0.03)
        vol += a * np.exp(-0.5 * (((z - c[0]) / s[0]) ** 2 + ((y - c[1]) / s[1]) ** 2
                                  + ((x - c[2]) / s[2]) ** 2))
    win = np.ones((nz, ny, nx))
    for ax, n in enumerate((nz, ny, nx)):
        w = np.clip((np.minimum(np.arange(n), n - 1 - np.arange(n)) - 1.0) / 3.0, 0.0, 1.0)
        win *= w.reshape([-1 if i == ax else 1 for i in range(3)])
    return vol * win
