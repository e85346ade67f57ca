"""Pins for the oracle's DVF synthesis + trilinear warp and its derivative (Eq. 1, A1, A2, A6)."""
import numpy as np

import oracle
from tests.util import geom, smooth_model


def test_identity_dvf_reproduces_reference_exactly():
    """north_star pin: w = 0, xbar = 0 reproduces f0 bit for bit, and its projection is P f0 exactly."""
    g = geom(nx=11, ny=9, nz=7, K=3)
    rng = np.random.default_rng(0)
    f0 = rng.random(g.vshape).astype(np.float32)
    xbar = np.zeros((3,) + g.vshape, np.float32)
    u = rng.standard_normal((g.K, 3) + g.vshape).astype(np.float32)
    f = oracle.warp(g, f0, xbar, u, np.zeros(g.K))
    assert np.array_equal(f, f0.astype(np.float64))
    assert np.array_equal(oracle.project(g, f, 0.8), oracle.project(g, f0.astype(np.float64), 0.8))


def test_integer_shift_dvf_shifts_the_volume():
    g = geom(nx=12, ny=10, nz=8, h=(2.0, 2.5, 3.0), K=1)
    rng = np.random.default_rng(1)
    f0 = rng.random(g.vshape).astype(np.float32)
    # x = xbar + u w with w = 2: (+2, -1, +3) voxels, in mm
    xbar = np.zeros((3,) + g.vshape, np.float32)
    u = np.zeros((1, 3) + g.vshape, np.float32)
    u[0, 0], u[0, 1], u[0, 2] = 1.0 * g.hx, -0.5 * g.hy, 1.5 * g.hz
    f = oracle.warp(g, f0, xbar, u, np.array([2.0]))
    want = np.zeros(g.vshape)
    # f(i,j,k) = f0(i+2, j-1, k+3), zero outside (reading A2)
    want[:g.nz - 3, 1:, :g.nx - 2] = f0[3:, :g.ny - 1, 2:]
    assert np.array_equal(f, want)


def test_affine_ramp_is_reproduced_and_has_constant_gradient():
    """Trilinear interpolation reproduces affine functions, so f(r) = ramp(r + x(r)) exactly for any
    DVF (away from the zero border) and df/dx = slope / h."""
    g = geom(nx=14, ny=12, nz=10, h=(2.0, 2.5, 3.0), K=2)
    Zi, Yi, Xi = np.meshgrid(np.arange(g.nz), np.arange(g.ny), np.arange(g.nx), indexing="ij")
    a0, sl = 0.5, np.array([0.25, -0.125, 0.0625])  # exactly representable
    f0 = (a0 + sl[0] * Xi + sl[1] * Yi + sl[2] * Zi).astype(np.float32)
    _, xbar, u, scale = smooth_model(g, seed=5, disp_vox=0.8)
    w = np.array([0.7, -0.4]) * scale
    x = xbar.astype(np.float64) + np.tensordot(w, u.astype(np.float64), axes=(0, 0))
    q = np.stack([Xi + x[0] / g.hx, Yi + x[1] / g.hy, Zi + x[2] / g.hz])
    inner = ((q[0] >= 0) & (q[0] <= g.nx - 1) & (q[1] >= 0) & (q[1] <= g.ny - 1)
             & (q[2] >= 0) & (q[2] <= g.nz - 1))
    assert inner.sum() > 0.5 * g.V
    f = oracle.warp(g, f0, xbar, u, w)
    want = a0 + sl[0] * q[0] + sl[1] * q[1] + sl[2] * q[2]
    np.testing.assert_allclose(f[inner], want[inner], rtol=0, atol=1e-12)
    G = oracle.warp_grad(g, f0, xbar, u, w)
    strict = ((q[0] >= 0) & (q[0] < g.nx - 1) & (q[1] >= 0) & (q[1] < g.ny - 1)
              & (q[2] >= 0) & (q[2] < g.nz - 1))
    for c, hc in enumerate((g.hx, g.hy, g.hz)):
        np.testing.assert_allclose(G[c][strict], sl[c] / hc, rtol=0, atol=1e-12)


def test_warp_matches_direct_trilinear_formula_on_random_points():
    """Independent numpy evaluation of the SURVEY 8(a) trilinear formula on sampled voxels."""
    g = geom(nx=10, ny=9, nz=8, K=2)
    f0, xbar, u, scale = smooth_model(g, seed=2, disp_vox=2.0)
    f0 = (f0 + np.random.default_rng(3).random(g.vshape).astype(np.float32) * 0.01)
    w = np.array([0.9, -1.3]) * scale
    f = oracle.warp(g, f0, xbar, u, w)
    pad = np.zeros((g.nz + 8, g.ny + 8, g.nx + 8))
    pad[4:-4, 4:-4, 4:-4] = f0
    rng = np.random.default_rng(4)
    for _ in range(200):
        i, j, k = rng.integers(g.nx), rng.integers(g.ny), rng.integers(g.nz)
        x = [float(xbar[c, k, j, i]) + sum(float(u[m, c, k, j, i]) * w[m] for m in range(g.K)) for c in range(3)]
        q = np.array([i + x[0] / g.hx, j + x[1] / g.hy, k + x[2] / g.hz])
        q = np.clip(q, -3.5, np.array([g.nx, g.ny, g.nz]) + 2.5)
        i0 = np.floor(q).astype(int)
        t = q - i0
        v = 0.0
        for a in range(2):
            for b in range(2):
                for c in range(2):
                    v += (pad[i0[2] + c + 4, i0[1] + b + 4, i0[0] + a + 4]
                          * (t[0] if a else 1 - t[0]) * (t[1] if b else 1 - t[1]) * (t[2] if c else 1 - t[2]))
        assert abs(f[k, j, i] - v) < 1e-14


def test_warp_grad_matches_finite_differences_of_warp():
    g = geom(nx=9, ny=8, nz=7, K=2)
    f0, xbar, u, scale = smooth_model(g, seed=9, disp_vox=1.2)
    w = np.array([0.31, 0.77]) * scale
    G = oracle.warp_grad(g, f0, xbar, u, w)
    eps = 1e-6
    for c in range(3):
        xb = xbar.astype(np.float64)
        # shift the whole DVF by +-eps mm along axis c through a one-component eigenvector
        u2 = np.zeros((1, 3) + g.vshape, np.float32)
        u2[0, c] = 1.0
        x_cur = (xb + np.tensordot(w, u.astype(np.float64), axes=(0, 0))).astype(np.float32)
        g1 = oracle.Geometry(**{**g.__dict__, "K": 1})
        fp = oracle.warp(g1, f0, x_cur, u2, np.array([eps]))
        fm = oracle.warp(g1, f0, x_cur, u2, np.array([-eps]))
        G1 = oracle.warp_grad(g1, f0, x_cur, u2, np.array([0.0]))
        fd = (fp - fm) / (2 * eps)
        # away from lattice kinks the central difference equals the analytic derivative
        ok = np.abs(fd - G1[c]) < 1e-7
        assert ok.mean() > 0.999
        # and the float32-rounded DVF gives nearly the same derivative as the float64 one
        assert np.abs(G1[c] - G[c]).max() < 1e-4 * max(np.abs(G[c]).max(), 1e-12) + 1e-9
