"""Pins for dJ/dw (readings A4-A6) and the intensity fit (Eq. 4, A8, A10)."""
import numpy as np
import pytest

import oracle
from tests.util import geom, smooth_model


def _setup(seed, K=3, noise=True):
    g = geom(nx=14, ny=12, nz=10, h=(3.0, 3.0, 3.5), K=K, nu=20, nv=16, pitch=(3.5, 3.5), centre=(0.37, 0.11, 0.23))
    f0, xbar, u, scale = smooth_model(g, seed=seed, disp_vox=1.3)
    rng = np.random.default_rng(seed)
    theta = float(rng.uniform(0, 2 * np.pi))
    w_true = rng.uniform(-1, 1, g.K) * scale
    _, p_true = oracle.evaluate(g, f0, xbar, u, w_true, theta)
    y = (1.3 * p_true + 0.05 + (0.002 * rng.standard_normal(p_true.shape) if noise else 0)).astype(np.float32)
    w = w_true + rng.uniform(-0.5, 0.5, g.K) * scale
    return g, f0, xbar, u, scale, theta, y, w


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_gradient_matches_central_finite_differences(seed):
    """north_star pin: dJ/dw_k vs central differences of J in float64, relative error <= 1e-5 per k.
    J is piecewise smooth in w (kinks where a sampling position crosses a lattice plane), so the test
    point is generic and the step small (1e-5 mm rms displacement)."""
    g, f0, xbar, u, scale, theta, y, w = _setup(seed)
    _, p = oracle.evaluate(g, f0, xbar, u, w, theta)
    rc, a, b = oracle.lsfit(p, y)
    assert rc == 0
    grad = oracle.gradient(g, f0, xbar, u, w, a, b, p, y, theta)
    step = 1e-5 * np.sqrt(g.V)
    gnorm = np.linalg.norm(grad)
    for k in range(g.K):
        e = np.zeros(g.K)
        e[k] = step
        Jp = oracle.cost(oracle.evaluate(g, f0, xbar, u, w + e, theta)[1], y, a, b)
        Jm = oracle.cost(oracle.evaluate(g, f0, xbar, u, w - e, theta)[1], y, a, b)
        fd = (Jp - Jm) / (2 * step)
        assert abs(fd - grad[k]) <= 1e-5 * max(abs(grad[k]), 1e-2 * gnorm), (k, fd, grad[k])


def test_gradient_is_zero_for_zero_residual():
    g, f0, xbar, u, scale, theta, y, w = _setup(5, noise=False)
    _, p = oracle.evaluate(g, f0, xbar, u, w, theta)
    grad = oracle.gradient(g, f0, xbar, u, w, 1.0, 0.0, p, p.astype(np.float32), theta)
    grad_ref = oracle.gradient(g, f0, xbar, u, w, 1.0, 0.5, p, p.astype(np.float32), theta)
    assert np.linalg.norm(grad) < 1e-6 * np.linalg.norm(grad_ref)


def test_gradient_from_explicit_chain():
    """g_k = 2 sum_j B_j (G_j . u_kj) assembled in numpy from the separately pinned pieces."""
    g, f0, xbar, u, scale, theta, y, w = _setup(7)
    _, p = oracle.evaluate(g, f0, xbar, u, w, theta)
    a, b = 1.1, -0.02
    r = p - a * y.astype(np.float64) - b
    B = oracle.backproject(g, r, theta)
    G = oracle.warp_grad(g, f0, xbar, u, w)
    want = np.array([2.0 * np.sum(B * np.sum(G * u[k].astype(np.float64), axis=0)) for k in range(g.K)])
    got = oracle.gradient(g, f0, xbar, u, w, a, b, p, y, theta)
    np.testing.assert_allclose(got, want, rtol=1e-12)


def test_lsfit_recovers_exact_linear_relation():
    rng = np.random.default_rng(0)
    p = rng.random(500) * 5
    c, d = 0.75, 0.125
    y = (c * p + d).astype(np.float32)
    p = (y.astype(np.float64) - d) / c   # make the relation exact for the float32 y
    rc, a, b = oracle.lsfit(p, y)
    assert rc == 0
    assert abs(a - 1 / c) < 1e-12 and abs(b + d / c) < 1e-12
    assert oracle.cost(p, y, a, b) < 1e-22


def test_lsfit_is_the_minimiser_and_cost_is_the_squared_norm():
    rng = np.random.default_rng(1)
    p = rng.random(300) * 4
    y = (0.8 * p + 0.1 + 0.05 * rng.standard_normal(300)).astype(np.float32)
    rc, a, b = oracle.lsfit(p, y)
    J = oracle.cost(p, y, a, b)
    assert abs(J - np.sum((p - a * y.astype(np.float64) - b) ** 2)) < 1e-12 * J
    for da, db in [(1e-3, 0), (-1e-3, 0), (0, 1e-3), (0, -1e-3), (1e-3, -1e-3)]:
        assert oracle.cost(p, y, a + da, b + db) > J
    # normal equations: the residual is orthogonal to y and to 1
    r = p - a * y.astype(np.float64) - b
    assert abs(r.sum()) < 1e-9 and abs((r * y).sum()) < 1e-9


def test_lsfit_constant_measurement_is_singular():
    rc, _, _ = oracle.lsfit(np.arange(10.0), np.full(10, 2.0, np.float32))
    assert rc == -5
