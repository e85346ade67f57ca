"""Pins for the alternating algorithm (Eq. 3-4; readings A7-A9, A16) and the
tumour localisation (reading A13)."""
import numpy as np
import pytest

import oracle
from tests.util import geom, smooth_model


def _planted(K=3, seed=11, n=(16, 14, 12), det=(24, 18), noise=0.0, disp_vox=1.0):
    g = geom(nx=n[0], ny=n[1], nz=n[2], h=(3.0, 3.0, 3.0), K=K, nu=det[0], nv=det[1], pitch=(3.2, 3.2),
             centre=(0.37, 0.11, 0.23))
    f0, xbar, u, scale = smooth_model(g, seed=seed, disp_vox=disp_vox)
    rng = np.random.default_rng(seed)
    theta = 0.6
    w_star = rng.uniform(0.4, 1.0, K) * rng.choice([-1, 1], K) * scale
    _, p = oracle.evaluate(g, f0, xbar, u, w_star, theta)
    y = (p + noise * rng.standard_normal(p.shape)).astype(np.float32)
    return g, f0, xbar, u, scale, theta, y, w_star


def test_cost_never_increases_and_armijo_holds():
    """'the cost function always decreases at each step' and J >= 0."""
    g, f0, xbar, u, scale, theta, y, w_star = _planted(noise=0.003)
    opts = oracle.Opts(max_iter=12)
    res = oracle.solve(g, f0, xbar, u, y, theta, np.zeros(g.K), opts)
    J = res["J_trace"]
    assert res["status"] == 1 and res["iters"] == 12 and len(J) == 13
    assert np.all(J >= 0) and np.all(np.diff(J) <= 1e-12 * J[0])
    assert J[-1] < 0.2 * J[0]
    # replay the accepted steps with the pinned primitives: each satisfies Armijo's inequality (A7)
    w = np.zeros(g.K)
    _, p = oracle.evaluate(g, f0, xbar, u, w, theta)
    _, a, b = oracle.lsfit(p, y)
    mu_prev = None
    for n in range(res["iters"]):
        Jn = oracle.cost(p, y, a, b)
        assert abs(Jn - J[n]) <= 1e-12 * J[0]
        grad = oracle.gradient(g, f0, xbar, u, w, a, b, p, y, theta)
        g2 = float(grad @ grad)
        assert abs(np.sqrt(g2) - res["gnorm_trace"][n]) <= 1e-10 * np.sqrt(g2)
        mu0 = (1.0 * min(g.hx, g.hy, g.hz) * np.sqrt(g.V) / np.sqrt(g2)) if n == 0 else 2 * mu_prev
        mu, t = res["mu_trace"][n], res["backtracks"][n]
        assert abs(mu - mu0 * 0.5 ** t) <= 1e-12 * mu
        for tt in range(t + 1):   # every earlier candidate failed, the accepted one passes
            m = mu0 * 0.5 ** tt
            Jt = oracle.cost(oracle.evaluate(g, f0, xbar, u, w - m * grad, theta)[1], y, a, b)
            assert (Jt <= Jn - 1e-4 * m * g2) == (tt == t)
        w = w - mu * grad
        _, p = oracle.evaluate(g, f0, xbar, u, w, theta)
        _, a, b = oracle.lsfit(p, y)
        mu_prev = mu
    np.testing.assert_allclose(w, res["w"], rtol=1e-12)
    np.testing.assert_allclose(res["p"], p, rtol=0, atol=1e-12)
    np.testing.assert_allclose(res["f"], oracle.warp(g, f0, xbar, u, w), rtol=0, atol=1e-12)


def test_batched_linesearch_equals_sequential():
    g, f0, xbar, u, scale, theta, y, w_star = _planted(noise=0.003, seed=4)
    r1 = oracle.solve(g, f0, xbar, u, y, theta, np.zeros(g.K), oracle.Opts(max_iter=8))
    r2 = oracle.solve(g, f0, xbar, u, y, theta, np.zeros(g.K), oracle.Opts(max_iter=8, batched_linesearch=1))
    assert np.array_equal(r1["backtracks"], r2["backtracks"])
    np.testing.assert_allclose(r1["w"], r2["w"], rtol=1e-13)
    np.testing.assert_allclose(r1["J_trace"], r2["J_trace"], rtol=1e-13)


def test_forced_steps_replay_reproduces_the_run():
    g, f0, xbar, u, scale, theta, y, w_star = _planted(noise=0.003, seed=5)
    r1 = oracle.solve(g, f0, xbar, u, y, theta, np.zeros(g.K), oracle.Opts(max_iter=6))
    r2 = oracle.solve(g, f0, xbar, u, y, theta, np.zeros(g.K), oracle.Opts(max_iter=6), forced_mu=r1["mu_trace"])
    np.testing.assert_allclose(r1["w"], r2["w"], rtol=1e-14)


def test_gradient_tolerance_stops_the_loop():
    g, f0, xbar, u, scale, theta, y, w_star = _planted(noise=0.0, seed=6)
    res = oracle.solve(g, f0, xbar, u, y, theta, w_star, oracle.Opts(max_iter=5, grad_tol=1e9))
    assert res["status"] == 2 and res["iters"] == 0
    np.testing.assert_allclose(res["w"], w_star)


@pytest.mark.parametrize("K,seed", [(3, 11), (2, 12)])
def test_planted_coefficients_are_recovered(K, seed):
    """north_star pin: noise-free y = P warp(w*) => the converged solve returns w*, a = 1, b = 0."""
    g, f0, xbar, u, scale, theta, y, w_star = _planted(K=K, seed=seed)
    res = oracle.solve(g, f0, xbar, u, y, theta, np.zeros(K), oracle.Opts(max_iter=400, grad_tol=0.0))
    assert np.linalg.norm(res["w"] - w_star) <= 1e-3 * np.linalg.norm(w_star), (res["w"], w_star, res["J_trace"][-1])
    assert abs(res["a"] - 1) < 1e-4 and abs(res["b"]) < 1e-4
    assert res["J"] < 1e-6 * res["J0"]


def test_brute_force_grid_confirms_the_minimiser():
    """K = 2: a dense grid over w around w* (min over a, b at each point) has its arg-min at the grid
    point nearest the solver's answer."""
    g, f0, xbar, u, scale, theta, y, w_star = _planted(K=2, seed=12, n=(10, 9, 8), det=(14, 10), noise=0.0005)
    res = oracle.solve(g, f0, xbar, u, y, theta, np.zeros(2), oracle.Opts(max_iter=300))
    assert res["status"] == 3  # no further decrease possible: converged
    # (with much larger noise the a*y form of Eq. 2 rewards shrinking p towards 0 -- see DESIGN.md)
    half, m = 0.02 * scale, 41
    ax0 = res["w"][0] + np.linspace(-half, half, m)
    ax1 = res["w"][1] + np.linspace(-half, half, m)
    best, arg = np.inf, None
    for i0, w0 in enumerate(ax0):
        for i1, w1 in enumerate(ax1):
            _, p = oracle.evaluate(g, f0, xbar, u, np.array([w0, w1]), theta)
            _, a, b = oracle.lsfit(p, y)
            J = oracle.cost(p, y, a, b)
            if J < best:
                best, arg = J, (i0, i1)
    assert arg == (m // 2, m // 2), (arg, best, res["J"])
    assert res["J"] <= best * (1 + 1e-9)


# ---------------------------------------------------------------- tumour localisation

def _const_model(g, c_mm):
    xbar = np.zeros((3,) + g.vshape, np.float32)
    u = np.zeros((1, 3) + g.vshape, np.float32)
    for c in range(3):
        u[0, c] = c_mm[c]
    return xbar, u


def test_inversion_of_zero_and_constant_dvf():
    g = geom(nx=10, ny=9, nz=8, h=(2.0, 2.0, 2.0), K=1)
    r0 = np.array([[1.0, -2.0, 0.5], [3.0, 3.0, -3.0]], np.float32)
    xbar, u = _const_model(g, (0.5, -1.25, 2.0))
    out, its = oracle.invert(g, xbar, u, np.array([0.0]), r0)
    assert np.array_equal(out, r0.astype(np.float64)) and np.all(its == 1)
    out, its = oracle.invert(g, xbar, u, np.array([2.0]), r0)
    np.testing.assert_allclose(out, r0 - 2.0 * np.array([0.5, -1.25, 2.0]), atol=1e-14)
    assert np.all(its == 2)  # exact after one iteration, the second confirms |dr| < tol


def test_inversion_of_affine_dvf_closed_form():
    """x(r) = A r + c with ||A|| < 1: r = (I + A)^-1 (r0 - c); trilinear interpolation of an affine
    field is exact, so the fixed point is reached to 1e-10."""
    g = geom(nx=12, ny=11, nz=10, h=(2.0, 2.5, 3.0), K=1, centre=(0.3, -0.2, 0.1))
    A = np.array([[0.10, -0.05, 0.02], [0.03, 0.08, -0.04], [-0.02, 0.06, 0.12]])
    c = np.array([0.7, -0.4, 1.1])
    xs = (np.arange(g.nx) - (g.nx - 1) / 2) * g.hx + np.float32(g.cx)
    ys = (np.arange(g.ny) - (g.ny - 1) / 2) * g.hy + np.float32(g.cy)
    zs = (np.arange(g.nz) - (g.nz - 1) / 2) * g.hz + np.float32(g.cz)
    Z, Y, X = np.meshgrid(zs, ys, xs, indexing="ij")
    R = np.stack([X, Y, Z])
    field = np.tensordot(A, R, axes=(1, 0)) + c[:, None, None, None]
    xbar = np.zeros((3,) + g.vshape, np.float32)
    u = field[None].astype(np.float32)
    r0 = np.array([[2.0, -3.0, 1.5], [-4.0, 2.0, -2.5]], np.float32)
    out, its = oracle.invert(g, xbar, u, np.array([1.0]), r0, max_iter=200, tol_mm=1e-13)
    want = np.linalg.solve(np.eye(3) + A, (r0.astype(np.float64) - c).T).T
    # the float32 storage of the field limits the agreement to ~1e-6 mm; the fixed point itself is tight
    np.testing.assert_allclose(out, want, atol=5e-6)
    x_at = oracle.dvf_at_points(g, xbar, u, np.array([1.0]), out)
    np.testing.assert_allclose(out + x_at, r0, atol=1e-10)


def test_dvf_interpolation_clamps_at_the_grid_edge():
    g = geom(nx=6, ny=5, nz=4, h=(2.0, 2.0, 2.0), K=1)
    rng = np.random.default_rng(0)
    xbar = rng.standard_normal((3,) + g.vshape).astype(np.float32)
    u = np.zeros((1, 3) + g.vshape, np.float32)
    far = np.array([[100.0, 100.0, 100.0], [-100.0, -100.0, -100.0]])
    x = oracle.dvf_at_points(g, xbar, u, np.array([0.0]), far)
    np.testing.assert_array_equal(x[0], xbar[:, -1, -1, -1].astype(np.float64))
    np.testing.assert_array_equal(x[1], xbar[:, 0, 0, 0].astype(np.float64))
    # on a voxel centre the interpolant returns the stored value
    ctr = np.array([[(2 - 2.5) * 2.0, (1 - 2.0) * 2.0, (3 - 1.5) * 2.0]])
    np.testing.assert_allclose(oracle.dvf_at_points(g, xbar, u, np.array([0.0]), ctr)[0],
                               xbar[:, 3, 1, 2].astype(np.float64), atol=1e-15)
