"""Pins for the oracle's ray-marching variant of P and its transpose (PAPER.md:L82
leaves the discretisation of P open; reading C1):

    p_i = d_i sum_m (T f)(E_i + (m + 1/2) d_i e_i),   M_i = ceil(L_i / step), d_i = L_i / M_i,

[E_i, E_i + L_i e_i] being the part of ray i inside the box spanned by the voxel centres and T f the
trilinear interpolant of the voxel-centre values.  The definition is pinned by what fixes it without
the oracle's code: closed forms (a constant and an affine volume: the midpoint rule is exact on both),
a dense matrix built here from the definition, the adjoint identity, the limit step -> 0 against a
fine quadrature, and finite differences of J for the gradient chain that uses P^T.
"""
import numpy as np
import pytest

import oracle
from tests.util import box_chord, f32r, geom, ray_endpoints, smooth_model


@pytest.fixture(autouse=True)
def _ray_marching():
    yield
    oracle.set_projector(oracle.SIDDON)


def centre_box(g):
    h = np.array([f32r(g.hx), f32r(g.hy), f32r(g.hz)])
    n = np.array([g.nx, g.ny, g.nz])
    c = np.array([f32r(g.cx), f32r(g.cy), f32r(g.cz)])
    return c - (n - 1) * h / 2.0, c + (n - 1) * h / 2.0, h


def chord_ends(S, D, lo, hi):
    """Entry and exit parameters of segment S -> D in the box [lo, hi] (None if it misses)."""
    d = D - S
    t0, t1 = 0.0, 1.0
    for c in range(3):
        if d[c] == 0.0:
            if S[c] < lo[c] or S[c] > hi[c]:
                return None
            continue
        a, b = (lo[c] - S[c]) / d[c], (hi[c] - S[c]) / d[c]
        t0, t1 = max(t0, min(a, b)), min(t1, max(a, b))
    return (t0, t1) if t0 < t1 else None


def dense_matrix(g, theta, step):
    """l_ij of reading C1 for every (pixel, voxel) pair, straight from the definition.  Tiny inputs only."""
    lo, hi, h = centre_box(g)
    n = np.array([g.nx, g.ny, g.nz])
    A = np.zeros((g.nu * g.nv, g.V))
    for iv in range(g.nv):
        for iu in range(g.nu):
            S, D = ray_endpoints(g, theta, iu, iv)
            ends = chord_ends(S, D, lo, hi)
            if ends is None:
                continue
            L = (ends[1] - ends[0]) * np.linalg.norm(D - S)
            M = int(np.ceil(L / step))
            for m in range(M):
                al = ends[0] + (m + 0.5) * (ends[1] - ends[0]) / M
                q = (S + al * (D - S) - lo) / h
                i0 = np.minimum(np.maximum(np.floor(q).astype(int), 0), n - 2)
                t = q - i0
                for a in range(2):
                    for b in range(2):
                        for c in range(2):
                            wgt = (t[0] if a else 1 - t[0]) * (t[1] if b else 1 - t[1]) * (t[2] if c else 1 - t[2])
                            A[iv * g.nu + iu, ((i0[2] + c) * g.ny + i0[1] + b) * g.nx + i0[0] + a] += wgt * L / M
    return A


@pytest.mark.parametrize("theta", [0.0, 0.37, np.pi / 2, 2.5, 4.4])
def test_matches_the_dense_matrix_of_the_definition(theta):
    g = geom(nx=5, ny=4, nz=3, h=(20.0, 25.0, 30.0), nu=9, nv=7, pitch=(14.0, 17.0), centre=(3.717, -1.129, 2.346))
    step = 7.3
    A = dense_matrix(g, theta, step)
    assert np.count_nonzero(A) > 200
    rng = np.random.default_rng(3)
    f = rng.standard_normal(g.vshape)
    r = rng.standard_normal(g.pshape)
    oracle.set_projector(oracle.RAY_MARCHING, step)
    np.testing.assert_allclose(oracle.project(g, f, theta).ravel(), A @ f.ravel(), rtol=0, atol=1e-10)
    np.testing.assert_allclose(oracle.backproject(g, r, theta).ravel(), A.T @ r.ravel(), rtol=0, atol=1e-10)


@pytest.mark.parametrize("theta", [0.0, 0.3, np.pi / 4, 2.1, 4.0, 5.5])
def test_uniform_volume_is_mu_times_the_chord_of_the_centre_box(theta):
    g = geom(nx=13, ny=11, nz=9, h=(3.0, 2.0, 2.5), nu=21, nv=15, pitch=(2.0, 2.0), centre=(1.1, 0.7, -0.4))
    mu = 0.0173
    oracle.set_projector(oracle.RAY_MARCHING, 0.9)
    p = oracle.project(g, np.full(g.vshape, mu), theta)
    lo, hi, _ = centre_box(g)
    hit = 0
    for iv in range(g.nv):
        for iu in range(g.nu):
            S, D = ray_endpoints(g, theta, iu, iv)
            chord = box_chord(S, D, lo, hi)
            assert abs(p[iv, iu] - mu * chord) < 1e-12 * 100
            hit += chord > 0
    assert hit > 100


@pytest.mark.parametrize("step", [0.4, 1.7, 50.0])
def test_affine_volume_is_integrated_exactly(step):
    """T reproduces an affine function and the midpoint rule integrates it exactly, whatever the step:
    p_i = L_i * (value at the chord's midpoint)."""
    g = geom(nx=12, ny=10, nz=8, h=(2.0, 2.5, 3.0), nu=15, nv=11, pitch=(2.2, 2.4), centre=(-0.6, 0.9, 0.3))
    lo, hi, h = centre_box(g)
    zz, yy, xx = np.meshgrid(np.arange(g.nz), np.arange(g.ny), np.arange(g.nx), indexing="ij")
    coef, c0 = np.array([0.011, -0.007, 0.004]), 0.3
    f = c0 + coef[0] * (lo[0] + xx * h[0]) + coef[1] * (lo[1] + yy * h[1]) + coef[2] * (lo[2] + zz * h[2])
    oracle.set_projector(oracle.RAY_MARCHING, step)
    for theta in (0.2, 1.9, 3.6):
        p = oracle.project(g, f, theta)
        for iv in range(g.nv):
            for iu in range(g.nu):
                S, D = ray_endpoints(g, theta, iu, iv)
                ends = chord_ends(S, D, lo, hi)
                want = 0.0
                if ends is not None:
                    mid = S + 0.5 * (ends[0] + ends[1]) * (D - S)
                    want = (ends[1] - ends[0]) * np.linalg.norm(D - S) * (c0 + coef @ mid)
                assert abs(p[iv, iu] - want) < 1e-10


def test_adjoint_identity_also_multithreaded():
    g = geom(nx=20, ny=17, nz=11, h=(2.0, 2.0, 3.0), nu=24, nv=18, pitch=(2.5, 2.5), centre=(0.4, -0.2, 0.1))
    rng = np.random.default_rng(11)
    f, r = rng.standard_normal(g.vshape), rng.standard_normal(g.pshape)
    oracle.set_projector(oracle.RAY_MARCHING, 1.1)
    for threads in (1, 3):
        oracle.set_threads(threads)
        lhs = np.vdot(oracle.project(g, f, 0.83), r)
        rhs = np.vdot(f, oracle.backproject(g, r, 0.83))
        assert abs(lhs - rhs) <= 1e-12 * abs(lhs)
    oracle.set_threads(oracle.max_threads())


def test_small_steps_converge_to_the_line_integral_of_the_interpolant():
    """step -> 0: the sum tends to the integral of T f along the chord (here by a 40 000-point quadrature
    written in numpy), with the midpoint rule's second order."""
    g = geom(nx=9, ny=8, nz=7, h=(4.0, 4.0, 4.0), nu=5, nv=5, pitch=(6.0, 6.0))
    rng = np.random.default_rng(5)
    f = rng.random(g.vshape)
    lo, hi, h = centre_box(g)
    n = np.array([g.nx, g.ny, g.nz])
    theta, iu, iv = 0.61, 2, 3
    S, D = ray_endpoints(g, theta, iu, iv)
    t0, t1 = chord_ends(S, D, lo, hi)
    al = t0 + (np.arange(40000) + 0.5) * (t1 - t0) / 40000
    q = (S[None, :] + al[:, None] * (D - S)[None, :] - lo) / h
    i0 = np.minimum(np.maximum(np.floor(q).astype(int), 0), n - 2)
    t = q - i0
    val = np.zeros(len(al))
    for a in range(2):
        for b in range(2):
            for c in range(2):
                wgt = (t[:, 0] if a else 1 - t[:, 0]) * (t[:, 1] if b else 1 - t[:, 1]) * (t[:, 2] if c else 1 - t[:, 2])
                val += wgt * f[i0[:, 2] + c, i0[:, 1] + b, i0[:, 0] + a]
    exact = val.mean() * (t1 - t0) * np.linalg.norm(D - S)
    errs = []
    for step in (2.0, 1.0, 0.5):
        oracle.set_projector(oracle.RAY_MARCHING, step)
        errs.append(abs(oracle.project(g, f, theta)[iv, iu] - exact))
    assert errs[2] < errs[0] and errs[2] < 2e-3 * exact


@pytest.mark.parametrize("seed", [1, 2])
def test_gradient_matches_finite_differences_of_J(seed):
    """The chain 2 U^T (df/dx) P^T r with the ray-marching P^T against central differences of J (the same
    pin as for Siddon)."""
    g = geom(nx=14, ny=12, nz=10, h=(3.0, 3.0, 3.5), K=3, nu=20, nv=16, pitch=(3.2, 3.2))
    f0, xbar, u, scale = smooth_model(g, seed=seed)
    rng = np.random.default_rng(seed)
    w = scale * 0.5 * rng.standard_normal(g.K)
    theta, a, b = 1.3, 0.9, 0.02
    oracle.set_projector(oracle.RAY_MARCHING, 1.3)
    _, p = oracle.evaluate(g, f0, xbar, u, w, theta)
    y = (p * (1 + 0.1 * rng.standard_normal(p.shape)) + 0.05).astype(np.float32)
    grad = oracle.gradient(g, f0, xbar, u, w, a, b, p, y, theta)

    def J(wv):
        _, pv = oracle.evaluate(g, f0, xbar, u, wv, theta)
        return oracle.cost(pv, y, a, b)

    eps = 1e-4 * scale
    for k in range(g.K):
        e = np.zeros(g.K)
        e[k] = eps
        fd = (J(w + e) - J(w - e)) / (2 * eps)
        assert abs(fd - grad[k]) <= 1e-5 * np.linalg.norm(grad), (k, fd, grad[k])


def test_solve_decreases_J_with_the_ray_marching_projector():
    g = geom(nx=16, ny=14, nz=12, h=(3.0, 3.0, 3.0), K=2, nu=24, nv=18, pitch=(3.0, 3.0))
    f0, xbar, u, scale = smooth_model(g, seed=4)
    w_true = scale * np.array([0.6, -0.4])
    oracle.set_projector(oracle.RAY_MARCHING, 1.5)
    _, y = oracle.evaluate(g, f0, xbar, u, w_true, 0.7)
    res = oracle.solve(g, f0, xbar, u, y.astype(np.float32), 0.7, np.zeros(g.K), oracle.Opts(max_iter=40))
    assert np.all(np.diff(res["J_trace"][:res["iters"] + 1]) <= 1e-12 * res["J0"])
    assert res["J"] < 1e-3 * res["J0"]
    assert np.linalg.norm(res["w"] - w_true) <= 2e-2 * np.linalg.norm(w_true)
