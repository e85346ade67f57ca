"""Parity of the ray-marching variant of P (pcamm_geometry.projector = 1, DESIGN.md
reading C1) against the oracle's (oracle.set_projector(RAY_MARCHING)), through the C ABI: projection,
matched transpose, adjoint identity, cost / gradient / fit, finite differences of the GPU cost, whole
solves (single, two candidates per pass, several in flight) with the tumour position.

Bars as for Siddon (north_star / DESIGN.md section 3): projections rel-L2 <= 1e-4, J rel <= 1e-4, gradient
rel-L2 <= 1e-3, w within 1e-3 ||w||, tumour <= 0.05 mm.  The transpose is scattered with float atomic
adds, so its results are reproducible to rounding, not bitwise.
"""
import numpy as np
import pytest

import oracle
from tests.gpu_util import make_model, oracle_opts, rel_l2, to_dev, to_host
from tests.util import geom, smooth_model

pytestmark = pytest.mark.gpu

STEP_VOX = 0.5
ANGLES = [0.0, 0.3, np.pi / 4, 0.9, np.pi / 2, 2.1, 3 * np.pi / 4, np.pi, 4.0, 5.5]


@pytest.fixture(autouse=True)
def _ray_marching_oracle():
    yield
    oracle.set_projector(oracle.SIDDON)


def _use_rm(g, step_vox=STEP_VOX):
    oracle.set_projector(oracle.RAY_MARCHING, step_vox * min(g.hx, g.hy, g.hz))


def _geom(K=3, n=(45, 38, 21), det=(70, 27), centre=(1.1151, 0.3387, 0.7038), h=(3.0, 3.0, 3.0), pitch=(3.2, 3.4)):
    return geom(nx=n[0], ny=n[1], nz=n[2], h=h, K=K, nu=det[0], nv=det[1], pitch=pitch, centre=centre)


@pytest.mark.parametrize("h,pitch,step", [((3.0, 3.0, 3.0), (3.2, 3.4), 0.5), ((2.0, 3.0, 4.0), (2.5, 4.1), 0.8),
                                          ((3.0, 3.0, 3.0), (3.2, 3.4), 1.7)])
def test_projection_and_transpose_match_the_oracle(h, pitch, step):
    g = _geom(h=h, pitch=pitch)
    _use_rm(g, step)
    f0, xbar, u, scale = smooth_model(g, seed=3)
    m = make_model(g, f0, xbar, u, projector=1, ray_step_vox=step)
    rng = np.random.default_rng(0)
    f = rng.random(g.vshape).astype(np.float32)
    r = rng.standard_normal(g.pshape).astype(np.float32)
    for theta in ANGLES:
        p_ref = oracle.project(g, f, theta)
        p_gpu = to_host(m.project(to_dev(f), theta))
        assert rel_l2(p_gpu, p_ref) <= 1e-5, theta
        assert np.count_nonzero(p_ref) > 0.3 * p_ref.size
        B_ref = oracle.backproject(g, r, theta)
        B_gpu = to_host(m.backproject(to_dev(r), theta))
        assert rel_l2(B_gpu, B_ref) <= 1e-5, theta
        # <P f, r> = <f, P^T r> on the GPU itself
        lhs, rhs = float(np.vdot(p_gpu.astype(np.float64), r)), float(np.vdot(f.astype(np.float64), B_gpu))
        assert abs(lhs - rhs) <= 1e-5 * abs(lhs)


def test_uniform_volume_is_mu_times_the_chord():
    """The closed form that pins the oracle, on the GPU as well."""
    from tests.util import box_chord, f32r, ray_endpoints
    g = _geom()
    f0, xbar, u, _ = smooth_model(g, seed=3)
    m = make_model(g, f0, xbar, u, projector=1, ray_step_vox=0.7)
    mu = 0.0173
    p = to_host(m.project(to_dev(np.full(g.vshape, mu, np.float32)), 0.77))
    h = np.array([f32r(g.hx), f32r(g.hy), f32r(g.hz)])
    n = np.array([g.nx, g.ny, g.nz])
    c = np.array([f32r(g.cx), f32r(g.cy), f32r(g.cz)])
    lo, hi = c - (n - 1) * h / 2, c + (n - 1) * h / 2
    for iv in range(0, g.nv, 3):
        for iu in range(0, g.nu, 5):
            S, D = ray_endpoints(g, 0.77, iu, iv)
            want = np.float32(mu) * box_chord(S, D, lo, hi)
            assert abs(p[iv, iu] - want) <= 2e-6 * max(want, 1.0)


@pytest.mark.parametrize("K,seed", [(3, 5), (5, 6), (2, 7)])
def test_cost_gradient_fit_match_the_oracle(K, seed):
    g = _geom(K=K)
    _use_rm(g)
    f0, xbar, u, scale = smooth_model(g, seed=seed)
    m = make_model(g, f0, xbar, u, projector=1, ray_step_vox=STEP_VOX)
    rng = np.random.default_rng(seed)
    theta = 1.1
    for _ in range(2):
        w = (rng.uniform(-0.7, 0.7, K) * scale).astype(np.float32)
        a, b = 0.9, 0.03
        _, p_ref = oracle.evaluate(g, f0, xbar, u, w, theta)
        y = (p_ref * (1 + 0.05 * rng.standard_normal(p_ref.shape)) + 0.02).astype(np.float32)
        J_ref = oracle.cost(p_ref, y, a, b)
        g_ref = oracle.gradient(g, f0, xbar, u, w, a, b, p_ref, y, theta)
        _, a_ref, b_ref = oracle.lsfit(p_ref, y)
        J, grad, (af, bf), p = m.eval(to_dev(y), theta, w, a, b)
        assert rel_l2(to_host(p), p_ref) <= 1e-5
        assert abs(J - J_ref) <= 1e-4 * J_ref
        assert np.linalg.norm(grad - g_ref) <= 1e-3 * np.linalg.norm(g_ref), (grad, g_ref)
        assert abs(af - a_ref) <= 1e-4 * abs(a_ref) and abs(bf - b_ref) <= 1e-4 * max(abs(b_ref), abs(a_ref))


def test_gpu_gradient_matches_finite_differences_of_gpu_cost():
    g = _geom(K=3, n=(40, 36, 24))
    f0, xbar, u, scale = smooth_model(g, seed=11)
    m = make_model(g, f0, xbar, u, projector=1, ray_step_vox=STEP_VOX)
    _use_rm(g)
    rng = np.random.default_rng(4)
    w = (rng.uniform(-0.5, 0.5, 3) * scale).astype(np.float64)
    theta, a, b = 2.3, 0.95, 0.01
    _, p0 = oracle.evaluate(g, f0, xbar, u, w, theta)
    y = to_dev((p0 * 1.1 + 0.05).astype(np.float32))
    _, grad, _, _ = m.eval(y, theta, w, a, b)
    eps = 2e-3 * scale
    for k in range(3):
        e = np.zeros(3)
        e[k] = eps
        Jp = m.eval(y, theta, w + e, a, b, want_proj=False)[0]
        Jm = m.eval(y, theta, w - e, a, b, want_proj=False)[0]
        fd = (Jp - Jm) / (2 * eps)
        assert abs(fd - grad[k]) <= 2e-2 * np.linalg.norm(grad), (k, fd, grad[k])


def _check_solve(g, f0, xbar, u, lm, res, y, theta, w0, opts):
    ref = oracle.solve(g, f0, xbar, u, y, theta, w0, oracle_opts(opts), want_volume=False)
    if not (res.iters == ref["iters"] and np.array_equal(res.backtracks, ref["backtracks"][:res.iters])):
        o2 = oracle_opts(opts)                                                     # A16 (ii): replay
        o2.max_iter = res.iters
        ref = oracle.solve(g, f0, xbar, u, y, theta, w0, o2, want_volume=False,
                           forced_mu=np.concatenate([res.mu_trace, np.zeros(opts.max_iter)]))
    assert np.linalg.norm(res.w - ref["w"]) <= 1e-3 * np.linalg.norm(ref["w"]), (res.w, ref["w"])
    assert abs(res.J - ref["J"]) <= 1e-3 * ref["J"] + 1e-12
    assert abs(res.a - ref["a"]) <= 1e-4 * abs(ref["a"]) and abs(res.b - ref["b"]) <= 1e-4
    r_ref, _ = oracle.invert(g, xbar, u, ref["w"], lm)
    assert np.max(np.linalg.norm(res.landmarks - r_ref, axis=1)) <= 0.05           # mm
    assert np.all(np.diff(res.J_trace) <= 1e-9 * res.J0)


def test_solves_match_the_oracle_single_fan_and_batch():
    import paper_1004_0014_b200 as pc
    g = _geom(K=3, n=(44, 40, 26), det=(64, 40))
    _use_rm(g)
    f0, xbar, u, scale = smooth_model(g, seed=21)
    lm = np.array([[5.0, -4.0, 3.0], [-12.0, 8.0, -6.0]], np.float32)
    m = make_model(g, f0, xbar, u, landmarks=lm, max_batch=3, max_candidates=2, projector=1, ray_step_vox=STEP_VOX)
    rng = np.random.default_rng(2)
    thetas = np.array([0.4, 2.0, 4.4], np.float32)
    ys = []
    for th in thetas:
        w_true = (rng.uniform(-0.6, 0.6, 3) * scale).astype(np.float32)
        _, p = oracle.evaluate(g, f0, xbar, u, w_true, float(th))
        ys.append((p * (1 + 0.01 * rng.standard_normal(p.shape))).astype(np.float32))
    w0 = np.zeros(3, np.float32)
    opts = pc.Opts(max_iter=6)
    res = m.reconstruct(to_dev(ys[0]), float(thetas[0]), w0, opts, trace=True)
    _check_solve(g, f0, xbar, u, lm, res, ys[0], float(thetas[0]), w0, opts)
    fan = m.reconstruct(to_dev(ys[0]), float(thetas[0]), w0, pc.Opts(max_iter=6, batched_linesearch=2), trace=True)
    assert np.array_equal(fan.backtracks, res.backtracks)
    assert np.linalg.norm(fan.w - res.w) <= 1e-5 * np.linalg.norm(res.w)       # atomics: equal to rounding
    batch = m.reconstruct_batch(to_dev(np.stack(ys)), thetas, np.zeros((3, 3), np.float32), opts, trace=True)
    for b in range(3):
        _check_solve(g, f0, xbar, u, lm, batch[b], ys[b], float(thetas[b]), w0, opts)


def test_traverse_needs_the_siddon_projector():
    import paper_1004_0014_b200 as pc
    g = _geom()
    f0, xbar, u, _ = smooth_model(g, seed=3)
    m = make_model(g, f0, xbar, u, projector=1)
    with pytest.raises(pc.PcammError):
        m.traverse(0.3, 5, 5)
