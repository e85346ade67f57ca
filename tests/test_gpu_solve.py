"""Parity of the whole per-projection solve against the oracle, through the C ABI.

Reading A16: the Armijo accept/reject is a discrete decision, so trajectories are compared when the
logged backtrack counts agree (level ii; otherwise the oracle is re-run with the GPU's logged steps
forced), and converged answers are compared directly (level iii).  Bars: ||w - w_or|| <= 1e-3 ||w_or||,
tumour position <= 0.05 mm (north_star).
"""
import numpy as np
import pytest

import oracle
from tests.gpu_util import make_model, oracle_opts, rel_l2, to_dev, to_host
from tests.util import geom, smooth_model

pytestmark = pytest.mark.gpu


def _problem(K=3, seed=11, n=(40, 36, 20), det=(66, 26), noise=0.003, disp_vox=1.0, theta=0.6, B=1, C=1,
             landmarks=True):
    g = geom(nx=n[0], ny=n[1], nz=n[2], h=(3.0, 3.0, 3.0), K=K, nu=det[0], nv=det[1], pitch=(3.2, 3.2),
             centre=(0.37, 0.11, 0.23))
    f0, xbar, u, scale = smooth_model(g, seed=seed, disp_vox=disp_vox)
    rng = np.random.default_rng(seed)
    w_star = rng.uniform(0.4, 1.0, K) * rng.choice([-1, 1], K) * scale
    _, p = oracle.evaluate(g, f0, xbar, u, w_star.astype(np.float32), theta)
    y = (p + noise * rng.standard_normal(p.shape)).astype(np.float32)
    lm = np.array([[10.0, -8.0, 5.0], [-14.0, 6.0, -9.0]], np.float32) if landmarks else None
    m = make_model(g, f0, xbar, u, landmarks=lm, max_batch=B, max_candidates=C)
    return g, f0, xbar, u, scale, theta, y, w_star, lm, m


def _compare_with_oracle(g, f0, xbar, u, y, theta, w0, lm, res, opts):
    import paper_1004_0014_b200 as pc
    ref = oracle.solve(g, f0, xbar, u, y, theta, w0, oracle_opts(opts))
    same_path = (res.iters == ref["iters"] and res.status == ref["status"]
                 and np.array_equal(res.backtracks, ref["backtracks"]))
    if not same_path:   # A16 (ii): replay the GPU's accepted steps in the oracle
        forced = np.concatenate([res.mu_trace, np.zeros(opts.max_iter)])
        o2 = oracle_opts(opts)
        o2.max_iter = res.iters
        ref = oracle.solve(g, f0, xbar, u, y, theta, w0, o2, forced_mu=forced)
    nw = np.linalg.norm(ref["w"])
    assert np.linalg.norm(res.w - ref["w"]) <= 1e-3 * nw, (res.w, ref["w"], same_path)
    assert abs(res.J - ref["J"]) <= 1e-3 * ref["J"] + 1e-9 * ref["J0"]
    assert abs(res.a - ref["a"]) <= 1e-4 * abs(ref["a"]) and abs(res.b - ref["b"]) <= 1e-4
    if lm is not None:
        r_ref, _ = oracle.invert(g, xbar, u, ref["w"], lm, opts.inv_max_iter, opts.inv_tol_mm)
        assert np.max(np.linalg.norm(res.landmarks - r_ref, axis=1)) <= 0.05
    return same_path, ref


@pytest.mark.parametrize("loop_mode", [0, 1])
def test_solve_trajectory_matches_oracle(loop_mode):
    import paper_1004_0014_b200 as pc
    g, f0, xbar, u, scale, theta, y, w_star, lm, m = _problem()
    opts = pc.Opts(max_iter=12, loop_mode=loop_mode)
    res = m.reconstruct(to_dev(y), theta, np.zeros(g.K), opts, trace=True)
    assert res.status == pc.S_MAXITER and res.iters == 12
    J = res.J_trace
    assert len(J) == 13 and np.all(J >= 0) and np.all(np.diff(J) <= 1e-9 * J[0])
    assert J[-1] < 0.2 * J[0]
    same_path, ref = _compare_with_oracle(g, f0, xbar, u, y, theta, np.zeros(g.K), lm, res, opts)
    assert same_path, (res.backtracks, ref["backtracks"])
    np.testing.assert_allclose(res.J_trace, ref["J_trace"], rtol=1e-3, atol=1e-9 * J[0])
    np.testing.assert_allclose(res.mu_trace, ref["mu_trace"], rtol=1e-3)


def test_graph_and_host_loop_modes_agree_bitwise():
    import paper_1004_0014_b200 as pc
    g, f0, xbar, u, scale, theta, y, w_star, lm, m = _problem(seed=5)
    yd = to_dev(y)
    r0 = m.reconstruct(yd, theta, np.zeros(g.K), pc.Opts(max_iter=8, loop_mode=0), trace=True)
    r1 = m.reconstruct(yd, theta, np.zeros(g.K), pc.Opts(max_iter=8, loop_mode=1), trace=True)
    assert np.array_equal(r0.w, r1.w) and r0.J == r1.J and np.array_equal(r0.backtracks, r1.backtracks)
    assert np.array_equal(r0.landmarks, r1.landmarks)
    # and a second graph launch reproduces the first (no state leaks between calls)
    r2 = m.reconstruct(yd, theta, np.zeros(g.K), pc.Opts(max_iter=8, loop_mode=0), trace=True)
    assert np.array_equal(r0.w, r2.w) and r0.J == r2.J


def test_volume_output_is_the_warp_at_the_final_w():
    import torch
    import paper_1004_0014_b200 as pc
    g, f0, xbar, u, scale, theta, y, w_star, lm, m = _problem(seed=6)
    vol = torch.empty(g.vshape, dtype=torch.float32, device="cuda:0")
    res = m.reconstruct(to_dev(y), theta, np.zeros(g.K), pc.Opts(max_iter=5), volume_out=vol)
    assert np.array_equal(to_host(vol), to_host(m.warp(res.w)))
    assert rel_l2(to_host(vol), oracle.warp(g, f0, xbar, u, res.w)) <= 5e-6


@pytest.mark.parametrize("K,seed", [(3, 11), (2, 12)])
def test_planted_coefficients_are_recovered(K, seed):
    """north_star: noise-free y = P warp(w*) => the converged solve returns w*, a = 1, b = 0."""
    import paper_1004_0014_b200 as pc
    g, f0, xbar, u, scale, theta, y, w_star, lm, m = _problem(K=K, seed=seed, noise=0.0, n=(16, 14, 12), det=(24, 18))
    res = m.reconstruct(to_dev(y), theta, np.zeros(K), pc.Opts(max_iter=400), trace=True)
    assert np.linalg.norm(res.w - w_star) <= 1e-3 * np.linalg.norm(w_star), (res.w, w_star, res.J, res.status)
    assert abs(res.a - 1) < 1e-4 and abs(res.b) < 1e-4
    r_ref, _ = oracle.invert(g, xbar, u, w_star.astype(np.float32), lm)
    assert np.max(np.linalg.norm(res.landmarks - r_ref, axis=1)) <= 0.05


def test_converged_solution_matches_oracle():
    """A16 (iii): both sides run to a tight stop; compare the minimisers."""
    import paper_1004_0014_b200 as pc
    g, f0, xbar, u, scale, theta, y, w_star, lm, m = _problem(seed=3, noise=0.002, n=(24, 20, 14), det=(36, 20))
    opts = pc.Opts(max_iter=300)
    res = m.reconstruct(to_dev(y), theta, np.zeros(g.K), opts)
    ref = oracle.solve(g, f0, xbar, u, y, theta, np.zeros(g.K), oracle_opts(opts))
    assert np.linalg.norm(res.w - ref["w"]) <= 1e-3 * np.linalg.norm(ref["w"])
    assert res.J <= ref["J"] * (1 + 1e-4)
    r_ref, _ = oracle.invert(g, xbar, u, ref["w"], lm)
    assert np.max(np.linalg.norm(res.landmarks - r_ref, axis=1)) <= 0.05


def test_batched_linesearch_equals_sequential():
    import paper_1004_0014_b200 as pc
    g, f0, xbar, u, scale, theta, y, w_star, lm, m = _problem(seed=4, C=8, K=5)
    yd = to_dev(y)
    r1 = m.reconstruct(yd, theta, np.zeros(g.K), pc.Opts(max_iter=8), trace=True)
    r2 = m.reconstruct(yd, theta, np.zeros(g.K), pc.Opts(max_iter=8, batched_linesearch=1), trace=True)
    assert np.array_equal(r1.backtracks, r2.backtracks)
    np.testing.assert_allclose(r1.w, r2.w, rtol=1e-6)
    np.testing.assert_allclose(r1.J_trace, r2.J_trace, rtol=1e-9)
    _compare_with_oracle(g, f0, xbar, u, y, theta, np.zeros(g.K), lm, r2, pc.Opts(max_iter=8, batched_linesearch=1))


@pytest.mark.parametrize("fan", [2, 3])
def test_partial_fan_takes_the_steps_of_sequential_backtracking(fan):
    """pcamm_opts.batched_linesearch = F >= 2: F candidates per pass, the next F if none passes; the
    accepted steps are those of sequential backtracking (reading A7), bit for bit."""
    import paper_1004_0014_b200 as pc
    g, f0, xbar, u, scale, theta, y, w_star, lm, m = _problem(seed=5, C=3)
    yd = to_dev(y)
    r1 = m.reconstruct(yd, theta, np.zeros(g.K), pc.Opts(max_iter=8, init_step_vox=6.0), trace=True)
    r2 = m.reconstruct(yd, theta, np.zeros(g.K), pc.Opts(max_iter=8, init_step_vox=6.0, batched_linesearch=fan), trace=True)
    assert r1.backtracks.max() >= 2                      # the runs do backtrack past one fan
    assert np.array_equal(r1.backtracks, r2.backtracks) and np.array_equal(r1.mu_trace, r2.mu_trace)
    assert np.array_equal(r1.w, r2.w) and r1.J == r2.J


def test_batch_of_solves_equals_single_solves():
    import paper_1004_0014_b200 as pc
    B = 5
    g, f0, xbar, u, scale, theta, y, w_star, lm, m = _problem(seed=8, B=B)
    rng = np.random.default_rng(8)
    angles = np.array([0.1, 0.8, 1.7, 3.3, 5.2], np.float32)
    ys, w0s = [], []
    for b in range(B):
        wb = rng.uniform(-1, 1, g.K) * scale
        _, p = oracle.evaluate(g, f0, xbar, u, wb.astype(np.float32), float(angles[b]))
        ys.append((p + 0.003 * rng.standard_normal(p.shape)).astype(np.float32))
        w0s.append(0.2 * rng.uniform(-1, 1, g.K) * scale)
    yd = to_dev(np.stack(ys))
    w0 = np.stack(w0s).astype(np.float32)
    opts = pc.Opts(max_iter=6)
    batch = m.reconstruct_batch(yd, angles, w0, opts, trace=True)
    for b in range(B):
        single = m.reconstruct(yd[b], float(angles[b]), w0[b], opts, trace=True)
        # same arithmetic per voxel and ray; the K gradient sums are grouped per tile in the batched
        # kernel and per thread in the single-solve one (both fixed orders), so equality holds to
        # float32 summation-order rounding, not bitwise
        assert np.linalg.norm(batch[b].w - single.w) <= 1e-5 * np.linalg.norm(single.w), b
        assert abs(batch[b].J - single.J) <= 1e-5 * single.J and np.array_equal(batch[b].backtracks, single.backtracks)
        np.testing.assert_allclose(batch[b].landmarks, single.landmarks, rtol=0, atol=1e-4)
    _compare_with_oracle(g, f0, xbar, u, ys[2], float(angles[2]), w0[2], lm, batch[2], opts)


def test_stopping_rules_and_soft_status():
    import paper_1004_0014_b200 as pc
    g, f0, xbar, u, scale, theta, y, w_star, lm, m = _problem(seed=6, noise=0.0)
    yd = to_dev(y)
    # gradient tolerance: stops before the first step
    res = m.reconstruct(yd, theta, w_star, pc.Opts(max_iter=5, grad_tol=1e9), trace=True)
    assert res.status == pc.S_GRADTOL and res.iters == 0
    np.testing.assert_array_equal(res.w, w_star.astype(np.float32))
    assert len(res.J_trace) == 1 and res.J_trace[0] == res.J == res.J0
    # max_iter = 0: only the initial fit
    res = m.reconstruct(yd, theta, w_star, pc.Opts(max_iter=0))
    assert res.status == pc.S_MAXITER and res.iters == 0 and abs(res.a - 1) < 1e-4
    # line search failure: at the noise-free optimum no step decreases J by Armijo's margin
    res = m.reconstruct(yd, theta, np.zeros(g.K), pc.Opts(max_iter=500), trace=True)
    assert res.status == pc.S_LINESEARCH and res.iters < 500
    assert res.backtracks.size == res.iters and np.all(np.diff(res.J_trace) <= 1e-9 * res.J0)


def test_hard_errors():
    import torch
    import paper_1004_0014_b200 as pc
    g, f0, xbar, u, scale, theta, y, w_star, lm, m = _problem(seed=6)
    # y constant: singular intensity fit (reading A8)
    with pytest.raises(pc.PcammError) as e:
        m.reconstruct(to_dev(np.full(g.pshape, 0.5, np.float32)), theta, np.zeros(g.K))
    assert e.value.code == pc.E_SINGULAR
    # non-finite y
    ybad = y.copy()
    ybad[3, 5] = np.nan
    with pytest.raises(pc.PcammError) as e:
        m.reconstruct(to_dev(ybad), theta, np.zeros(g.K))
    assert e.value.code == pc.E_NONFINITE
    # invalid arguments
    with pytest.raises(pc.PcammError) as e:
        m.reconstruct(to_dev(y), theta, np.zeros(g.K), pc.Opts(max_backtracks=0))
    assert e.value.code == pc.E_INVALID
    with pytest.raises(pc.PcammError) as e:
        m.reconstruct(to_dev(y), theta, np.zeros(g.K), pc.Opts(batched_linesearch=1))   # max_candidates = 1
    assert e.value.code == pc.E_INVALID
    # non-finite model input
    fbad = f0.copy()
    fbad[1, 2, 3] = np.inf
    with pytest.raises(pc.PcammError) as e:
        make_model(g, fbad, xbar, u)
    assert e.value.code == pc.E_NONFINITE
    # source inside the volume's bounding sphere
    gbad = geom(nx=40, ny=36, nz=20, h=(3.0, 3.0, 3.0), K=3, nu=66, nv=26, pitch=(3.2, 3.2), sad=60.0, sdd=400.0)
    with pytest.raises(pc.PcammError) as e:
        make_model(gbad, f0, xbar, u)
    assert e.value.code == pc.E_INVALID
    # the model is still usable after errors
    res = m.reconstruct(to_dev(y), theta, np.zeros(g.K), pc.Opts(max_iter=2))
    assert res.status == pc.S_MAXITER


def test_host_projection_entry_point_matches_device_one():
    import paper_1004_0014_b200 as pc
    g, f0, xbar, u, scale, theta, y, w_star, lm, m = _problem(seed=9)
    r0 = m.reconstruct(to_dev(y), theta, np.zeros(g.K), pc.Opts(max_iter=4))
    r1 = m.reconstruct(y, theta, np.zeros(g.K), pc.Opts(max_iter=4), host_y=True)
    assert np.array_equal(r0.w, r1.w) and r0.J == r1.J
