"""Parity at the FULL sizes of BASELINE.json configs[3] and configs[4] (north_star: "matching the
oracle within the stated tolerances on all five configs"), in the launch configurations bench.py
times them in:

  C3  256x256x256 volume, K = 5 with hysteresis, detector 512x384, line search with all 8 candidate
      steps per pass (max_candidates = 8, batched_linesearch = 1);
  C4  512x512x128 volume, K = 3, detector 1024x768, several solves in flight (max_batch = 4,
      pcamm_reconstruct_batch), solves b = 0 and b = 3 checked.

Per config, against the oracle (fp64 C++, OpenMP) on the same float32 arrays: the whole warp element
by element, the projection at two gantry angles, one evaluation (J, g, the (a, b) fit) at a generic
w, and a 2-iteration solve with the tumour position (reading A16: the trajectory when the backtrack
counts agree, else the oracle replays the GPU's accepted steps).  Only the iteration count is
reduced; the grids are the configs'.  y always comes from the oracle's projector.

Bars (north_star / DESIGN.md section 3): warp rel-L2 <= 5e-6, projections rel-L2 <= 1e-5 (bar 1e-4),
J rel <= 1e-4, gradient rel-L2 <= 1e-3, w within 1e-3 ||w||, tumour <= 0.05 mm.
"""
import numpy as np
import pytest

import oracle
from tests.gpu_util import oracle_opts, rel_l2, to_dev, to_host

pytestmark = pytest.mark.gpu


def _fixture(name, frame_ids, **model_kw):
    import paper_1004_0014_b200 as pc
    from workloads import get_config
    from workloads.build import build_workload, ground_truth_volume
    from workloads.noise import add_noise
    cfg = get_config(name)
    wl = build_workload(cfg)
    g = oracle.Geometry(cfg.nx, cfg.ny, cfg.nz, cfg.hx, cfg.hy, cfg.hz, cfg.K, cfg.nu, cfg.nv, cfg.pu, cfg.pv,
                        cfg.sad, cfg.sdd)
    m = pc.Model(nx=cfg.nx, ny=cfg.ny, nz=cfg.nz, hx=cfg.hx, hy=cfg.hy, hz=cfg.hz, K=cfg.K, nu=cfg.nu, nv=cfg.nv,
                 pu=cfg.pu, pv=cfg.pv, f0=to_dev(wl.f0), mean_dvf=to_dev(wl.model.mean), eig_dvf=to_dev(wl.model.eig),
                 landmarks_mm=wl.landmarks, sad=cfg.sad, sdd=cfg.sdd, **model_kw)
    frames = [wl.frames[i] for i in frame_ids]
    # the measured projections come from the oracle's projector (never from the CUDA path)
    ys = [add_noise(oracle.project(g, ground_truth_volume(wl, fr), fr.angle_rad), cfg.noise, seed=fr.index)
          for fr in frames]
    return cfg, wl, g, m, frames, ys


def _w_probe(wl):
    # a generic point of coefficient space: the training coefficients' scale, no lattice alignment
    c = np.asarray(wl.model.coeffs)
    f = np.array([0.83, -0.61, 0.47, -0.38, 0.29, 0.21, -0.17, 0.13])[:c.shape[1]]
    return (f * np.abs(c).max(axis=0)).astype(np.float32)


def _check_functions(cfg, wl, g, m, fr, y, angles):
    w = _w_probe(wl)
    f_ref = oracle.warp(g, wl.f0, wl.model.mean, wl.model.eig, w)
    f_gpu = to_host(m.warp(w))
    assert rel_l2(f_gpu, f_ref) <= 5e-6
    assert np.max(np.abs(f_gpu - f_ref)) <= 1e-5 * np.max(np.abs(f_ref))
    f32 = f_ref.astype(np.float32)
    del f_gpu
    for theta in angles:
        p_ref = oracle.project(g, f32, theta)
        p_gpu = to_host(m.project(to_dev(f32), theta))
        assert rel_l2(p_gpu, p_ref) <= 1e-5, theta          # north_star bar is 1e-4
        assert np.max(np.abs(p_gpu - p_ref)) <= 1e-4 * np.max(np.abs(p_ref))
    a, b = 0.93, 0.04
    p_ref = oracle.project(g, f32, fr.angle_rad)
    J_ref = oracle.cost(p_ref, y, a, b)
    g_ref = oracle.gradient(g, wl.f0, wl.model.mean, wl.model.eig, w, a, b, p_ref, y, fr.angle_rad)
    _, a_ref, b_ref = oracle.lsfit(p_ref, y)
    J, grad, (af, bf), p = m.eval(to_dev(y), fr.angle_rad, w, a, b)
    assert rel_l2(to_host(p), p_ref) <= 1e-5
    assert abs(J - J_ref) <= 1e-4 * J_ref
    assert np.linalg.norm(grad - g_ref) <= 1e-3 * np.linalg.norm(g_ref), (grad, g_ref)
    assert abs(af - a_ref) <= 1e-4 * abs(a_ref) and abs(bf - b_ref) <= 1e-4 * max(abs(b_ref), abs(a_ref))


def _check_solve(wl, g, res, y, theta, w0, opts):
    ref = oracle.solve(g, wl.f0, wl.model.mean, wl.model.eig, y, theta, w0, oracle_opts(opts), want_volume=False)
    if not (res.iters == ref["iters"] and np.array_equal(res.backtracks, ref["backtracks"][:res.iters])):
        o2 = oracle_opts(opts)                                                     # A16 (ii): replay
        o2.max_iter = res.iters
        ref = oracle.solve(g, wl.f0, wl.model.mean, wl.model.eig, y, theta, w0, o2, want_volume=False,
                           forced_mu=np.concatenate([res.mu_trace, np.zeros(opts.max_iter)]))
    assert np.linalg.norm(res.w - ref["w"]) <= 1e-3 * np.linalg.norm(ref["w"]), (res.w, ref["w"])
    assert abs(res.J - ref["J"]) <= 1e-3 * ref["J"]
    assert abs(res.a - ref["a"]) <= 1e-4 * abs(ref["a"]) and abs(res.b - ref["b"]) <= 1e-4
    r_ref, _ = oracle.invert(g, wl.model.mean, wl.model.eig, ref["w"], wl.landmarks)
    assert np.max(np.linalg.norm(res.landmarks - r_ref, axis=1)) <= 0.05           # mm
    assert np.all(np.diff(res.J_trace) <= 1e-9 * res.J0)


@pytest.fixture(scope="module")
def c3():
    out = _fixture("C3", [63], max_candidates=8)
    yield out
    del out


def test_c3_functions_full_size(c3):
    cfg, wl, g, m, frames, ys = c3
    _check_functions(cfg, wl, g, m, frames[0], ys[0], (frames[0].angle_rad, np.deg2rad(200.0)))


def test_c3_solve_all_candidates_per_pass_full_size(c3):
    import paper_1004_0014_b200 as pc
    cfg, wl, g, m, frames, ys = c3
    opts = pc.Opts(max_iter=2, batched_linesearch=1)
    w0 = np.zeros(cfg.K, np.float32)
    res = m.reconstruct(to_dev(ys[0]), frames[0].angle_rad, w0, opts, trace=True)
    assert res.iters == 2
    _check_solve(wl, g, res, ys[0], frames[0].angle_rad, w0, opts)


@pytest.fixture(scope="module")
def c4():
    out = _fixture("C4", [17, 111, 203, 310], max_batch=4)
    yield out
    del out


def test_c4_functions_full_size(c4):
    cfg, wl, g, m, frames, ys = c4
    _check_functions(cfg, wl, g, m, frames[0], ys[0], (frames[0].angle_rad, np.deg2rad(135.0)))


def test_c4_four_solves_in_flight_full_size(c4):
    import paper_1004_0014_b200 as pc
    cfg, wl, g, m, frames, ys = c4
    opts = pc.Opts(max_iter=2)
    w0 = np.zeros((4, cfg.K), np.float32)
    angles = np.array([fr.angle_rad for fr in frames], np.float32)
    batch = m.reconstruct_batch(to_dev(np.stack(ys)), angles, w0, opts, trace=True)
    for b in (0, 3):
        assert batch[b].iters == 2
        _check_solve(wl, g, batch[b], ys[b], float(angles[b]), w0[b], opts)
