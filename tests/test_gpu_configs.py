"""The five workload configurations of BASELINE.json as parity cases (the headline one, C2, is
tests/test_gpu_fullsize.py): whole per-projection solves on the DESIGN.md workload recipe (analytic
phantom, PCA of the training DVFs, measured projection from the oracle's projector plus the config's
noise), CUDA path against the oracle through the C ABI.

C0 and C1 run at full size.  C3 (K = 5 with hysteresis, all 8 candidate steps per line-search pass)
and C4 (fine detector, several solves in flight) run here on reduced grids with the same recipe and
more iterations; their FULL sizes are tests/test_gpu_fullsize_c3c4.py.

Bars (north_star; reading A16): w within 1e-3 ||w||, tumour position <= 0.05 mm, J and (a, b) to
1e-3 / 1e-4; trajectories compared when the backtrack counts agree, else the oracle replays the
GPU's accepted steps.
"""
import numpy as np
import pytest

import oracle
from tests.gpu_util import oracle_opts, to_dev

pytestmark = pytest.mark.gpu


def _setup(cfg, frame_ids, max_batch=1, max_candidates=1):
    import paper_1004_0014_b200 as pc
    from workloads.build import build_workload, ground_truth_volume
    from workloads.noise import add_noise
    wl = build_workload(cfg)
    g = oracle.Geometry(cfg.nx, cfg.ny, cfg.nz, cfg.hx, cfg.hy, cfg.hz, cfg.K, cfg.nu, cfg.nv, cfg.pu, cfg.pv,
                        cfg.sad, cfg.sdd)
    m = pc.Model(nx=cfg.nx, ny=cfg.ny, nz=cfg.nz, hx=cfg.hx, hy=cfg.hy, hz=cfg.hz, K=cfg.K, nu=cfg.nu, nv=cfg.nv,
                 pu=cfg.pu, pv=cfg.pv, f0=to_dev(wl.f0), mean_dvf=to_dev(wl.model.mean), eig_dvf=to_dev(wl.model.eig),
                 landmarks_mm=wl.landmarks, sad=cfg.sad, sdd=cfg.sdd, max_batch=max_batch,
                 max_candidates=max_candidates)
    frames = [wl.frames[i] for i in frame_ids]
    # measured projections from the oracle's projector (never from the CUDA path)
    ys = [add_noise(oracle.project(g, ground_truth_volume(wl, fr), fr.angle_rad), cfg.noise, seed=fr.index)
          for fr in frames]
    return wl, g, m, frames, ys


def _check(wl, g, res, y, theta, w0, opts):
    ref = oracle.solve(g, wl.f0, wl.model.mean, wl.model.eig, y, theta, w0, oracle_opts(opts), want_volume=False)
    if not (res.iters == ref["iters"] and np.array_equal(res.backtracks, ref["backtracks"][:res.iters])):
        o2 = oracle_opts(opts)
        o2.max_iter = res.iters
        ref = oracle.solve(g, wl.f0, wl.model.mean, wl.model.eig, y, theta, w0, o2, want_volume=False,
                           forced_mu=np.concatenate([res.mu_trace, np.zeros(opts.max_iter)]))
    assert np.linalg.norm(res.w - ref["w"]) <= 1e-3 * np.linalg.norm(ref["w"]), (res.w, ref["w"])
    assert abs(res.J - ref["J"]) <= 1e-3 * ref["J"]
    assert abs(res.a - ref["a"]) <= 1e-4 * abs(ref["a"]) and abs(res.b - ref["b"]) <= 1e-4
    r_ref, _ = oracle.invert(g, wl.model.mean, wl.model.eig, ref["w"], wl.landmarks)
    assert np.max(np.linalg.norm(res.landmarks - r_ref, axis=1)) <= 0.05           # mm
    assert np.all(np.diff(res.J_trace) <= 1e-9 * res.J0)
    return ref


def test_c0_full_size_two_projections():
    import paper_1004_0014_b200 as pc
    from workloads import get_config
    cfg = get_config("C0")                                     # 32^3 @ 4 mm, 64x48 detector, 30 iterations
    wl, g, m, frames, ys = _setup(cfg, [2, 5])
    opts = pc.Opts(max_iter=cfg.iterations)
    w = np.zeros(cfg.K, np.float32)
    for fr, y in zip(frames, ys):                              # the second starts from the first's answer (L141)
        res = m.reconstruct(to_dev(y), fr.angle_rad, w, opts, trace=True)
        _check(wl, g, res, y, fr.angle_rad, w, opts)
        w = res.w


def test_c1_full_size():
    import paper_1004_0014_b200 as pc
    from workloads import get_config
    cfg = get_config("C1")                                     # 128x128x64 @ 3 mm, 256x192 detector
    wl, g, m, frames, ys = _setup(cfg, [100])
    opts = pc.Opts(max_iter=6)
    res = m.reconstruct(to_dev(ys[0]), frames[0].angle_rad, np.zeros(cfg.K, np.float32), opts, trace=True)
    assert res.iters == 6
    _check(wl, g, res, ys[0], frames[0].angle_rad, np.zeros(cfg.K, np.float32), opts)


def test_c3_recipe_batched_line_search():
    """K = 5, hysteresis between the AP and SI motion, all 8 candidate steps per pass (config C3's
    recipe on a 64x64x64 grid)."""
    import paper_1004_0014_b200 as pc
    from workloads.configs import small_config
    cfg = small_config("C3s", 64, 64, 64, 6.0, 128, 96, 3.1, K=5, hysteresis=True, batched_linesearch=True)
    wl, g, m, frames, ys = _setup(cfg, [40], max_candidates=8)
    opts = pc.Opts(max_iter=5, batched_linesearch=1)
    w0 = np.zeros(cfg.K, np.float32)
    res = m.reconstruct(to_dev(ys[0]), frames[0].angle_rad, w0, opts, trace=True)
    _check(wl, g, res, ys[0], frames[0].angle_rad, w0, opts)
    seq = m.reconstruct(to_dev(ys[0]), frames[0].angle_rad, w0, pc.Opts(max_iter=5), trace=True)
    assert np.array_equal(seq.backtracks, res.backtracks) and np.array_equal(seq.w, res.w)


def test_c4_recipe_solves_in_flight():
    """Fine detector (4 pixels per voxel shadow), four independent solves in flight at different
    gantry angles and breathing states (config C4's recipe on a 128x128x32 grid)."""
    import paper_1004_0014_b200 as pc
    from workloads.configs import small_config
    cfg = small_config("C4s", 128, 128, 32, 3.92, 256, 192, 1.55)
    ids = [17, 111, 203, 310]
    wl, g, m, frames, ys = _setup(cfg, ids, max_batch=4)
    opts = pc.Opts(max_iter=4)
    w0 = np.zeros((4, cfg.K), np.float32)
    angles = np.array([fr.angle_rad for fr in frames], np.float32)
    batch = m.reconstruct_batch(to_dev(np.stack(ys)), angles, w0, opts, trace=True)
    for b in (0, 3):
        _check(wl, g, batch[b], ys[b], float(angles[b]), w0[b], opts)
