"""Parity at BASELINE.json's headline size (configs[2] = C2: 256x256x128 volume, K = 3, detector
512x384), in the launch configuration bench.py times (one CUDA graph per solve, TMA-fed warp and
gradient kernels on a persistent grid, segmented projector), on the workload recipe of DESIGN.md.

The oracle (fp64 C++, OpenMP) needs about a second per primitive at this size, so whole outputs are
compared, not samples: warp and projection element by element, cost / gradient / intensity fit at
the same (w, a, b), then a short solve (reading A16: trajectory when the backtrack counts agree, else
the oracle replays the GPU's accepted steps) and the tumour position.

Bars (north_star): projections rel-L2 <= 1e-4, J rel <= 1e-4, gradient rel-L2 <= 1e-3,
w within 1e-3 ||w||, tumour <= 0.05 mm; warp rel-L2 <= 5e-6.
"""
import numpy as np
import pytest

import oracle
from tests.gpu_util import oracle_opts, rel_l2, to_dev, to_host

pytestmark = pytest.mark.gpu

FRAME = 63      # a frame of the block bench.py times (gantry at 63 degrees, mid-inhale)


@pytest.fixture(scope="module")
def c2():
    import paper_1004_0014_b200 as pc
    from workloads import get_config
    from workloads.build import build_workload, ground_truth_volume
    from workloads.noise import add_noise
    cfg = get_config("C2")
    wl = build_workload(cfg)
    g = oracle.Geometry(cfg.nx, cfg.ny, cfg.nz, cfg.hx, cfg.hy, cfg.hz, cfg.K, cfg.nu, cfg.nv, cfg.pu, cfg.pv,
                        cfg.sad, cfg.sdd)
    m = pc.Model(nx=cfg.nx, ny=cfg.ny, nz=cfg.nz, hx=cfg.hx, hy=cfg.hy, hz=cfg.hz, K=cfg.K, nu=cfg.nu, nv=cfg.nv,
                 pu=cfg.pu, pv=cfg.pv, f0=to_dev(wl.f0), mean_dvf=to_dev(wl.model.mean), eig_dvf=to_dev(wl.model.eig),
                 landmarks_mm=wl.landmarks, sad=cfg.sad, sdd=cfg.sdd)
    fr = wl.frames[FRAME]
    # the measured projection comes from the oracle's projector (never from the CUDA path)
    y = add_noise(oracle.project(g, ground_truth_volume(wl, fr), fr.angle_rad), cfg.noise, seed=FRAME)
    return cfg, wl, g, m, fr, y


def _w_probe(wl):
    # a generic point of coefficient space: the training coefficients' scale, no lattice alignment
    c = np.asarray(wl.model.coeffs)
    return (np.array([0.83, -0.61, 0.47])[:c.shape[1]] * np.abs(c).max(axis=0)).astype(np.float32)


def test_c2_warp_and_projection(c2):
    cfg, wl, g, m, fr, y = c2
    w = _w_probe(wl)
    f_ref = oracle.warp(g, wl.f0, wl.model.mean, wl.model.eig, w)
    f_gpu = to_host(m.warp(w))
    assert rel_l2(f_gpu, f_ref) <= 5e-6
    assert np.max(np.abs(f_gpu - f_ref)) <= 1e-5 * np.max(np.abs(f_ref))
    # identity DVF coefficients do not exist here (xbar != 0): bit-exactness is covered at small size
    for theta in (fr.angle_rad, np.deg2rad(45.0), np.deg2rad(200.0)):
        p_ref = oracle.project(g, f_ref.astype(np.float32), theta)
        p_gpu = to_host(m.project(to_dev(f_ref.astype(np.float32)), theta))
        assert rel_l2(p_gpu, p_ref) <= 1e-5, theta          # north_star bar is 1e-4
        assert np.max(np.abs(p_gpu - p_ref)) <= 1e-4 * np.max(np.abs(p_ref))


def test_c2_cost_gradient_fit(c2):
    cfg, wl, g, m, fr, y = c2
    w = _w_probe(wl)
    a, b = 0.93, 0.04
    _, p_ref = oracle.evaluate(g, wl.f0, wl.model.mean, wl.model.eig, w, fr.angle_rad)
    J_ref = oracle.cost(p_ref, y, a, b)
    g_ref = oracle.gradient(g, wl.f0, wl.model.mean, wl.model.eig, w, a, b, p_ref, y, fr.angle_rad)
    _, a_ref, b_ref = oracle.lsfit(p_ref, y)
    J, grad, (af, bf), p = m.eval(to_dev(y), fr.angle_rad, w, a, b)
    assert rel_l2(to_host(p), p_ref) <= 1e-5
    assert abs(J - J_ref) <= 1e-4 * J_ref
    assert np.linalg.norm(grad - g_ref) <= 1e-3 * np.linalg.norm(g_ref), (grad, g_ref)
    assert abs(af - a_ref) <= 1e-4 * abs(a_ref) and abs(bf - b_ref) <= 1e-4 * max(abs(b_ref), abs(a_ref))


def test_c2_solve_and_tumour_position(c2):
    import paper_1004_0014_b200 as pc
    cfg, wl, g, m, fr, y = c2
    opts = pc.Opts(max_iter=4)
    w0 = np.zeros(cfg.K, np.float32)
    res = m.reconstruct(to_dev(y), fr.angle_rad, w0, opts, trace=True)
    assert res.iters == 4 and np.all(np.diff(res.J_trace) <= 1e-9 * res.J0)
    ref = oracle.solve(g, wl.f0, wl.model.mean, wl.model.eig, y, fr.angle_rad, w0, oracle_opts(opts), want_volume=False)
    if not np.array_equal(res.backtracks, ref["backtracks"]):                      # A16 (ii): replay
        o2 = oracle_opts(opts)
        ref = oracle.solve(g, wl.f0, wl.model.mean, wl.model.eig, y, fr.angle_rad, w0, o2,
                           forced_mu=np.concatenate([res.mu_trace, np.zeros(opts.max_iter)]), want_volume=False)
    assert np.linalg.norm(res.w - ref["w"]) <= 1e-3 * np.linalg.norm(ref["w"]), (res.w, ref["w"])
    assert abs(res.J - ref["J"]) <= 1e-3 * ref["J"]
    assert abs(res.a - ref["a"]) <= 1e-4 * abs(ref["a"]) and abs(res.b - ref["b"]) <= 1e-4
    r_ref, _ = oracle.invert(g, wl.model.mean, wl.model.eig, ref["w"], wl.landmarks)
    assert np.max(np.linalg.norm(res.landmarks - r_ref, axis=1)) <= 0.05           # mm
    # and the volume handed back is the warp at the final coefficients
    import torch
    vol_dev = torch.empty((cfg.nz, cfg.ny, cfg.nx), dtype=torch.float32, device="cuda:0")
    m.reconstruct(to_dev(y), fr.angle_rad, w0, opts, volume_out=vol_dev)
    vol = to_host(vol_dev)
    assert rel_l2(vol, oracle.warp(g, wl.f0, wl.model.mean, wl.model.eig, ref["w"].astype(np.float32))) <= 2e-5


def test_c2_solve_in_the_bench_configuration(c2):
    """What bench.py times by default: a model with two candidate slots, two Armijo candidates per
    line-search pass (reading B7), the gradient from the records the warp kernel leaves, the certain
    passes in front of the graph's loop.  Against the sequential solve of the default model (the same
    accepted steps, bit for bit) and against the oracle."""
    import paper_1004_0014_b200 as pc
    cfg, wl, g, m, fr, y = c2
    m2 = pc.Model(nx=cfg.nx, ny=cfg.ny, nz=cfg.nz, hx=cfg.hx, hy=cfg.hy, hz=cfg.hz, K=cfg.K, nu=cfg.nu, nv=cfg.nv,
                  pu=cfg.pu, pv=cfg.pv, f0=to_dev(wl.f0), mean_dvf=to_dev(wl.model.mean), eig_dvf=to_dev(wl.model.eig),
                  landmarks_mm=wl.landmarks, sad=cfg.sad, sdd=cfg.sdd, max_candidates=2)
    w0 = np.zeros(cfg.K, np.float32)
    seq = m.reconstruct(to_dev(y), fr.angle_rad, w0, pc.Opts(max_iter=4), trace=True)
    opts = pc.Opts(max_iter=4, batched_linesearch=2)
    res = m2.reconstruct(to_dev(y), fr.angle_rad, w0, opts, trace=True)
    assert res.iters == 4 and np.array_equal(res.backtracks, seq.backtracks)
    assert np.array_equal(res.w, seq.w) and res.J == seq.J and res.a == seq.a and res.b == seq.b
    assert np.array_equal(res.landmarks, seq.landmarks)
    ref = oracle.solve(g, wl.f0, wl.model.mean, wl.model.eig, y, fr.angle_rad, w0, oracle_opts(pc.Opts(max_iter=4)),
                       forced_mu=np.concatenate([res.mu_trace, np.zeros(4)]), want_volume=False)
    assert np.linalg.norm(res.w - ref["w"]) <= 1e-3 * np.linalg.norm(ref["w"]), (res.w, ref["w"])
    assert abs(res.J - ref["J"]) <= 1e-3 * ref["J"]
    r_ref, _ = oracle.invert(g, wl.model.mean, wl.model.eig, ref["w"], wl.landmarks)
    assert np.max(np.linalg.norm(res.landmarks - r_ref, axis=1)) <= 0.05           # mm
    # the records really were in use: the gradient loaded no field tiles
    m2.eval(to_dev(y), fr.angle_rad, res.w, res.a, res.b, want_proj=False)
    m2.tile_counts(reset=True)
    m2.time_kernel(2, 1)
    tc = m2.tile_counts(reset=True)
    assert tc[1] == 0 and tc[4] > 0
