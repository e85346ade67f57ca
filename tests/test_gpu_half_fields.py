"""Reduced-precision field storage (pcamm_geometry.field_storage = 1): u_k kept in
half precision with a power-of-two scale per eigenvector field, x-bar in float.

Two things are checked.  (1) Parity: the model then IS the rounded one, so the CUDA path is compared
with the oracle run on the rounded fields (pcamm_model_fields) to the same bars as the float path.
(2) What the rounding costs against the float32 model, on the DESIGN.md workload recipe: the bars
SURVEY 8(f).4 names (w to 1e-3 ||w||, tumour to 0.05 mm).
"""
import numpy as np
import pytest

import oracle
from tests.gpu_util import to_dev
from tests.test_gpu_configs import _check, _setup

pytestmark = pytest.mark.gpu


def _models(cfg, frame_ids, **kw):
    import paper_1004_0014_b200 as pc
    wl, g, m32, frames, ys = _setup(cfg, frame_ids, **kw)
    m16 = pc.Model(nx=cfg.nx, ny=cfg.ny, nz=cfg.nz, hx=cfg.hx, hy=cfg.hy, hz=cfg.hz, K=cfg.K, nu=cfg.nu, nv=cfg.nv,
                   pu=cfg.pu, pv=cfg.pv, f0=to_dev(wl.f0), mean_dvf=to_dev(wl.model.mean), eig_dvf=to_dev(wl.model.eig),
                   landmarks_mm=wl.landmarks, sad=cfg.sad, sdd=cfg.sdd, field_storage=1, **kw)
    return wl, g, m32, m16, frames, ys


def test_stored_values_are_halves_times_a_power_of_two():
    from workloads.configs import small_config
    cfg = small_config("H0", 64, 64, 32, 6.0, 128, 96, 3.1)
    wl, g, m32, m16, frames, ys = _models(cfg, [5])
    mean, eig = (t.cpu().numpy() for t in m16.fields())
    mean32, eig32 = (t.cpu().numpy() for t in m32.fields())
    np.testing.assert_allclose(mean32, wl.model.mean, rtol=2e-7, atol=0)          # float storage: the inputs again
    np.testing.assert_allclose(eig32, wl.model.eig, rtol=2e-7, atol=0)
    assert np.array_equal(mean, mean32)                                           # x-bar is not rounded
    h = np.array([cfg.hx, cfg.hy, cfg.hz], np.float32)[None, :, None, None, None]
    v = eig.astype(np.float64) / h                                                # voxel units
    for k in range(cfg.K):
        mx = np.abs(wl.model.eig[k] / h[0]).max()
        s = 2.0 ** (14 - np.frexp(np.float32(mx))[1])
        q = v[k] * s
        assert np.abs(q).max() < 16384.5
        np.testing.assert_allclose(q, np.float16(q).astype(np.float64), rtol=3e-7, atol=0)   # representable in half
    # rounding to 11 significant bits: relative error of an entry <= 2^-11
    big = np.abs(wl.model.eig) > 1e-3 * np.abs(wl.model.eig).max()
    assert np.max(np.abs(eig[big] / wl.model.eig[big] - 1)) <= 2.0 ** -11 * 1.001


@pytest.mark.parametrize("K,hysteresis", [(3, False), (5, True)])
def test_parity_with_the_oracle_on_the_rounded_model(K, hysteresis):
    import paper_1004_0014_b200 as pc
    from workloads.configs import small_config
    cfg = small_config("H1", 64, 64, 64, 6.0, 128, 96, 3.1, K=K, hysteresis=hysteresis)
    wl, g, m32, m16, frames, ys = _models(cfg, [40, 41])
    mean, eig = (t.cpu().numpy() for t in m16.fields())
    wl.model.mean, wl.model.eig = mean, eig                 # the oracle gets the rounded model
    w0 = np.array([3.0, -2.0, 1.0, 0.5, -0.25][:K], np.float32)
    f_gpu = m16.warp(w0).cpu().numpy()
    f_ref = oracle.warp(g, wl.f0, mean, eig, w0)
    assert np.abs(f_gpu - f_ref).max() <= 2e-5 * np.abs(f_ref).max()
    J, grad, ab, _ = m16.eval(to_dev(ys[0]), frames[0].angle_rad, w0, 1.0, 0.0, want_proj=False)
    _, p_ref = oracle.evaluate(g, wl.f0, mean, eig, w0, frames[0].angle_rad)
    g_ref = oracle.gradient(g, wl.f0, mean, eig, w0, 1.0, 0.0, p_ref, ys[0], frames[0].angle_rad)
    assert np.linalg.norm(grad - g_ref) <= 1e-4 * np.linalg.norm(g_ref)
    opts = pc.Opts(max_iter=4)
    w = np.zeros(K, np.float32)
    for fr, y in zip(frames, ys):
        res = m16.reconstruct(to_dev(y), fr.angle_rad, w, opts, trace=True)
        _check(wl, g, res, y, fr.angle_rad, w, opts)
        w = res.w


def test_rounding_cost_against_the_float_model():
    """'re-validated against the 1e-4 / 1e-3 / 0.05 mm tolerances'."""
    import paper_1004_0014_b200 as pc
    from workloads.configs import small_config
    cfg = small_config("H2", 128, 128, 64, 3.0, 256, 192, 1.55)
    wl, g, m32, m16, frames, ys = _models(cfg, [100, 101, 102])
    opts = pc.Opts(max_iter=10)
    w32 = w16 = np.zeros(cfg.K, np.float32)
    for fr, y in zip(frames, ys):
        a = m32.reconstruct(to_dev(y), fr.angle_rad, w32, opts, trace=True)
        b = m16.reconstruct(to_dev(y), fr.angle_rad, w16, opts, trace=True)
        pa = m32.project(m32.warp(a.w), fr.angle_rad).cpu().numpy()
        pb = m16.project(m16.warp(a.w), fr.angle_rad).cpu().numpy()
        assert np.linalg.norm(pa - pb) <= 1e-4 * np.linalg.norm(pa)               # same w, the two models
        assert np.linalg.norm(a.w - b.w) <= 1e-3 * np.linalg.norm(a.w), (a.w, b.w)
        assert np.max(np.linalg.norm(a.landmarks - b.landmarks, axis=1)) <= 0.05
        assert abs(a.J - b.J) <= 1e-3 * a.J
        w32, w16 = a.w, b.w


def test_batched_and_fan_paths_and_errors():
    import paper_1004_0014_b200 as pc
    from workloads.configs import small_config
    cfg = small_config("H3", 64, 64, 32, 6.0, 128, 96, 3.1)
    wl, g, m32, m16, frames, ys = _models(cfg, [17, 111, 203], max_batch=3, max_candidates=8)
    opts = pc.Opts(max_iter=3)
    angles = np.array([fr.angle_rad for fr in frames], np.float32)
    w0 = np.zeros((3, cfg.K), np.float32)
    batch = m16.reconstruct_batch(to_dev(np.stack(ys)), angles, w0, opts)
    for b in range(3):
        one = m16.reconstruct(to_dev(ys[b]), float(angles[b]), w0[b], opts)
        assert np.linalg.norm(batch[b].w - one.w) <= 1e-5 * np.linalg.norm(one.w)
    fan = m16.reconstruct(to_dev(ys[0]), float(angles[0]), w0[0], pc.Opts(max_iter=3, batched_linesearch=1))
    seq = m16.reconstruct(to_dev(ys[0]), float(angles[0]), w0[0], opts)
    assert np.array_equal(fan.w, seq.w)
    z = to_dev(np.zeros((4, 4, 12), np.float32))
    with pytest.raises(pc.PcammError, match="multiple of 8"):
        pc.Model(nx=12, ny=4, nz=4, hx=1, hy=1, hz=1, K=1, nu=8, nv=8, pu=1, pv=1, f0=z,
                 mean_dvf=to_dev(np.zeros((3, 4, 4, 12), np.float32)), eig_dvf=to_dev(np.ones((1, 3, 4, 4, 12), np.float32)),
                 field_storage=1)
    with pytest.raises(pc.PcammError, match="field_storage"):
        pc.Model(nx=16, ny=4, nz=4, hx=1, hy=1, hz=1, K=1, nu=8, nv=8, pu=1, pv=1,
                 f0=to_dev(np.zeros((4, 4, 16), np.float32)), mean_dvf=to_dev(np.zeros((3, 4, 4, 16), np.float32)),
                 eig_dvf=to_dev(np.ones((1, 3, 4, 4, 16), np.float32)), field_storage=2)
