"""The frame stream (pcamm_frames_*; reading B9) on
the GPU against the oracle: consecutive projections 1 degree and 1/6 s apart on the DESIGN.md
workload recipe, each solve started from the coefficients predicted from the frames before it.

Parity is teacher-forced per frame: the oracle predicts from the history the library holds (the
GPU path's previous results, which are its to hold) and solves the frame from that start; starts
are compared as float32 values, results to the bars of tests/test_gpu_configs.py.
"""
import numpy as np
import pytest

import oracle
from tests.gpu_util import oracle_opts, to_dev
from tests.test_gpu_configs import _check, _setup

pytestmark = pytest.mark.gpu


def _cfg():
    from workloads.configs import small_config
    return small_config("F1", 64, 64, 32, 6.0, 128, 96, 3.1)


@pytest.mark.parametrize("order", [0, 1, 2])
def test_frames_follow_the_oracle(order):
    import paper_1004_0014_b200 as pc
    cfg = _cfg()
    ids = [30, 31, 32, 33, 34]
    wl, g, m, frames, ys = _setup(cfg, ids)
    opts = pc.Opts(max_iter=4)
    fs = pc.Frames(m, order=order)
    hist_t, hist_w = [], []
    for fr, y in zip(frames, ys):
        want_init = oracle.predict_w(hist_t, np.array(hist_w, dtype=np.float64).reshape(len(hist_w), cfg.K),
                                     fr.time_s, order, np.zeros(cfg.K)).astype(np.float32)
        peek = fs.predict(fr.time_s)
        res = fs.push(to_dev(y), fr.angle_rad, fr.time_s, opts, trace=True)
        assert np.array_equal(peek, res.w_init)
        np.testing.assert_allclose(res.w_init, want_init, rtol=3e-7, atol=1e-6)
        _check(wl, g, res, y, fr.angle_rad, res.w_init, opts)
        hist_t.append(fr.time_s)
        hist_w.append(res.w.astype(np.float64))
    assert fs.count() == 3
    fs.reset()
    assert fs.count() == 0 and np.array_equal(fs.predict(9.0), np.zeros(cfg.K, np.float32))


def test_frames_equal_explicit_warm_starts_and_host_y():
    """Order 0 is PAPER.md:L141: the same numbers as calling reconstruct with the previous w by hand,
    with y in device or in host memory."""
    import paper_1004_0014_b200 as pc
    cfg = _cfg()
    wl, g, m, frames, ys = _setup(cfg, [50, 51, 52])
    opts = pc.Opts(max_iter=3)
    fs, fh = pc.Frames(m, order=0), pc.Frames(m, order=0)
    w = np.zeros(cfg.K, np.float32)
    for fr, y in zip(frames, ys):
        ref = m.reconstruct(to_dev(y), fr.angle_rad, w, opts)
        a = fs.push(to_dev(y), fr.angle_rad, fr.time_s, opts)
        b = fh.push(np.ascontiguousarray(y, dtype=np.float32), fr.angle_rad, fr.time_s, opts, host_y=True)
        assert np.array_equal(a.w, ref.w) and np.array_equal(b.w, ref.w) and a.J == ref.J == b.J
        assert np.array_equal(a.landmarks, ref.landmarks)
        w = ref.w


def test_frames_errors_leave_the_history_alone():
    import paper_1004_0014_b200 as pc
    cfg = _cfg()
    wl, g, m, frames, ys = _setup(cfg, [10, 11])
    fs = pc.Frames(m, order=1, w0=np.full(cfg.K, 0.5, np.float32))
    assert np.array_equal(fs.predict(0.0), np.full(cfg.K, 0.5, np.float32))
    r0 = fs.push(to_dev(ys[0]), frames[0].angle_rad, 1.0, pc.Opts(max_iter=2))
    with pytest.raises(pc.PcammError, match="decrease"):
        fs.push(to_dev(ys[1]), frames[1].angle_rad, 0.5, pc.Opts(max_iter=2))
    bad = ys[1].copy()
    bad[3, 5] = np.nan
    with pytest.raises(pc.PcammError):
        fs.push(to_dev(bad), frames[1].angle_rad, 2.0, pc.Opts(max_iter=2))
    assert fs.count() == 1 and np.array_equal(fs.predict(2.0), r0.w)
    with pytest.raises(pc.PcammError, match="order"):
        pc.Frames(m, order=3)


def test_fixed_angle_sequence():
    """fixed-angle geometry (fluoroscopy) is the same call with a constant angle."""
    import paper_1004_0014_b200 as pc
    from workloads.build import ground_truth_volume
    cfg = _cfg()
    wl, g, m, frames, _ = _setup(cfg, [20, 23, 26])
    theta = 0.3
    ys = [oracle.project(g, ground_truth_volume(wl, fr), theta).astype(np.float32) for fr in frames]
    opts = pc.Opts(max_iter=3)
    fs = pc.Frames(m, order=1)
    for fr, y in zip(frames, ys):
        res = fs.push(to_dev(y), theta, fr.time_s, opts, trace=True)
        _check(wl, g, res, y, theta, res.w_init, opts)
