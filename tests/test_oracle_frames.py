"""Pins for the frame-stream part of the oracle (PAPER.md:L141 'initialized the PCA
coefficients to those at its previous frame', PAPER.md:L154 'use the predicted PCA coefficients from
previous histories to serve as the initial guess'; reading B9: polynomial of degree
`order` through the last order + 1 frames)."""
import numpy as np

import oracle
from tests.test_oracle_solve import _planted


def test_uniform_spacing_reduces_to_the_textbook_extrapolation_formulas():
    rng = np.random.default_rng(0)
    ws = rng.standard_normal((5, 3))
    ts = [0.0, 1.0, 2.0, 3.0, 4.0]
    np.testing.assert_allclose(oracle.predict_w(ts, ws, 5.0, 0), ws[-1], rtol=0, atol=0)
    np.testing.assert_allclose(oracle.predict_w(ts, ws, 5.0, 1), 2 * ws[-1] - ws[-2], rtol=1e-14, atol=1e-14)
    np.testing.assert_allclose(oracle.predict_w(ts, ws, 5.0, 2), 3 * ws[-1] - 3 * ws[-2] + ws[-3], rtol=1e-13,
                               atol=1e-13)


def test_exact_on_polynomials_with_uneven_time_stamps():
    """A predictor of order d reproduces any polynomial of degree <= d; numpy's polyfit through the
    same points is an independent route to the same number."""
    ts = [0.0, 0.21, 0.35, 0.61, 0.70]
    c = np.array([[0.3, -1.2, 2.0], [1.5, 0.4, -0.7], [-2.0, 0.9, 0.1]])      # w_k(t) = c0 + c1 t + c2 t^2
    for order in (0, 1, 2):
        cc = c.copy()
        cc[:, order + 1:] = 0.0
        ws = np.array([[np.polyval(row[::-1], t) for row in cc] for t in ts])
        t = 0.93
        want = np.array([np.polyval(row[::-1], t) for row in cc])
        np.testing.assert_allclose(oracle.predict_w(ts, ws, t, order), want, rtol=1e-12, atol=1e-12)
    rng = np.random.default_rng(3)
    ws = rng.standard_normal((5, 4))
    for order in (1, 2):
        m = order + 1
        fit = np.array([np.polyval(np.polyfit(ts[-m:], ws[-m:, k], order), 0.93) for k in range(4)])
        np.testing.assert_allclose(oracle.predict_w(ts, ws, 0.93, order), fit, rtol=1e-9, atol=1e-9)
    # a dropped or transposed factor would break the interpolation property at the nodes
    for i in (2, 3, 4):
        np.testing.assert_allclose(oracle.predict_w(ts, ws, ts[i], 2), ws[i], rtol=1e-12, atol=1e-12)


def test_short_history_and_degenerate_cases():
    w0 = np.array([0.5, -0.25])
    assert np.array_equal(oracle.predict_w([], np.zeros((0, 2)), 1.0, 2, w0), w0)          # first frame
    ws = np.array([[1.0, 2.0], [2.0, 0.0]])
    assert np.array_equal(oracle.predict_w([0.0], ws[:1], 1.0, 2, w0), ws[0])              # one frame: hold
    np.testing.assert_allclose(oracle.predict_w([0.0, 1.0], ws, 2.0, 2, w0), [3.0, -2.0])  # two frames: linear
    assert np.array_equal(oracle.predict_w([0.0, 1.0], ws, 2.0, -1, w0), w0)               # order < 0: always w0
    assert np.array_equal(oracle.predict_w([1.0, 1.0], ws, 2.0, 1, w0), ws[1])             # equal stamps: hold


def test_frame_loop_starts_each_solve_from_the_prediction():
    g, f0, xbar, u, scale, theta, y, w_star = _planted(noise=0.002, seed=5, n=(12, 10, 8), det=(16, 12))
    ys, thetas, times = [y, y, y], [theta, theta + 0.02, theta + 0.04], [0.0, 0.5, 1.0]
    opts = oracle.Opts(max_iter=2)
    for order in (0, 1):
        res = oracle.solve_frames(g, f0, xbar, u, ys, thetas, times, order, opts)
        assert np.array_equal(res[0]["w_init"], np.zeros(g.K, np.float32))
        w_a, w_b = (np.float32(r["w"]).astype(np.float64) for r in res[:2])
        assert np.array_equal(res[1]["w_init"], w_a.astype(np.float32))
        want = w_b if order == 0 else 2 * w_b - w_a
        np.testing.assert_allclose(res[2]["w_init"], want.astype(np.float32), rtol=1e-6, atol=0)
        # each frame is the plain solve from its w_init
        ref = oracle.solve(g, f0, xbar, u, ys[2], thetas[2], res[2]["w_init"], opts, want_volume=False)
        assert np.array_equal(ref["w"], res[2]["w"]) and ref["J"] == res[2]["J"]
