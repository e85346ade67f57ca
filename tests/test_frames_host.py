"""The frame stream's predictor through the C ABI (pcamm_predict_w: host arithmetic, no device)
against the oracle's (oracle.predict_w, Lagrange form in float64).  PAPER.md:L141, L154; DESIGN.md
reading B9.  The library evaluates Newton's divided differences, so the two share no formula."""
import ctypes as C

import numpy as np
import pytest

import oracle
import paper_1004_0014_b200 as pc


@pytest.mark.parametrize("order", [-1, 0, 1, 2])
@pytest.mark.parametrize("n", [0, 1, 2, 3, 7])
def test_predictor_matches_the_oracle(order, n):
    rng = np.random.default_rng(100 * (order + 1) + n)
    K = 5
    ts = np.cumsum(rng.uniform(0.05, 0.3, n))
    ws = (40 * rng.standard_normal((n, K))).astype(np.float32)
    w0 = rng.standard_normal(K).astype(np.float32)
    t = (ts[-1] if n else 0.0) + 0.17
    got = pc.predict_w(order, ts, ws, t, w0, K=K)
    want = oracle.predict_w(list(ts), ws.astype(np.float64).reshape(n, K), t, order, w0)
    assert got.dtype == np.float32
    # the result is rounded once to float32; the double arithmetic before it differs by a few ulp of double
    np.testing.assert_allclose(got, want.astype(np.float32), rtol=2e-7, atol=1e-6)


def test_predictor_degenerate_inputs():
    ws = np.array([[1.0, 2.0], [2.0, 0.0]], np.float32)
    assert np.array_equal(pc.predict_w(1, [1.0, 1.0], ws, 2.0), ws[1])            # equal stamps: hold
    assert np.array_equal(pc.predict_w(2, [], np.zeros((0, 2), np.float32), 2.0, K=2), np.zeros(2, np.float32))
    out = np.zeros(2, np.float32)
    lib = pc.lib()
    assert lib.pcamm_predict_w(3, 2, 0, None, None, None, C.c_double(0.0), out.ctypes.data_as(C.c_void_p)) == pc.E_INVALID
    assert "order" in pc.last_error()
    assert lib.pcamm_predict_w(1, 2, 0, None, None, None, C.c_double(float("nan")),
                               out.ctypes.data_as(C.c_void_p)) == pc.E_INVALID
    assert lib.pcamm_predict_w(1, 99, 0, None, None, None, C.c_double(0.0), out.ctypes.data_as(C.c_void_p)) == pc.E_INVALID
    h = C.c_void_p()
    assert lib.pcamm_frames_create(None, 0, None, C.byref(h)) == pc.E_INVALID
    assert lib.pcamm_frames_count(None) == 0
    assert lib.pcamm_frames_reset(None) == pc.E_INVALID
    lib.pcamm_frames_destroy(None)
