"""pcamm_fit_cost_static: the entry point that allocates nothing (its scratch is a static device array,
csrc/noalloc.cu) against the existing path (pcamm_eval on a model, whose scratch is cudaMalloc'ed):
the intensity fit of Eq. 4 and the cost of Eq. 2 for the same (p, y), on two calls in a row, then a
third that repeats the first (the array keeps the previous call's contents: nothing of it may leak).

Collected last on purpose (the suite runs with pytest -x).  Bars as in tests/test_gpu_functions.py:
a, b and J within 1e-4 relative (both sides sum in double: they agree far closer than that).
"""
import ctypes as C

import numpy as np
import pytest

import paper_1004_0014_b200 as pc


def test_sizes_beyond_the_static_array_are_rejected_before_any_cuda_call():
    """No GPU needed: the size check comes before the first CUDA call (the pointers are never used)."""
    lib = pc.lib()
    dummy = C.c_void_p(256)
    for n in (0, -5, pc.STATIC_MAX_PIXELS + 1, 1 << 40):
        rc = lib.pcamm_fit_cost_static(dummy, dummy, C.c_int64(n), dummy, None)
        assert rc == -1                                               # PCAMM_E_INVALID
        assert "PCAMM_STATIC_MAX_PIXELS" in pc.last_error()
    assert lib.pcamm_fit_cost_static(None, dummy, C.c_int64(16), dummy, None) == -1
    assert "NULL" in pc.last_error()


@pytest.mark.gpu
def test_static_scratch_entry_point_matches_the_model_path_on_calls_in_a_row():
    import torch
    import oracle
    from tests.gpu_util import make_model, to_dev
    from tests.util import geom, smooth_model

    g = geom(nx=96, ny=70, nz=64, h=(2.0, 2.0, 2.0), K=3, nu=96, nv=64, pitch=(3.4, 2.6))
    f0, xbar, u, scale = smooth_model(g, seed=5, disp_vox=1.0)
    m = make_model(g, f0, xbar, u)
    rng = np.random.default_rng(17)
    cases = []
    for i, theta in enumerate((0.9, 2.4)):
        w = (0.4 * scale * rng.uniform(-1, 1, 3)).astype(np.float32)
        _, p_true = oracle.evaluate(g, f0, xbar, u, 1.3 * w, theta)
        y = to_dev((p_true * (0.8 + 0.1 * i) * (1 + 0.05 * rng.standard_normal(p_true.shape)) + 0.03 * (i + 1)).astype(np.float32))
        # the existing path: pcamm_eval gives p and the fit; a second evaluation gives J at that fit
        _, _, (af, bf), p = m.eval(y, theta, w, 1.0, 0.0)
        J_ref = m.eval(y, theta, w, af, bf, want_proj=False)[0]
        cases.append((p.contiguous(), y, af, bf, J_ref))

    out = torch.empty(8, dtype=torch.float64, device="cuda")          # the caller's output, allocated once
    results = []
    for p, y, af, bf, J_ref in cases + cases[:1]:                     # two calls in a row, then the first again
        got = pc.fit_cost_static(p, y, out=out).cpu().numpy().copy()
        results.append(got)
        a, b, J, Sp, Sy, Syy, Syp, status = got
        assert status == 0
        assert abs(a - af) <= 1e-4 * abs(af) and abs(b - bf) <= 1e-4 * max(abs(bf), abs(af))
        assert abs(J - J_ref) <= 1e-4 * J_ref
        # and the definitions (oracle: Eq. 4 and Eq. 2 in double on the same float32 inputs)
        ph, y32 = p.cpu().numpy().astype(np.float64), y.cpu().numpy()
        yh = y32.astype(np.float64)
        _, a_o, b_o = oracle.lsfit(ph, y32)
        assert abs(a - a_o) <= 1e-9 * abs(a_o) and abs(b - b_o) <= 1e-9 * max(abs(b_o), abs(a_o))
        assert abs(J - oracle.cost(ph, y32, a, b)) <= 1e-9 * J
        assert abs(Sp - ph.sum()) <= 1e-9 * abs(ph.sum()) and abs(Syp - (ph * yh).sum()) <= 1e-9 * (ph * yh).sum()
        assert abs(Sy - yh.sum()) <= 1e-9 * abs(yh.sum()) and abs(Syy - (yh * yh).sum()) <= 1e-9 * (yh * yh).sum()
    assert not np.array_equal(results[0], results[1])                 # different inputs, different results
    assert np.array_equal(results[0], results[2])                     # same inputs: the same bits, whatever ran between

    # ragged sizes: one pixel, one short of / one past a block's 4096 pixels, several blocks and a tail
    for n in (1, 4095, 4097, 3 * 4096 + 77):
        pv = torch.from_numpy(rng.random(n).astype(np.float32)).cuda()
        yv = torch.from_numpy(rng.random(n).astype(np.float32)).cuda()
        a, b, J, Sp, Sy, Syy, Syp, status = pc.fit_cost_static(pv, yv, out=out).cpu().numpy()
        ph, y32 = pv.cpu().numpy().astype(np.float64), yv.cpu().numpy()
        if n == 1:
            assert status == -5 and a == 0 and b == 0                 # PCAMM_E_SINGULAR: y is constant
            continue
        _, a_o, b_o = oracle.lsfit(ph, y32)
        assert status == 0 and abs(a - a_o) <= 1e-9 * max(abs(a_o), 1) and abs(b - b_o) <= 1e-9 * max(abs(b_o), 1)
        assert abs(J - oracle.cost(ph, y32, a, b)) <= 1e-9 * max(J, 1e-30)

    # beyond the static array: a clear error, nothing launched
    big = torch.zeros(pc.STATIC_MAX_PIXELS + 1, dtype=torch.float32, device="cuda")
    with pytest.raises(pc.PcammError, match="PCAMM_STATIC_MAX_PIXELS"):
        pc.fit_cost_static(big, big, out=out)
    del big
    ramp = torch.arange(pc.STATIC_MAX_PIXELS, dtype=torch.float32, device="cuda") / pc.STATIC_MAX_PIXELS
    a, b, J, *_, status = pc.fit_cost_static(2 * ramp + 0.25, ramp, out=out).cpu().numpy()       # the largest size it takes
    assert status == 0 and abs(a - 2) <= 1e-6 and abs(b - 0.25) <= 1e-6 and J <= 1e-6 * pc.STATIC_MAX_PIXELS
