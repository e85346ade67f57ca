"""The measurement hooks of the C ABI (they feed bench.py's roofline block and the timeline under
profiles/): the tile counters of the two streaming kernels, the in-kernel timeline, the timing hooks
over several candidate slots, the tuning knobs.  No parity claims here; what is checked is that the
numbers mean what bench.py takes them to mean.
"""
import numpy as np
import pytest

import oracle
from tests.gpu_util import make_model, to_dev
from tests.util import geom, smooth_model

pytestmark = pytest.mark.gpu


_FIELDS = []          # (f0, xbar, u) of the last _setup, for the oracle


def _setup(tile_skipping=1, **kw):
    g = geom(nx=96, ny=70, nz=64, h=(2.0, 2.0, 2.0), K=3, nu=96, nv=64, pitch=(3.4, 2.6))
    f0, xbar, u, scale = smooth_model(g, seed=5, disp_vox=1.0)
    zz, yy, xx = np.meshgrid(np.arange(g.nz), np.arange(g.ny), np.arange(g.nx), indexing="ij")
    body = ((xx - 60) / 20.0) ** 2 + ((yy - 30) / 14.0) ** 2 + ((zz - 30) / 18.0) ** 2 <= 1.0
    f0 = np.where(body, 0.5 + f0, 0.0).astype(np.float32)            # a body in a lot of air: tiles to skip
    m = make_model(g, f0, xbar, u, tile_skipping=tile_skipping, **kw)
    _FIELDS.append((f0, xbar, u))
    w = (0.4 * scale * np.array([1.0, -0.6, 0.8])).astype(np.float32)
    _, p = oracle.evaluate(g, f0, xbar, u, w, 0.9)
    return g, m, w, to_dev(p.astype(np.float32))


def test_tile_counters_count_the_tiles_the_timed_launches_loaded():
    import paper_1004_0014_b200 as pc
    # default: the warp kernel leaves gradient records, the gradient of one solve gathers over them
    g, m, w, y = _setup(tile_skipping=1)
    m.eval(y, 0.9, w, 1.0, 0.0, want_proj=False)
    m.tile_counts(reset=True)
    m.time_kernel(0, 5)
    warp_tiles, grad_tiles, total, vox, gathered, written = m.tile_counts(reset=True)
    assert vox == 32 * 32 and total == 3 * g.ny * 2
    assert grad_tiles == 0 and gathered == 0 and warp_tiles % 5 == 0 and 0 < warp_tiles // 5 < total
    assert written % 5 == 0 and 0 < written // 5 < g.V
    m.time_kernel(2, 4)
    warp_tiles, grad_tiles, _, _, gathered, w2 = m.tile_counts(reset=True)
    assert warp_tiles == 0 and grad_tiles == 0 and w2 == 0
    assert gathered == 4 * (written // 5)                       # the records of the accepted slot, all of them
    # the number of records is the number of voxels with G_j != 0 (oracle: the warped volume's gradient)
    # (float against double: a voxel whose G cancels to zero in one of the two is counted differently)
    Gf = oracle.warp_grad(g, *_FIELDS[-1], w)
    n_ref = int(np.count_nonzero(np.any(np.asarray(Gf).reshape(3, -1) != 0, axis=0)))
    assert abs(written // 5 - n_ref) <= 0.002 * n_ref and n_ref < 0.5 * g.V
    try:
        pc.tune("grad_records", 0)                              # the gradient streams the fields itself
        g, m, w, y = _setup(tile_skipping=1)
        m.eval(y, 0.9, w, 1.0, 0.0, want_proj=False)
        m.tile_counts(reset=True)
        m.time_kernel(0, 5)
        warp_tiles, grad_tiles, total, vox, gathered, written = m.tile_counts(reset=True)
        assert grad_tiles == 0 and written == 0 and warp_tiles % 5 == 0 and 0 < warp_tiles // 5 < total
        m.time_kernel(2, 4)
        warp_tiles, grad_tiles, _, _, gathered, _ = m.tile_counts(reset=True)
        assert warp_tiles == 0 and gathered == 0 and grad_tiles % 4 == 0 and 0 < grad_tiles // 4 < total
        # with skipping off every tile is loaded
        g2, m2, w2, y2 = _setup(tile_skipping=2)
        m2.eval(y2, 0.9, w2, 1.0, 0.0, want_proj=False)
        m2.tile_counts(reset=True)
        m2.time_kernel(0, 3)
        m2.time_kernel(2, 3)
        a, b, total2 = m2.tile_counts()[:3]
        assert a == 3 * total2 and b == 3 * total2
    finally:
        pc.tune("grad_records", 1)


def test_gradient_from_records_and_streamed_gradient_agree():
    """pcamm_tune("grad_records"): the same a-4 either from the records the warp kernel left or by a pass of
    its own over the fields; the sums differ in order only."""
    import paper_1004_0014_b200 as pc
    g, m, w, y = _setup(max_candidates=2)
    J1, g1, fit1, _ = m.eval(y, 0.9, 0.7 * w, 0.95, 0.01)
    r1 = m.reconstruct(y, 0.9, np.zeros(3, np.float32), pc.Opts(max_iter=5), trace=True)
    f1 = m.reconstruct(y, 0.9, np.zeros(3, np.float32), pc.Opts(max_iter=5, batched_linesearch=2), trace=True)
    try:
        pc.tune("grad_records", 0)
        g, m0, w, y = _setup()
        J0, g0, fit0, _ = m0.eval(y, 0.9, 0.7 * w, 0.95, 0.01)
        r0 = m0.reconstruct(y, 0.9, np.zeros(3, np.float32), pc.Opts(max_iter=5), trace=True)
    finally:
        pc.tune("grad_records", 1)
    assert J1 == J0 and fit1 == fit0
    assert np.linalg.norm(g1 - g0) <= 1e-5 * np.linalg.norm(g0)
    assert np.array_equal(r1.backtracks, r0.backtracks) and np.array_equal(f1.backtracks, r0.backtracks)
    assert np.linalg.norm(r1.w - r0.w) <= 1e-4 * np.linalg.norm(r0.w)
    assert np.array_equal(f1.w, r1.w)                           # reading B7 holds with the records too


def test_timing_over_two_candidate_slots():
    """pcamm_time_slots: the warp and projection timings then run over two candidates per launch; the fields
    are still loaded once per tile."""
    g, m, w, y = _setup(max_candidates=2)
    m.eval(y, 0.9, w, 1.0, 0.0, want_proj=False)
    m.tile_counts(reset=True)
    m.time_kernel(0, 4)
    one = m.tile_counts(reset=True)[0]
    m.time_slots(np.stack([w, 1.05 * w]))
    t_warp, t_proj = m.time_kernel(0, 4), m.time_kernel(1, 4)
    two = m.tile_counts(reset=True)[0]
    assert t_warp > 0 and t_proj > 0
    assert one > 0 and two >= one                  # the same tiles (a few more where the larger w reaches further)
    assert two <= 1.2 * one
    with pytest.raises(Exception):
        m.time_slots(np.stack([w, w, w]))          # more slots than the model has


def test_timeline_lists_the_kernels_of_a_solve_in_order():
    import paper_1004_0014_b200 as pc
    pc.tune("timeline", 1)
    try:
        g, m, w, y = _setup(landmarks=np.array([[5.0, -4.0, 3.0]], np.float32))
    finally:
        pc.tune("timeline", 0)
    res = m.reconstruct(y, 0.9, np.zeros(3, np.float32), pc.Opts(max_iter=3), trace=True)
    kind, t0, t1 = m.timeline()
    names = ("ysums", "begin", "view", "warp", "project", "ctl_proj", "resid", "grad", "ctl_grad", "-", "final", "invert")
    seq = [names[k] for k in kind]
    assert seq[:6] == ["ysums", "begin", "view", "warp", "project", "ctl_proj"]
    assert seq[-3:] == ["resid", "final", "invert"]
    body = seq[6:-3]
    assert len(body) % 6 == 0 and len(body) // 6 >= res.iters
    for i in range(0, len(body), 6):
        assert body[i:i + 6] == ["resid", "grad", "ctl_grad", "warp", "project", "ctl_proj"]
    assert np.all(t1 >= t0) and np.all(t0[1:] >= t1[:-1])          # one after the other
    assert pc.launch_count() >= len(kind)
    # a model created without the knob has no timeline
    g2, m2, _, _ = _setup()
    with pytest.raises(pc.PcammError):
        m2.timeline()


def test_unknown_knob_is_an_error():
    import paper_1004_0014_b200 as pc
    with pytest.raises(pc.PcammError):
        pc.tune("no_such_knob", 1)


def test_projector_knobs_change_the_launch_not_the_result():
    import paper_1004_0014_b200 as pc
    g, m, w, y = _setup()
    _, _, _, p_ref = m.eval(y, 0.9, w, 1.0, 0.0)
    p_ref = p_ref.cpu().numpy()
    try:
        for sc, cps in ((2, 1), (1, 3), (4, 2)):
            pc.tune("project_scan_slabs", sc)
            pc.tune("project_chunks_per_segment", cps)
            g2, m2, _, _ = _setup()
            p = m2.eval(y, 0.9, w, 1.0, 0.0)[3].cpu().numpy()
            assert np.max(np.abs(p - p_ref)) <= 2e-6 * np.max(np.abs(p_ref))
    finally:
        pc.tune("project_scan_slabs", 0)
        pc.tune("project_chunks_per_segment", 0)


def test_solves_in_flight_from_records_and_from_the_streamed_gradient_agree():
    """Several solves in flight take their gradients from the records as well (one gather over the solves):
    against the streamed kernel, which sums in another order, and against the same solves one at a time."""
    import torch
    import paper_1004_0014_b200 as pc
    g, m, w, y0 = _setup(max_batch=3, max_candidates=2)
    f0, xbar, u = _FIELDS[-1]
    thetas = np.array([0.9, 2.3, 4.0], np.float32)
    ys = []
    for i, th in enumerate(thetas):
        _, p = oracle.evaluate(g, f0, xbar, u, (0.6 + 0.3 * i) * w, float(th))
        ys.append(p.astype(np.float32))
    yd = to_dev(np.stack(ys))
    w0 = np.zeros((3, 3), np.float32)
    for fan in (1, 2):
        opts = pc.Opts(max_iter=4, batched_linesearch=fan if fan > 1 else 0)
        rec = m.reconstruct_batch(yd, thetas, w0, opts, trace=True)
        assert m.tile_counts(reset=True)[4] > 0                      # records were gathered
        one = [m.reconstruct(yd[b], float(thetas[b]), w0[b], opts, trace=True) for b in range(3)]
        try:
            pc.tune("grad_records", 0)
            g2, m0, _, _ = _setup(max_batch=3, max_candidates=2)
            ref = m0.reconstruct_batch(yd, thetas, w0, opts, trace=True)
            assert m0.tile_counts(reset=True)[4] == 0
        finally:
            pc.tune("grad_records", 1)
        for b in range(3):
            assert np.array_equal(rec[b].backtracks, ref[b].backtracks) and rec[b].iters == ref[b].iters
            assert np.linalg.norm(rec[b].w - ref[b].w) <= 1e-4 * np.linalg.norm(ref[b].w)
            assert abs(rec[b].J - ref[b].J) <= 1e-5 * ref[b].J
            # in flight or alone: the same gather in the same order, the same bits
            assert np.array_equal(rec[b].w, one[b].w) and rec[b].J == one[b].J


def test_graph_knobs_change_the_launch_not_the_result():
    """pcamm_tune("pdl") and ("static_passes"): the same kernels in the same order with the same memory effects,
    so a solve gives the same bits whatever the edges of its graph are and wherever its while-loop starts."""
    import paper_1004_0014_b200 as pc
    g, m, w, y = _setup(max_candidates=2)
    opts = pc.Opts(max_iter=5, batched_linesearch=2)
    ref = m.reconstruct(y, 0.9, np.zeros(3, np.float32), opts, trace=True)
    try:
        for knob, value in (("pdl", 0), ("static_passes", 0), ("static_passes", 3), ("static_passes", 9)):
            pc.tune(knob, value)
            g2, m2, _, _ = _setup(max_candidates=2)
            r = m2.reconstruct(y, 0.9, np.zeros(3, np.float32), opts, trace=True)
            assert r.iters == ref.iters and np.array_equal(r.backtracks, ref.backtracks)
            assert np.array_equal(r.w, ref.w) and r.J == ref.J and r.a == ref.a and r.b == ref.b
            pc.tune("pdl", 1)
            pc.tune("static_passes", -1)
    finally:
        pc.tune("pdl", 1)
        pc.tune("static_passes", -1)


def test_passes_behind_the_end_of_a_solve_do_nothing():
    """A solve that stops early (here: it starts at the minimiser of a noise-free problem, so its first line
    searches find no decreasing step) leaves the passes laid out in front of the loop with nothing to do: the
    result is that of a graph without them, bit for bit, and the launch count says they ran."""
    import paper_1004_0014_b200 as pc
    g, m, w, y = _setup(max_candidates=2)               # y = P f(w), noise-free
    opts = pc.Opts(max_iter=8, batched_linesearch=2)
    pc.launch_count(reset=True)
    res = m.reconstruct(y, 0.9, w, opts, trace=True)
    assert res.iters < 8 and res.status == 3            # PCAMM_S_LINESEARCH
    n_auto = pc.launch_count(reset=True)
    try:
        pc.tune("static_passes", 0)
        g2, m2, _, _ = _setup(max_candidates=2)
        pc.launch_count(reset=True)
        ref = m2.reconstruct(y, 0.9, w, opts, trace=True)
        n_loop = pc.launch_count(reset=True)
    finally:
        pc.tune("static_passes", -1)
    assert ref.iters == res.iters and ref.status == res.status and np.array_equal(ref.backtracks, res.backtracks)
    assert np.array_equal(ref.w, res.w) and ref.J == res.J and ref.a == res.a and ref.b == res.b
    assert np.array_equal(ref.landmarks, res.landmarks) if res.landmarks is not None else True
    assert n_auto > n_loop                              # the idle passes were launched (and counted)


def test_model_on_a_second_device():
    """The opt-in to large dynamic shared memory is per device."""
    import torch
    import paper_1004_0014_b200 as pc
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two visible GPUs")
    g, m, w, y = _setup()
    with torch.cuda.device(1):
        f0, xbar, u, scale = smooth_model(g, seed=5, disp_vox=1.0)
        t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to("cuda:1")
        m1 = pc.Model(nx=g.nx, ny=g.ny, nz=g.nz, hx=g.hx, hy=g.hy, hz=g.hz, K=g.K, nu=g.nu, nv=g.nv, pu=g.pu, pv=g.pv,
                      f0=t(f0), mean_dvf=t(xbar), eig_dvf=t(u), sad=g.sad, sdd=g.sdd)
        out = m1.warp(w)
        assert out.device.index == 1
