"""Function-level parity of the CUDA path against the fp64 oracle (reading A16 level i), through
the C ABI.  Sizes span several 32-wide tiles with ragged tails in every dimension.

Tolerances (derived in DESIGN.md "Tolerances"): warp rel-L2 <= 5e-6 and bit-exact for an
identity DVF; projections rel-L2 <= 1e-4 (north_star); J rel <= 1e-4; gradient rel-L2 <= 1e-3;
(a, b) <= 1e-4; index sets of non-degenerate rays bit-exact; landmarks <= 0.05 mm.
"""
import numpy as np
import pytest

import oracle
from tests.gpu_util import make_model, rel_l2, to_dev, to_host
from tests.util import geom, smooth_model

pytestmark = pytest.mark.gpu

ANGLES = [0.0, 0.3, np.pi / 4, 0.9, np.pi / 2, 2.1, 3 * np.pi / 4, np.pi, 4.0, 5.5]


def _geom(K=3, n=(45, 38, 21), det=(70, 27), centre=(0.3717 * 3, 0.1129 * 3, 0.2346 * 3), h=(3.0, 3.0, 3.0),
          pitch=(3.2, 3.4)):
    return geom(nx=n[0], ny=n[1], nz=n[2], h=h, K=K, nu=det[0], nv=det[1], pitch=pitch, centre=centre)


def _model(g, seed=7, disp_vox=1.5):
    f0, xbar, u, scale = smooth_model(g, seed=seed, disp_vox=disp_vox)
    return f0, xbar, u, scale, make_model(g, f0, xbar, u)


# ------------------------------------------------------------------ a-1 warp

def test_identity_dvf_reproduces_f0_bit_exactly():
    g = _geom()
    rng = np.random.default_rng(0)
    f0 = rng.random(g.vshape).astype(np.float32)
    xbar = np.zeros((3,) + g.vshape, np.float32)
    u = rng.standard_normal((g.K, 3) + g.vshape).astype(np.float32)
    m = make_model(g, f0, xbar, u)
    out = to_host(m.warp(np.zeros(g.K)))
    assert np.array_equal(out, f0)


def test_integer_voxel_shift_is_exact():
    g = _geom(K=1)
    rng = np.random.default_rng(1)
    f0 = rng.random(g.vshape).astype(np.float32)
    xbar = np.zeros((3,) + g.vshape, np.float32)
    u = np.zeros((1, 3) + g.vshape, np.float32)
    u[0, 0], u[0, 1], u[0, 2] = 2 * g.hx, -1 * g.hy, 3 * g.hz     # w = 1: shift by (2, -1, 3) voxels
    m = make_model(g, f0, xbar, u)
    out = to_host(m.warp(np.array([1.0])))
    want = np.zeros_like(f0)
    want[:-3, 1:, :-2] = f0[3:, :-1, 2:]
    assert np.array_equal(out, want)
    np.testing.assert_array_equal(out, oracle.warp(g, f0, xbar, u, np.array([1.0])).astype(np.float32))


@pytest.mark.parametrize("K,seed", [(3, 7), (5, 8), (1, 9), (8, 10)])
def test_warp_matches_oracle(K, seed):
    g = _geom(K=K)
    f0, xbar, u, scale, m = _model(g, seed=seed, disp_vox=2.5)
    rng = np.random.default_rng(seed)
    for _ in range(2):
        w = rng.uniform(-1, 1, K) * scale
        ref = oracle.warp(g, f0, xbar, u, w.astype(np.float32))
        out = to_host(m.warp(w))
        assert rel_l2(out, ref) <= 5e-6
        assert np.max(np.abs(out - ref)) <= 2e-6 * np.max(np.abs(ref))


@pytest.mark.parametrize("K,seed", [(3, 21), (5, 22), (7, 23)])
def test_streaming_kernels_over_many_tiles_per_cta(K, seed):
    """A volume of 2048 field tiles: every persistent CTA of the TMA-fed warp and gradient kernels
    goes round its shared-memory stages several times (a 148-SM GPU gives each CTA ~14 tiles), so
    a stage handed to the wrong consumer group or polled a phase too early shows up here."""
    g = geom(nx=64, ny=256, nz=128 if K <= 4 else 64, h=(2.0, 2.0, 2.0), K=K, nu=48, nv=40, pitch=(6.0, 6.0))
    f0, xbar, u, scale, m = _model(g, seed=seed, disp_vox=2.0)
    rng = np.random.default_rng(seed)
    w = (rng.uniform(0.4, 1.0, K) * rng.choice([-1, 1], K) * scale).astype(np.float32)
    ref = oracle.warp(g, f0, xbar, u, w)
    out = to_host(m.warp(w))
    assert rel_l2(out, ref) <= 5e-6
    theta = 0.7
    _, p_ref = oracle.evaluate(g, f0, xbar, u, w, theta)
    y = (1.1 * p_ref + 0.02 * np.abs(p_ref).max() * rng.standard_normal(p_ref.shape)).astype(np.float32)
    J, grad, ab, p = m.eval(to_dev(y), theta, w, 1.0, 0.0)
    g_ref = oracle.gradient(g, f0, xbar, u, w, 1.0, 0.0, p_ref, y, theta)
    assert rel_l2(to_host(p), p_ref) <= 1e-5
    assert np.linalg.norm(grad - g_ref) <= 1e-3 * np.linalg.norm(g_ref), (grad, g_ref)


def test_warp_outside_the_grid_is_zero_padded():
    """Reading A2: a displacement larger than the volume samples zeros; one cell inside tapers."""
    g = _geom(K=1, n=(20, 18, 10))
    f0 = np.ones(g.vshape, np.float32)
    xbar = np.zeros((3,) + g.vshape, np.float32)
    u = np.zeros((1, 3) + g.vshape, np.float32)
    u[0, 0] = g.hx
    m = make_model(g, f0, xbar, u)
    assert np.all(to_host(m.warp(np.array([100.0]))) == 0)
    out = to_host(m.warp(np.array([0.25])))
    ref = oracle.warp(g, f0, xbar, u, np.array([0.25]))
    np.testing.assert_allclose(out, ref, rtol=0, atol=1e-7)
    assert abs(out[0, 0, -1] - 0.75) < 1e-7


# ------------------------------------------------------------------ a-2 projection

@pytest.mark.parametrize("theta", ANGLES)
def test_projection_matches_oracle(theta):
    g = _geom()
    rng = np.random.default_rng(3)
    f = rng.random(g.vshape).astype(np.float32)
    f0, xbar, u, scale, m = _model(g)
    ref = oracle.project(g, f, theta)
    out = to_host(m.project(to_dev(f), theta))
    assert ref.max() > 1.0
    assert rel_l2(out, ref) <= 1e-5          # north_star bar is 1e-4
    assert np.max(np.abs(out - ref)) <= 2e-5 * ref.max()


@pytest.mark.parametrize("theta", [0.0, 0.4, np.pi / 4, 1.2, np.pi / 2, 2.8, 4.1])
def test_projection_skips_air_exactly(theta):
    """The projector trims every 64-slab segment of a ray to the slabs whose voxel columns hold
    something non-zero (occupancy bytes written with the volume).  Volumes that are mostly air
    (an off-centre ellipsoid, a thin slab, a single voxel, nothing at all) long enough for several
    segments, both through pcamm_project (occupancy from the layout kernel) and through pcamm_eval
    (occupancy from the warp kernel)."""
    g = geom(nx=150, ny=140, nz=40, h=(2.0, 2.0, 2.0), K=2, nu=90, nv=36, pitch=(3.6, 3.1), centre=(0.7, 0.2, 0.5))
    rng = np.random.default_rng(5)
    zz, yy, xx = np.meshgrid(np.arange(g.nz), np.arange(g.ny), np.arange(g.nx), indexing="ij")
    blob = ((xx - 95) / 30.0) ** 2 + ((yy - 50) / 22.0) ** 2 + ((zz - 17) / 11.0) ** 2 <= 1.0
    slab = (np.abs(yy - 100) <= 1) & (zz >= 33)
    dot = (xx == 3) & (yy == 137) & (zz == 0)
    f0, xbar, u, scale, m = _model(g, seed=31, disp_vox=1.5)
    for mask in (blob, blob | slab | dot, dot, np.zeros_like(blob)):
        f = (rng.random(g.vshape) * mask).astype(np.float32)
        ref = oracle.project(g, f, theta)
        out = to_host(m.project(to_dev(f), theta))
        assert np.max(np.abs(out - ref)) <= 2e-5 * max(ref.max(), 1e-3)
        assert np.array_equal(out == 0, ref == 0) or np.max(np.abs(ref[out == 0])) <= 1e-6
    # the same through the warp kernel: the reference image is the masked volume
    m2 = make_model(g, (f0 * (blob | slab)).astype(np.float32), xbar, u)
    w = (0.6 * scale * np.array([1.0, -0.7])).astype(np.float32)
    _, p_ref = oracle.evaluate(g, (f0 * (blob | slab)).astype(np.float32), xbar, u, w, theta)
    _, _, _, p = m2.eval(to_dev(p_ref.astype(np.float32)), theta, w, 1.0, 0.0)
    assert rel_l2(to_host(p), p_ref) <= 1e-5


@pytest.mark.parametrize("aniso", [((2.0, 3.0, 2.5), (2.5, 2.0)), ((3.0, 2.0, 4.0), (2.0, 3.0))])
def test_projection_anisotropic_voxels_and_offsets(aniso):
    h, pitch = aniso
    g = geom(nx=37, ny=41, nz=19, h=h, K=2, nu=45, nv=22, pitch=pitch, centre=(1.3, -0.7, 0.9), off=(1.25, -0.5))
    rng = np.random.default_rng(4)
    f = rng.random(g.vshape).astype(np.float32)
    f0, xbar, u, scale, m = _model(g)
    for theta in (0.2, 0.8, 2.3, 3.9, 5.1):
        ref = oracle.project(g, f, theta)
        out = to_host(m.project(to_dev(f), theta))
        assert rel_l2(out, ref) <= 1e-5


def test_uniform_volume_gives_box_chords():
    """Closed form independent of the oracle: uniform mu => p_i = mu x chord of the ray through the
    volume's bounding box."""
    from tests.util import box_chord, ray_endpoints, volume_box
    g = _geom(n=(33, 31, 17), det=(40, 19))
    f0, xbar, u, scale, m = _model(g)
    mu = 0.0173
    f = np.full(g.vshape, mu, np.float32)
    lo, hi, _ = volume_box(g)
    for theta in (0.0, 0.7, np.pi / 2, 2.9):
        out = to_host(m.project(to_dev(f), theta))
        want = np.array([[np.float32(mu) * box_chord(*ray_endpoints(g, theta, iu, iv), lo, hi)
                          for iu in range(g.nu)] for iv in range(g.nv)])
        np.testing.assert_allclose(out, want, rtol=0, atol=3e-5 * want.max())


@pytest.mark.parametrize("theta", [0.0, 0.37, np.pi / 4, 1.3, np.pi / 2, 2.5, 4.4, 5.9])
def test_traversal_index_sets_are_bit_exact(theta):
    """north_star: bit-exact ray/voxel index sets.  Isocentre shifted by an irrational fraction of a
    voxel (reading A22); rays whose smallest crossing gap is < 1e-5 min(h) are degenerate and are
    compared on total length only (crossing positions are carried in 32.32 fixed point from a
    double-precision set-up, so the order of crossings is resolved far below that gap)."""
    g = _geom(n=(24, 20, 12), det=(30, 14), pitch=(4.0, 4.0))
    f0, xbar, u, scale, m = _model(g)
    n_deg = n_cmp = 0
    for iv in range(0, g.nv, 3):
        for iu in range(g.nu):
            ijk_o, len_o, gap = oracle.traverse(g, theta, iu, iv)
            ijk_g, len_g = m.traverse(theta, iu, iv)
            assert abs(len_g.sum() - len_o.sum()) <= 1e-4
            if gap < 1e-5 * min(g.hx, g.hy, g.hz):
                n_deg += 1
                continue
            n_cmp += 1
            assert np.array_equal(ijk_g, ijk_o), (iu, iv, ijk_g, ijk_o)
            np.testing.assert_allclose(len_g, len_o, rtol=0, atol=2e-4)
    assert n_cmp > 50 and n_deg <= 0.01 * (n_cmp + n_deg) + 1


def test_traversal_golden_central_ray():
    """tests/golden/central_ray.txt (closed form): the central ray at theta = 0 visits the five
    voxels of the middle row in descending x, 4 mm each."""
    import os
    g = geom(nx=5, ny=3, nz=3, h=(4.0, 4.0, 4.0), K=1, nu=5, nv=5, pitch=(2.0, 2.0))
    f0 = np.zeros(g.vshape, np.float32)
    m = make_model(g, f0, np.zeros((3,) + g.vshape, np.float32), np.zeros((1, 3) + g.vshape, np.float32))
    ijk, ln = m.traverse(0.0, 2, 2)
    gold = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "central_ray.txt"))
    assert np.array_equal(ijk, gold[:, :3].astype(np.int32))
    np.testing.assert_allclose(ln, gold[:, 3], atol=1e-5)


# ------------------------------------------------------------------ a-4 adjoint, gradient

@pytest.mark.parametrize("theta", [0.0, 0.5, np.pi / 4, 1.9, np.pi / 2, 3.6, 5.0])
def test_backprojection_is_the_transpose(theta):
    g = _geom()
    f0, xbar, u, scale, m = _model(g)
    rng = np.random.default_rng(5)
    f = rng.random(g.vshape).astype(np.float32)
    r = rng.standard_normal(g.pshape).astype(np.float32)
    Pf = to_host(m.project(to_dev(f), theta)).astype(np.float64)
    Ptr = to_host(m.backproject(to_dev(r), theta)).astype(np.float64)
    lhs, rhs = float(np.sum(Pf * r)), float(np.sum(f.astype(np.float64) * Ptr))
    scale_ = float(np.sqrt(np.sum(Pf * Pf) * np.sum(r.astype(np.float64) ** 2)))
    assert abs(lhs - rhs) <= 1e-5 * scale_
    ref = oracle.backproject(g, r, theta)
    assert rel_l2(Ptr, ref) <= 1e-4


@pytest.mark.parametrize("K,seed,theta", [(3, 11, 0.6), (5, 12, 2.2), (2, 13, 4.1), (3, 14, np.pi / 4), (8, 15, 1.1), (6, 16, 3.0)])
def test_eval_matches_oracle(K, seed, theta):
    g = _geom(K=K)
    f0, xbar, u, scale, m = _model(g, seed=seed, disp_vox=1.2)
    rng = np.random.default_rng(seed)
    w_star = rng.uniform(0.4, 1.0, K) * rng.choice([-1, 1], K) * scale
    _, p_star = oracle.evaluate(g, f0, xbar, u, w_star.astype(np.float32), theta)
    y = (1.7 * p_star + 0.05 + 0.003 * rng.standard_normal(p_star.shape)).astype(np.float32)
    w = (0.5 * w_star).astype(np.float32)
    a, b = np.float32(0.6), np.float32(-0.02)
    _, p_ref = oracle.evaluate(g, f0, xbar, u, w, theta)
    J_ref = oracle.cost(p_ref, y, float(a), float(b))
    g_ref = oracle.gradient(g, f0, xbar, u, w, float(a), float(b), p_ref, y, theta)
    _, a_ref, b_ref = oracle.lsfit(p_ref, y)
    J, grad, (af, bf), p = m.eval(to_dev(y), theta, w, float(a), float(b))
    assert rel_l2(to_host(p), p_ref) <= 1e-5
    assert abs(J - J_ref) <= 1e-4 * J_ref
    assert np.linalg.norm(grad - g_ref) <= 1e-3 * np.linalg.norm(g_ref), (grad, g_ref)
    assert abs(af - a_ref) <= 1e-4 * abs(a_ref) and abs(bf - b_ref) <= 1e-4 * max(abs(b_ref), abs(a_ref))


def test_gradient_matches_finite_differences_of_the_gpu_cost():
    """df/dx 'has to be consistent with the interpolation process'.  Central
    differences of the GPU's own J (double accumulators) agree with its analytic gradient."""
    g = _geom(K=3)
    f0, xbar, u, scale, m = _model(g, seed=21, disp_vox=1.0)
    rng = np.random.default_rng(21)
    theta = 1.1
    w_star = rng.uniform(0.4, 1.0, 3) * scale
    _, p_star = oracle.evaluate(g, f0, xbar, u, w_star.astype(np.float32), theta)
    y = to_dev(p_star.astype(np.float32))
    w = (0.37 * w_star).astype(np.float32)
    J, grad, _, _ = m.eval(y, theta, w, 1.0, 0.0, want_proj=False)
    for k in range(3):
        step = np.float32(2e-3 * scale)
        wp, wm = w.copy(), w.copy()
        wp[k] += step
        wm[k] -= step
        Jp = m.eval(y, theta, wp, 1.0, 0.0, want_proj=False)[0]
        Jm = m.eval(y, theta, wm, 1.0, 0.0, want_proj=False)[0]
        fd = (Jp - Jm) / float(np.float64(wp[k]) - np.float64(wm[k]))
        assert abs(fd - grad[k]) <= 2e-2 * np.linalg.norm(grad), (k, fd, grad)


# ------------------------------------------------------------------ a-6 localisation

def test_localisation_matches_oracle_and_closed_forms():
    g = _geom(K=3)
    f0, xbar, u, scale = smooth_model(g, seed=5, disp_vox=2.0)
    lm = np.array([[10.0, -8.0, 5.0], [-20.0, 12.0, -9.0], [0.0, 0.0, 0.0], [500.0, 0.0, 0.0]], np.float32)
    m = make_model(g, f0, xbar, u, landmarks=lm)
    rng = np.random.default_rng(5)
    w = (rng.uniform(-1, 1, 3) * scale).astype(np.float32)
    ref, _ = oracle.invert(g, xbar, u, w, lm)
    out = m.localise(w)
    assert np.max(np.linalg.norm(out - ref, axis=1)) <= 1e-4     # bar: 0.05 mm
    # constant DVF: r = r0 - c exactly
    xb = np.zeros((3,) + g.vshape, np.float32)
    uc = np.zeros((1, 3) + g.vshape, np.float32)
    uc[0, 0], uc[0, 1], uc[0, 2] = 0.5, -1.25, 2.0
    g1 = _geom(K=1)
    m1 = make_model(g1, f0, xb, uc, landmarks=lm[:2])
    np.testing.assert_allclose(m1.localise(np.array([2.0])), lm[:2] - 2.0 * np.array([0.5, -1.25, 2.0]), atol=1e-6)
    np.testing.assert_array_equal(m1.localise(np.array([0.0])), lm[:2])


@pytest.mark.parametrize("disp_vox", [0.4, 3.0, 9.0])
def test_tiles_that_cannot_contribute_are_skipped_exactly(disp_vox):
    """DESIGN.md reading B8, per tile: the warp kernel writes a tile as zeros without reading its
    fields when f0 is 0 on everything its stencils can reach, the gradient kernel does not visit a
    tile whose voxels can only land in constant cells.  Both rest on a bound of the displacement
    from the field maxima; a reference image that is a few small bodies in a lot of air, with
    displacements from a fraction of a voxel to well beyond a tile's neighbours, through grids
    with ragged tiles.  Where f0's support cannot reach, the result is exactly 0 on both sides."""
    g = geom(nx=136, ny=70, nz=75, h=(2.0, 2.0, 2.0), K=3, nu=96, nv=64, pitch=(3.4, 2.6), centre=(0.3, -0.4, 0.2))
    rng = np.random.default_rng(int(disp_vox * 10))
    zz, yy, xx = np.meshgrid(np.arange(g.nz), np.arange(g.ny), np.arange(g.nx), indexing="ij")
    body = ((xx - 100) / 14.0) ** 2 + ((yy - 20) / 9.0) ** 2 + ((zz - 50) / 12.0) ** 2 <= 1.0
    plate = (np.abs(xx - 30) <= 2) & (yy >= 50) & (zz <= 20)          # constant inside: gradient only at its faces
    dot = (xx == 70) & (yy == 35) & (zz == 37)
    f0, xbar, u, scale, _ = _model(g, seed=17, disp_vox=disp_vox)
    f0 = (np.where(body, 0.5 + f0, 0.0) + 0.7 * plate + 1.3 * dot).astype(np.float32)
    m = make_model(g, f0, xbar, u, tile_skipping=1)
    m_all = make_model(g, f0, xbar, u, tile_skipping=2)               # visits every tile
    theta = 0.9
    for wf in (0.0, 1.0, -1.7):
        w = (wf * scale * np.array([1.0, -0.6, 0.8])).astype(np.float32)
        f_ref = oracle.warp(g, f0, xbar, u, w)
        f_gpu = to_host(m.warp(w))
        assert np.array_equal(f_gpu, to_host(m_all.warp(w)))          # the shortcut changes no bit
        assert np.max(np.abs(f_gpu - f_ref)) <= 2e-5 * np.abs(f_ref).max()
        assert np.all(f_gpu[f_ref == 0] == 0)
        _, p_ref = oracle.evaluate(g, f0, xbar, u, w, theta)
        y = (p_ref * (1 + 0.05 * rng.standard_normal(p_ref.shape))).astype(np.float32)
        J, grad, ab, p = m.eval(to_dev(y), theta, w, 0.9, 0.01)
        assert rel_l2(to_host(p), p_ref) <= 1e-5
        g_ref = oracle.gradient(g, f0, xbar, u, w, 0.9, 0.01, p_ref, y, theta)
        assert np.linalg.norm(grad - g_ref) <= 1e-4 * np.linalg.norm(g_ref)
        J2, grad2, _, p2 = m_all.eval(to_dev(y), theta, w, 0.9, 0.01)
        assert J2 == J and np.array_equal(grad2, grad) and np.array_equal(to_host(p2), to_host(p))
    # nothing but air: every tile goes the short way
    m0 = make_model(g, np.zeros(g.vshape, np.float32), xbar, u)
    assert not to_host(m0.warp(w)).any()
