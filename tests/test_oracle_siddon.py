"""Pins for the oracle's projector P and its transpose (readings A3, A4, A21, A22).

P has a plain definition -- l_ij is the length of the source->pixel segment
inside voxel box j -- so it is pinned by brute force over every (ray, voxel)
pair, by closed-form chords, and by analytic ellipsoid line integrals.
"""
import numpy as np
import pytest

import oracle
from tests.util import box_chord, dense_system_matrix, geom, ray_endpoints, volume_box

ANGLES = [0.0, 0.3, np.pi / 4, np.pi / 2, 2.1, np.pi, 4.0, 5.5]


@pytest.mark.parametrize("theta", [0.0, 0.37, np.pi / 2, 2.5, 4.4])
def test_traversal_matches_brute_force(theta):
    g = geom(nx=5, ny=4, nz=3, h=(20.0, 25.0, 30.0), nu=9, nv=7, pitch=(14.0, 17.0),
             centre=(3.717, -1.129, 2.346))
    A = dense_system_matrix(g, theta)
    hits = 0
    for iv in range(g.nv):
        for iu in range(g.nu):
            ijk, ln, gap = oracle.traverse(g, theta, iu, iv)
            row = A[iv * g.nu + iu]
            lin = (ijk[:, 2] * g.ny + ijk[:, 1]) * g.nx + ijk[:, 0]
            assert len(set(lin.tolist())) == len(lin), "a voxel listed twice"
            dense = np.zeros(g.V)
            dense[lin] = ln
            np.testing.assert_allclose(dense, row, rtol=0, atol=1e-9)
            if gap > 1e-3:  # non-degenerate ray: the index sets agree exactly
                assert set(lin.tolist()) == set(np.nonzero(row > 1e-9)[0].tolist())
            hits += len(lin)
    assert hits > 100


@pytest.mark.parametrize("theta", ANGLES)
def test_uniform_volume_is_mu_times_box_chord(theta):
    g = geom(nx=13, ny=11, nz=9, h=(3.0, 2.0, 2.5), nu=21, nv=15, pitch=(2.0, 2.0), centre=(1.1, 0.7, -0.4))
    mu = 0.0173
    p = oracle.project(g, np.full(g.vshape, mu), theta)
    lo, hi, _ = volume_box(g)
    for iv in range(g.nv):
        for iu in range(g.nu):
            S, D = ray_endpoints(g, theta, iu, iv)
            assert abs(p[iv, iu] - mu * box_chord(S, D, lo, hi)) < 1e-12 * 100


def test_lengths_sum_to_box_chord():
    g = geom(nx=16, ny=12, nz=10, h=(2.0, 2.0, 3.0), nu=17, nv=13, pitch=(3.0, 3.0))
    lo, hi, _ = volume_box(g)
    for theta in ANGLES:
        for iu, iv in [(0, 0), (8, 6), (16, 12), (3, 11)]:
            _, ln, _ = oracle.traverse(g, theta, iu, iv)
            S, D = ray_endpoints(g, theta, iu, iv)
            # the reported list drops slivers shorter than 1e-6 min(h) (reading A22)
            assert abs(ln.sum() - box_chord(S, D, lo, hi)) < 1e-6 * 2.0 * 48


def test_voxel_aligned_cuboid():
    g = geom(nx=12, ny=10, nz=8, h=(2.0, 2.0, 2.0), nu=15, nv=11, pitch=(2.5, 2.5))
    f = np.zeros(g.vshape)
    f[2:6, 3:8, 4:10] = 0.5  # z 2..5, y 3..7, x 4..9
    lo, _, h = volume_box(g)
    blo = lo + np.array([4, 3, 2]) * h
    bhi = lo + np.array([10, 8, 6]) * h
    for theta in ANGLES:
        p = oracle.project(g, f, theta)
        for iv in range(g.nv):
            for iu in range(g.nu):
                S, D = ray_endpoints(g, theta, iu, iv)
                assert abs(p[iv, iu] - 0.5 * box_chord(S, D, blo, bhi)) < 1e-10


def test_central_ray_through_odd_volume_golden():
    """Closed form (tests/golden/central_ray.txt): at theta = 0 the central ray of an odd-sized
    detector runs along -x through the centre row of an odd-sized volume: nx voxels, length hx each."""
    g = geom(nx=5, ny=3, nz=3, h=(4.0, 4.0, 4.0), nu=5, nv=5, pitch=(2.0, 2.0))
    ijk, ln, _ = oracle.traverse(g, 0.0, 2, 2)
    import os
    rows = [l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "central_ray.txt"))
            if l.strip() and not l.startswith("#")]
    want_ijk = np.array([[int(v) for v in r[:3]] for r in rows])
    want_len = np.array([float(r[3]) for r in rows])
    assert np.array_equal(ijk, want_ijk)
    np.testing.assert_allclose(ln, want_len, rtol=0, atol=1e-12)


def test_ray_in_a_voxel_face_belongs_to_higher_index():
    """Reading A21: even-sized volume, the central ray lies in the planes y = 0 and z = 0."""
    g = geom(nx=4, ny=4, nz=4, h=(4.0, 4.0, 4.0), nu=5, nv=5, pitch=(2.0, 2.0))
    ijk, ln, _ = oracle.traverse(g, 0.0, 2, 2)
    assert np.array_equal(ijk, np.array([[3, 2, 2], [2, 2, 2], [1, 2, 2], [0, 2, 2]]))
    np.testing.assert_allclose(ln, 4.0, atol=1e-12)


def test_ray_missing_the_volume_is_zero():
    g = geom(nx=4, ny=4, nz=4, h=(1.0, 1.0, 1.0), nu=41, nv=3, pitch=(5.0, 5.0))
    p = oracle.project(g, np.ones(g.vshape), 0.7)
    assert p[:, 0].max() == 0.0 and p[:, -1].max() == 0.0 and p[1, 20] > 0


def _ellipsoid_chord(S, D, centre, semi):
    d = (D - S) / semi
    o = (S - centre) / semi
    a, b, c = d @ d, 2 * (o @ d), o @ o - 1.0
    disc = b * b - 4 * a * c
    if disc <= 0:
        return 0.0
    t0, t1 = (-b - np.sqrt(disc)) / (2 * a), (-b + np.sqrt(disc)) / (2 * a)
    return (min(t1, 1.0) - max(t0, 0.0)) * float(np.linalg.norm(D - S))


def test_analytic_ellipsoid_convergence():
    """north_star pin: voxelised uniform ellipsoid vs mu x analytic chord.  Agreement is limited by
    voxelisation, so the pin is the convergence: the error falls roughly in proportion to h."""
    centre, semi, mu = np.array([5.0, -3.0, 2.0]), np.array([40.0, 28.0, 33.0]), 0.02
    errs = []
    for n in (16, 32, 64):
        h = 128.0 / n
        g = geom(nx=n, ny=n, nz=n, h=(h, h, h), nu=32, nv=24, pitch=(4.0, 4.0))
        ax = (np.arange(n) - (n - 1) / 2.0) * h
        sub = (np.arange(4) + 0.5) / 4 - 0.5
        fine = (ax[:, None] + sub[None, :] * h).ravel()
        Z, Y, X = np.meshgrid(fine, fine, fine, indexing="ij", sparse=True)
        inside = (((X - centre[0]) / semi[0]) ** 2 + ((Y - centre[1]) / semi[1]) ** 2
                  + ((Z - centre[2]) / semi[2]) ** 2 <= 1.0).astype(np.float64)
        f = mu * inside.reshape(n, 4, n, 4, n, 4).mean(axis=(1, 3, 5))
        num = den = 0.0
        for theta in (0.2, 1.3, 2.9):
            p = oracle.project(g, f, theta)
            for iv in range(g.nv):
                for iu in range(g.nu):
                    S, D = ray_endpoints(g, theta, iu, iv)
                    want = mu * _ellipsoid_chord(S, D, centre, semi)
                    num += (p[iv, iu] - want) ** 2
                    den += want ** 2
        errs.append(np.sqrt(num / den))
    # measured rel-L2 over all rays (grazing rays included): 0.133, 0.056, 0.027 at h = 8, 4, 2 mm, i.e.
    # the per-ray error is about +-0.3 h mu at each of the two surface crossings.  Pin: first-order convergence.
    assert errs[0] < 0.2 and errs[1] < errs[0] / 1.6 and errs[2] < errs[1] / 1.6, errs


def test_adjoint_dense_transpose():
    g = geom(nx=4, ny=3, nz=3, h=(20.0, 25.0, 30.0), nu=6, nv=5, pitch=(15.0, 18.0), centre=(2.0, 1.0, -3.0))
    theta = 0.9
    A = dense_system_matrix(g, theta)
    rng = np.random.default_rng(0)
    f = rng.standard_normal(g.V)
    r = rng.standard_normal(g.nu * g.nv)
    np.testing.assert_allclose(oracle.project(g, f.reshape(g.vshape), theta).ravel(), A @ f, atol=1e-9)
    np.testing.assert_allclose(oracle.backproject(g, r, theta).ravel(), A.T @ r, atol=1e-9)


@pytest.mark.parametrize("threads", [1, 3])
def test_adjoint_dot_product(threads):
    g = geom(nx=24, ny=20, nz=16, h=(3.0, 3.0, 4.0), nu=40, nv=30, pitch=(2.5, 2.5), centre=(0.4, -0.3, 0.2))
    rng = np.random.default_rng(1)
    f = rng.standard_normal(g.vshape)
    r = rng.standard_normal(g.pshape)
    oracle.set_threads(threads)
    try:
        for theta in (0.1, 1.7, 3.9):
            lhs = float(np.sum(oracle.project(g, f, theta) * r))
            rhs = float(np.sum(f * oracle.backproject(g, r, theta)))
            assert abs(lhs - rhs) <= 1e-12 * max(abs(lhs), 1.0)
    finally:
        oracle.set_threads(1)
