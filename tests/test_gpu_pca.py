"""pcamm_pca_fit (Eq. 1; readings A12, B10) against the oracle's
PCA (SVD of the centred samples in float64) on the training DVFs of the DESIGN.md workload recipe and
on ragged synthetic samples.

Bars: eigenvalues to 1e-5 relative to the largest; mean to 2 float32 ulp of the
largest sample value; u_k to 2e-5 in relative L2 (float32 products summed over <= 128-element runs,
double above: rounding errors of random sign, so the scatter matrix is good to about 1e-7 sqrt(n) / n
of lambda_1, and an eigenvector moves by that error over its eigenvalue gap); training coefficients
to 2e-5 of sqrt(lambda_1).
"""
import numpy as np
import pytest

import oracle
from tests.gpu_util import to_dev

pytestmark = pytest.mark.gpu


def _compare(D, K, sign_ref=-1):
    import paper_1004_0014_b200 as pc
    D = np.ascontiguousarray(D, dtype=np.float32)
    N = D.shape[0]
    mean, eig, lam, coeffs = pc.pca_fit(to_dev(D), K, sign_ref)
    ref = oracle.pca_fit(D, K, None if sign_ref < 0 else sign_ref)
    np.testing.assert_allclose(lam, ref["eigenvalues"], rtol=0, atol=1e-5 * ref["eigenvalues"][0])
    np.testing.assert_allclose(mean.cpu().numpy(), ref["mean"], rtol=0, atol=2.4e-7 * np.abs(D).max())
    e = eig.cpu().numpy().astype(np.float64)
    for k in range(K):
        assert np.linalg.norm(e[k] - ref["eig"][k]) <= 2e-5, k            # unit-norm vectors
        assert abs(np.linalg.norm(e[k]) - 1.0) <= 1e-5
    np.testing.assert_allclose(coeffs[:N, :K], ref["coeffs"], rtol=0, atol=2e-5 * np.sqrt(ref["eigenvalues"][0]))
    return mean, eig, lam, coeffs, ref


def test_training_dvfs_of_the_workload_recipe():
    """Nine training phases, K = 3 on a 64 x 64 x 32 grid of the recipe; the model
    the harness feeds to both sides (workloads.pca, the same definition) comes out as well."""
    from workloads.build import build_workload
    from workloads.configs import small_config
    from workloads.motion import motion_spec, training_dvfs
    cfg = small_config("P1", 64, 64, 32, 6.0, 128, 96, 3.1)
    dvfs = np.asarray(training_dvfs(cfg, motion_spec(cfg)), dtype=np.float32)
    assert dvfs.shape == (9, 3, 32, 64, 64)
    mean, eig, lam, coeffs, ref = _compare(dvfs, 3)
    wl = build_workload(cfg)
    assert np.abs(mean.cpu().numpy() - wl.model.mean).max() <= 1e-5
    for k in range(3):
        assert np.linalg.norm(eig[k].cpu().numpy().astype(np.float64) - wl.model.eig[k]) <= 3e-5


@pytest.mark.parametrize("N,K,n", [(2, 1, 1001), (5, 4, 12345), (9, 3, 40000), (16, 8, 7777), (9, 8, 4 * 5003)])
def test_ragged_sizes_and_sample_counts(N, K, n):
    """Odd lengths take the scalar path, multiples of 4 the float4 path; several waves of blocks."""
    rng = np.random.default_rng(N * 100 + K)
    scale = np.linspace(3.0, 0.4, N)[:, None] * (1 + 0.3 * rng.standard_normal((N, 1)))
    D = rng.standard_normal((N, n)) * scale + 5.0 * rng.standard_normal((1, n))
    _compare(D, K, sign_ref=N - 1)


def test_large_sample_many_blocks():
    rng = np.random.default_rng(9)
    D = (rng.standard_normal((9, 3 * 128 * 128 * 16)) * np.linspace(2.0, 0.3, 9)[:, None]).astype(np.float32)
    _compare(D, 3)


def test_planted_model_and_errors():
    import paper_1004_0014_b200 as pc
    from tests.test_oracle_pca import _planted
    D, m, P, A = _planted(n=(3, 4, 6, 10))
    mean, eig, lam, coeffs, ref = _compare(D, 3, sign_ref=4)
    np.testing.assert_allclose(lam[:3], [49.0, 9.0, 2.25], rtol=2e-5)
    for k in range(3):
        np.testing.assert_allclose(eig[k].cpu().numpy(), np.sign(A[4, k]) * P[k], atol=3e-6)
    with pytest.raises(pc.PcammError) as e:                          # only 3 independent modes
        pc.pca_fit(to_dev(D.astype(np.float32)), 5)
    assert e.value.code == pc.E_SINGULAR
    with pytest.raises(pc.PcammError) as e:
        pc.pca_fit(to_dev(D.astype(np.float32)), 9)                   # K > N - 1
    assert e.value.code == pc.E_INVALID
    bad = D.astype(np.float32).copy()
    bad[3, 1, 2, 3, 4] = np.inf
    with pytest.raises(pc.PcammError) as e:
        pc.pca_fit(to_dev(bad), 3)
    assert e.value.code == pc.E_NONFINITE


def test_model_built_from_the_fitted_fields_solves_like_the_recipe_model():
    """The fitted fields go straight into pcamm_model_create: one solve with them against the
    oracle run on the same (GPU-fitted, float32) fields."""
    import paper_1004_0014_b200 as pc
    from tests.test_gpu_configs import _check
    from workloads.build import build_workload, ground_truth_volume
    from workloads.configs import small_config
    from workloads.motion import motion_spec, training_dvfs
    cfg = small_config("P2", 64, 64, 32, 6.0, 128, 96, 3.1)
    wl = build_workload(cfg)
    dvfs = np.asarray(training_dvfs(cfg, motion_spec(cfg)), dtype=np.float32)
    mean, eig, lam, coeffs = pc.pca_fit(to_dev(dvfs), cfg.K)
    m = pc.Model(nx=cfg.nx, ny=cfg.ny, nz=cfg.nz, hx=cfg.hx, hy=cfg.hy, hz=cfg.hz, K=cfg.K, nu=cfg.nu, nv=cfg.nv,
                 pu=cfg.pu, pv=cfg.pv, f0=to_dev(wl.f0), mean_dvf=mean, eig_dvf=eig, landmarks_mm=wl.landmarks,
                 sad=cfg.sad, sdd=cfg.sdd)
    g = oracle.Geometry(cfg.nx, cfg.ny, cfg.nz, cfg.hx, cfg.hy, cfg.hz, cfg.K, cfg.nu, cfg.nv, cfg.pu, cfg.pv,
                        cfg.sad, cfg.sdd)
    fr = wl.frames[77]
    y = oracle.project(g, ground_truth_volume(wl, fr), fr.angle_rad).astype(np.float32)
    opts = pc.Opts(max_iter=4)
    res = m.reconstruct(to_dev(y), fr.angle_rad, np.zeros(cfg.K, np.float32), opts, trace=True)
    wl.model.mean, wl.model.eig = mean.cpu().numpy(), eig.cpu().numpy()     # the oracle gets the same fields
    _check(wl, g, res, y, fr.angle_rad, np.zeros(cfg.K, np.float32), opts)
