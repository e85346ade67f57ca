"""Host-side harness checks: PCA on a known orthonormal basis (north_star pin; PAPER.md:L63-69,
reading A12), phantom recipe, test trajectory, determinism."""
import numpy as np

from workloads import get_config
from workloads.build import build_workload, ground_truth_volume
from workloads.configs import small_config
from workloads.motion import motion_spec, test_trajectory as make_trajectory, training_dvfs, true_tumour_position, dvf_at_points
from workloads.noise import add_noise
from workloads.pca import fit_pca
from workloads.phantom import mu_c0, voxelise, tumour_centre_mm
from workloads.planted import orthonormal_basis


def test_pca_recovers_known_basis_and_coefficients():
    shape = (6, 7, 8)
    K, n = 3, 9
    U = orthonormal_basis(shape, K + 1, seed=2)
    rng = np.random.default_rng(0)
    # coefficient matrix with distinct singular values and zero column means
    Q, _ = np.linalg.qr(rng.standard_normal((n, n)))
    W = Q[:, 1:K + 1] * np.array([40.0, 17.0, 5.0])[None, :]
    W -= W.mean(axis=0, keepdims=True)
    xbar = 3.0 * U[K]
    dvfs = xbar[None] + np.tensordot(W, U[:K], axes=(1, 0))
    m = fit_pca(dvfs, K, sign_ref=0)
    Uf = U[:K].reshape(K, -1)
    Em = m.eig.reshape(K, -1).astype(np.float64)
    # the float32 cast of the eigenvectors is the only loss
    assert np.linalg.norm(Em.T @ Em - Uf.T @ Uf) <= 1e-6
    np.testing.assert_allclose(m.mean.astype(np.float64), xbar, atol=1e-6)
    Wc = W.T @ W  # its eigenvectors give the rotation between W's columns and the principal axes
    lam, R = np.linalg.eigh(Wc)
    np.testing.assert_allclose(np.sort(lam)[::-1], m.eigenvalues[:K], rtol=1e-10)
    # coefficients reproduce the data: d_i = mean + sum_k c_ik u_k
    recon = m.mean.astype(np.float64)[None] + np.tensordot(m.coeffs, m.eig.astype(np.float64), axes=(1, 0))
    np.testing.assert_allclose(recon, dvfs, atol=2e-5)
    # sign convention: u_k . (d_ref - mean) >= 0
    ref = dvfs[0] - dvfs.mean(axis=0)
    assert all(np.sum(m.eig[k].astype(np.float64) * ref) >= 0 for k in range(K))


def test_pca_float64_subspace_is_exact():
    """Same recovery before the float32 cast: projector difference <= 1e-10 (SURVEY 8(c) PCA pin)."""
    shape = (5, 6, 7)
    K, n = 3, 9
    U = orthonormal_basis(shape, K, seed=5).reshape(K, -1)
    rng = np.random.default_rng(1)
    W = rng.standard_normal((n, K)) * np.array([30.0, 11.0, 4.0])
    W -= W.mean(axis=0, keepdims=True)
    D = W @ U
    mean = D.mean(axis=0)
    C = D - mean
    lam, vec = np.linalg.eigh(C @ C.T)
    E = (vec[:, ::-1][:, :K] / np.sqrt(lam[::-1][:K])).T @ C
    assert np.linalg.norm(E.T @ E - U.T @ U) <= 1e-10
    m = fit_pca(D.reshape((n, 3) + shape), K)
    np.testing.assert_allclose(np.abs(m.eig.reshape(K, -1).astype(np.float64) @ E.T), np.eye(K), atol=1e-6)


def test_phantom_structures_and_partial_volume():
    assert mu_c0(0, 0, 0, False) == 0.02          # mediastinum between the lungs
    assert mu_c0(28, 0, 0, False) == 0.004        # left lung
    assert mu_c0(-28, 0, 0, False) == 0.02        # tumour centred in the right lung
    assert mu_c0(-28, 0, 20, False) == 0.004
    assert mu_c0(6, 8, -15, True) == 0.021        # heart
    assert mu_c0(70, 0, 0, True) == 0.0
    cfg = get_config("C0")
    f0 = voxelise(cfg)
    assert f0.shape == (32, 32, 32) and f0.max() <= 0.02 + 1e-15 and f0.min() == 0.0
    frac = np.mean((f0 > 0) & (f0 < 0.02) & (np.abs(f0 - 0.004) > 1e-12))
    assert 0.02 < frac < 0.5  # partial-volume voxels exist
    for face in (f0[0], f0[-1], f0[:, 0], f0[:, -1], f0[:, :, 0], f0[:, :, -1]):
        assert face.max() == 0.0  # air at all faces (reading A2 is benign)
    # volume of the body ellipsoid is preserved by the 4x4x4 sub-sampling to ~0.1 %
    body = voxelise(cfg.with_(heart_and_ribs=False), sub=4)
    assert abs((body > 0).sum() * 64.0 / (4 / 3 * np.pi * 60 * 40 * 60) - 1) < 0.15


def test_c0_workload_shapes_rank_and_determinism():
    cfg = get_config("C0")
    wl = build_workload(cfg)
    assert wl.f0.dtype == np.float32 and wl.f0.shape == cfg.shape_zyx
    assert wl.model.mean.shape == (3,) + cfg.shape_zyx and wl.model.eig.shape == (3, 3) + cfg.shape_zyx
    for k in range(3):
        assert abs(np.linalg.norm(wl.model.eig[k].astype(np.float64)) - 1) < 1e-6
    lam = wl.model.eigenvalues
    assert lam[0] > 10 * lam[1] and lam[7] > 1e-3 * lam[1]   # rank 8 thanks to the perturbation (A20)
    wl2 = build_workload(cfg)
    assert np.array_equal(wl.f0, wl2.f0) and np.array_equal(wl.model.eig, wl2.model.eig)
    np.testing.assert_allclose(wl.landmarks, [[-28.0, 0.0, 0.0]])
    assert len(wl.frames) == 8 and abs(wl.frames[1].angle_rad - np.pi / 4) < 1e-12
    gt = ground_truth_volume(wl, wl.frames[4])
    assert gt.shape == wl.f0.shape and np.abs(gt - wl.f0).max() > 0.005


def test_training_dvf_recipe_values():
    cfg = get_config("C0")
    spec = motion_spec(cfg)
    d = training_dvfs(cfg.with_(pert_rms_mm=0.0), motion_spec(cfg.with_(pert_rms_mm=0.0)))
    assert d.shape == (9, 3, 32, 32, 32)
    # phase 5 (t = 0.5) is end of inhale: 8 mm SI at the diaphragm side (z <= -45), 0 at the apex
    assert abs(d[4, 2, 0, 16, 16] - 8.0) < 1e-6 and abs(d[4, 2, -1, 16, 16]) < 1e-6
    assert abs(d[4, 1, 16, -1, 16] - 2.0) < 1e-6 and abs(d[4, 0]).max() == 0.0
    # the perturbation has the requested rms
    pert = training_dvfs(cfg, spec)[2].astype(np.float64) - d[2]
    assert abs(np.sqrt(np.mean(np.sum(pert ** 2, axis=0))) - 0.5) < 1e-4


def test_trajectories():
    fr = make_trajectory(get_config("C1"))
    assert len(fr) == 360 and abs(fr[359].angle_rad - np.deg2rad(359)) < 1e-12
    assert abs(fr[24].phase) < 1e-9 and abs(fr[12].phase - 0.5) < 1e-9      # 24 projections per 4 s cycle
    assert all(f.amplitude == 1.5 for f in fr)
    ir = make_trajectory(get_config("C2"))
    amps = np.array([f.amplitude for f in ir])
    assert len(ir) == 360 and amps.min() >= 1.2 and amps.max() <= 1.8 and len(set(amps.round(9))) >= 12
    assert all(0 <= f.phase < 1 for f in ir)
    assert [f.phase for f in ir] == [f.phase for f in make_trajectory(get_config("C2"))]


def test_true_tumour_position_solves_the_pullback_equation():
    cfg = small_config("T", 24, 24, 16, 6.0, 32, 24, 4.0)
    spec = motion_spec(cfg)
    fr = make_trajectory(cfg.with_(n_proj=8, angle_step_deg=45.0))[3]
    r0 = tumour_centre_mm(cfg)
    r = true_tumour_position(cfg, spec, fr, r0)
    np.testing.assert_allclose(r + dvf_at_points(cfg, spec, fr.phase, fr.amplitude, r[None])[0], r0, atol=1e-9)
    assert np.linalg.norm(r - r0) > 1.0


def test_noise_models():
    y = np.linspace(0, 6, 1000).reshape(20, 50)
    g = add_noise(y, "gaussian", 0)
    assert g.dtype == np.float32 and abs(np.std(g - y) - 0.03) < 0.003
    assert np.array_equal(g, add_noise(y, "gaussian", 0))
    p = add_noise(y, "poisson", 0)
    assert np.all(np.isfinite(p)) and abs(np.mean(p[:, :10] - y[:, :10])) < 0.01


def test_bench_moved_bytes_model():
    """bench.py's bytes-moved model (the roofline numerators): with every tile loaded it equals SURVEY 8(a)'s
    dense algorithmic bytes, and a skipped tile saves its fields and its f0 gathers but not the warp
    kernel's store."""
    import bench
    cfg = get_config("C2")
    vox = 32 * 32
    n_tiles = cfg.V // vox
    dense = bench.algorithmic_bytes(cfg)
    full = bench.moved_bytes(cfg, 0, {"warp": n_tiles, "gradient": n_tiles}, vox)
    assert full["warp"] == dense["warp"] == 56 * cfg.V
    assert full["gradient"] == dense["gradient"] == 52 * cfg.V + 4 * cfg.npix
    half = bench.moved_bytes(cfg, 0, {"warp": n_tiles // 2, "gradient": n_tiles // 2}, vox)
    assert half["warp"] == 26 * cfg.V + 4 * cfg.V and half["gradient"] == 26 * cfg.V + 4 * cfg.npix
    assert bench.moved_bytes(cfg, 1, {"warp": n_tiles, "gradient": n_tiles}, vox)["warp"] == (12 + 18 + 8) * cfg.V


    # gradient records (one solve): the warp kernel writes them, the gradient gathers over the accepted slot's
    rec = bench.moved_bytes(cfg, 0, {"warp": n_tiles, "gradient": 0}, vox, {"written": 2000.0, "gathered": 1000.0}, n_tiles)
    assert rec["warp"] == 56 * cfg.V + 48 * 2000 + 32 * n_tiles
    assert rec["gradient"] == (48 + 12 * cfg.K) * 1000 + 32 * n_tiles + 4 * cfg.npix
