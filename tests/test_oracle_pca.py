"""Pins for the oracle's PCA motion model (section 2.1 Eq. 1;
DESIGN.md readings A12, B10)."""
import numpy as np

import oracle


def _planted(N=9, n=(3, 5, 6, 7), K=3, seed=0):
    """Samples m + sum_k a_ik p_k with orthonormal p_k and centred, mutually orthogonal coefficient
    columns of distinct size: the PCA is known in closed form (u_k = +-p_k, lambda_k = sum_i a_ik^2)."""
    rng = np.random.default_rng(seed)
    size = int(np.prod(n))
    P, _ = np.linalg.qr(rng.standard_normal((size, K)))
    A = rng.standard_normal((N, K))
    A -= A.mean(axis=0)
    A, _ = np.linalg.qr(A)                      # orthonormal, still centred (columns stay in 1-perp)
    A = A * np.array([7.0, 3.0, 1.5, 0.8, 0.4][:K])
    m = rng.standard_normal(size)
    D = m[None, :] + A @ P.T
    return D.reshape((N,) + n), m.reshape(n), P.T.reshape((K,) + n), A


def test_planted_low_rank_model_is_recovered():
    D, m, P, A = _planted()
    D32 = D.astype(np.float32)
    r = oracle.pca_fit(D32, 3, sign_ref=4)
    # against the closed form, to the float32 rounding of the samples
    np.testing.assert_allclose(r["mean"], m, atol=2e-6)
    np.testing.assert_allclose(r["eigenvalues"][:3], [49.0, 9.0, 2.25], rtol=1e-5)
    assert np.all(r["eigenvalues"][3:] < 1e-9)
    for k in range(3):
        s = np.sign(A[4, k])                   # the sign rule: positive coefficient of sample sign_ref
        np.testing.assert_allclose(r["eig"][k], s * P[k], atol=2e-6)
        np.testing.assert_allclose(r["coeffs"][:, k], s * A[:, k], atol=2e-5)
        assert r["coeffs"][4, k] > 0


def test_orthonormal_axes_and_best_rank_k_approximation():
    rng = np.random.default_rng(2)
    D = (rng.standard_normal((9, 3, 4, 5, 6)) * np.linspace(3, 0.5, 9)[:, None, None, None, None]).astype(np.float32)
    K = 4
    r = oracle.pca_fit(D, K)
    U = r["eig"].reshape(K, -1)
    np.testing.assert_allclose(U @ U.T, np.eye(K), atol=1e-12)
    X = D.reshape(9, -1).astype(np.float64) - r["mean"].reshape(-1)
    # Eckart-Young: the residual of the projection onto the K axes is the sum of the other eigenvalues
    resid = X - (X @ U.T) @ U
    np.testing.assert_allclose(np.sum(resid ** 2), np.sum(r["eigenvalues"][K:]), rtol=1e-10)
    np.testing.assert_allclose(np.sum(X ** 2), np.sum(r["eigenvalues"]), rtol=1e-12)
    # eigenvalues of the scatter matrix, by another library route
    np.testing.assert_allclose(np.sort(np.linalg.eigvalsh(X @ X.T))[::-1][:8], r["eigenvalues"][:8], rtol=1e-9)
    # u_k is an eigenvector of the scatter matrix X^T X
    for k in range(K):
        np.testing.assert_allclose(X.T @ (X @ U[k]), r["eigenvalues"][k] * U[k], atol=1e-9)
    np.testing.assert_allclose(r["coeffs"], X @ U.T, atol=1e-12)
    assert np.all(r["coeffs"][9 // 2] >= 0)


def test_against_scikit_learn_and_the_input_recipe():
    from sklearn.decomposition import PCA
    from workloads.pca import fit_pca
    rng = np.random.default_rng(5)
    D = (rng.standard_normal((7, 3, 6, 5, 4)) * np.linspace(2, 0.3, 7)[:, None, None, None, None]).astype(np.float32)
    r = oracle.pca_fit(D, 3)
    sk = PCA(n_components=3, svd_solver="full").fit(D.reshape(7, -1).astype(np.float64))
    np.testing.assert_allclose(sk.mean_, r["mean"].reshape(-1), atol=1e-12)
    np.testing.assert_allclose(sk.explained_variance_ * 6, r["eigenvalues"][:3], rtol=1e-10)
    for k in range(3):
        a, b = sk.components_[k], r["eig"][k].reshape(-1)
        np.testing.assert_allclose(a * np.sign(a @ b), b, atol=1e-10)
    w = fit_pca(D, 3)                          # the workload generator's snapshot-method PCA (same sign rule)
    np.testing.assert_allclose(w.eig.astype(np.float64), r["eig"], atol=2e-7)
    np.testing.assert_allclose(w.mean.astype(np.float64), r["mean"], atol=2e-7)
    np.testing.assert_allclose(w.eigenvalues[:6], r["eigenvalues"][:6], rtol=1e-9)
