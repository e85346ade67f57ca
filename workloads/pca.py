"""PCA motion model from training DVFs (offline step; Eq. 1).

Snapshot method in float64: the mean is over the N-1 training DVFs (the zero
DVF of the reference phase is not a sample), eigen-decomposition of the
(N-1)x(N-1) Gram matrix of the centred DVFs, u_k = D~^T v_k / sqrt(lambda_k)
(unit L2 norm over all 3V entries).  Sign convention: u_k . (d_ref - mean) >= 0
for the DVF of the end-of-inhale phase (index ``sign_ref``); if that product
is zero the largest-magnitude entry is made positive.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass
class PCAModel:
    mean: np.ndarray         # float32 [3][nz][ny][nx]
    eig: np.ndarray          # float32 [K][3][nz][ny][nx], unit norm each
    eigenvalues: np.ndarray  # float64 [N-1], descending
    coeffs: np.ndarray       # float64 [N-1][K], training coefficients u_k . (d_i - mean)


def fit_pca(dvfs: np.ndarray, K: int, sign_ref: int | None = None) -> PCAModel:
    """dvfs: [n][3][nz][ny][nx] (any float dtype)."""
    n = dvfs.shape[0]
    field_shape = dvfs.shape[1:]
    D = dvfs.reshape(n, -1)
    mean = np.zeros(D.shape[1], dtype=np.float64)
    for i in range(n):
        mean += D[i]
    mean /= n
    # Gram matrix of centred samples, accumulated in float64 chunk by chunk
    G = np.zeros((n, n))
    chunk = 1 << 22
    for s in range(0, D.shape[1], chunk):
        C = D[:, s:s + chunk].astype(np.float64) - mean[None, s:s + chunk]
        G += C @ C.T
    lam, vec = np.linalg.eigh(G)
    order = np.argsort(lam)[::-1]
    lam, vec = lam[order], vec[:, order]
    eig = np.zeros((K, D.shape[1]), dtype=np.float64)
    for s in range(0, D.shape[1], chunk):
        C = D[:, s:s + chunk].astype(np.float64) - mean[None, s:s + chunk]
        eig[:, s:s + chunk] = (vec[:, :K] / np.sqrt(lam[:K])[None, :]).T @ C
    if sign_ref is None:
        sign_ref = n // 2  # phases 1..9 -> index 4 is t = 0.5, end of inhale
    ref = D[sign_ref].astype(np.float64) - mean
    for k in range(K):
        eig[k] /= np.linalg.norm(eig[k])
        d = float(eig[k] @ ref)
        if d < 0 or (d == 0 and eig[k][np.argmax(np.abs(eig[k]))] < 0):
            eig[k] = -eig[k]
    coeffs = np.stack([eig @ (D[i].astype(np.float64) - mean) for i in range(n)])
    return PCAModel(mean.astype(np.float32).reshape(field_shape),
                    eig.astype(np.float32).reshape((K,) + field_shape), lam, coeffs)
