"""Measurement noise on simulated line integrals (BASELINE.json configs).

gaussian: sigma = 0.5 % of max(y_true), rng(seed).
poisson : photon counts N ~ Poisson(I0 exp(-y_true)), I0 = 1e5, y = -ln(max(N, 1)/I0).
The paper's simulated projections carry no stated noise; these
models come from BASELINE.json only.
"""
from __future__ import annotations

import numpy as np

I0 = 1.0e5


def add_noise(y_true: np.ndarray, kind: str, seed: int = 0) -> np.ndarray:
    y = np.asarray(y_true, dtype=np.float64)
    rng = np.random.default_rng(seed)
    if kind == "none":
        out = y
    elif kind == "gaussian":
        out = y + rng.normal(0.0, 0.005 * float(y.max()), size=y.shape)
    elif kind == "poisson":
        counts = rng.poisson(I0 * np.exp(-y))
        out = -np.log(np.maximum(counts, 1) / I0)
    else:
        raise ValueError(kind)
    return out.astype(np.float32)
