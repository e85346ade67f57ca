"""Assemble the inputs of one configuration: reference volume, PCA model, landmarks, frames."""
from __future__ import annotations

from dataclasses import dataclass
from typing import List

import numpy as np

from .configs import Config
from .motion import Frame, MotionSpec, dvf_grid, motion_spec, test_trajectory, training_dvfs
from .pca import PCAModel, fit_pca
from .phantom import tumour_centre_mm, voxelise


@dataclass
class Workload:
    cfg: Config
    f0: np.ndarray            # float32 [nz][ny][nx]
    model: PCAModel
    spec: MotionSpec
    landmarks: np.ndarray     # float32 [M][3], mm (the tumour centre in the reference image)
    frames: List[Frame]


def build_workload(cfg: Config) -> Workload:
    spec = motion_spec(cfg)
    dvfs = training_dvfs(cfg, spec)
    model = fit_pca(dvfs, cfg.K)
    del dvfs
    f0 = voxelise(cfg).astype(np.float32)
    lm = tumour_centre_mm(cfg).astype(np.float32)[None, :]
    return Workload(cfg, f0, model, spec, lm, test_trajectory(cfg))


def ground_truth_volume(wl: Workload, frame: Frame) -> np.ndarray:
    """The phantom deformed by the test DVF of this frame: float32 [nz][ny][nx]."""
    x = dvf_grid(wl.cfg, wl.spec, frame.phase, frame.amplitude)
    return voxelise(wl.cfg, x).astype(np.float32)
