"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This package builds *inputs only*: analytic phantoms, training deformation
fields, the PCA motion model (offline step), test
trajectories and noise.  It holds none of the hot path's arithmetic (no warp,
no projector, no gradient, no line search): those live in ``oracle/`` (CPU
fp64 reference) and ``paper_1004_0014_b200/csrc`` (CUDA), which never import
each other.  Everything is deterministic from integer seeds and generated in
float64, then cast once to float32 so both sides consume identical arrays.
"""
from .configs import Config, get_config, CONFIG_NAMES  # noqa: F401
