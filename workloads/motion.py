"""Training deformation fields and the test breathing trajectory.

Stands in for the demons-registered NCAT phases of PAPER.md:L59, L115 (10
phases, reference = phase 0, nine pull-back DVFs) and for the 360-projection
test rotation of PAPER.md:L117 (4 s breathing, 1.5x amplitude, 6 Hz).  All
displacements are pull-back, in millimetres: f(r) = f0(r + x(r)).

Recipe (config-0 coordinates are scaled per axis by cfg.scale; amplitudes in mm
are not scaled), phase t_i = i/10, s(t) = (1 - cos 2 pi t)/2:

  SI:  x_z = 8 s(t) tau(z),  tau = clamp((z_apex - z)/(z_apex - z_dia), 0, 1),
       z_apex = +45, z_dia = -45
  AP:  x_y = 2 s(t) clamp((y + 40)/80, 0, 1);  with hysteresis (C3) the AP time
       course is s(t - 0.1) - s(-0.1)
  plus a smooth per-phase perturbation: white Gaussian noise, rng(1000 + i), on
  a 5 mm lattice covering the field of view (+1 cell), Gaussian-filtered with
  sigma = 10 mm, trilinearly interpolated, rescaled so the rms vector length
  over the voxel grid is cfg.pert_rms_mm.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List

import numpy as np
from scipy import ndimage, optimize

from .configs import Config
from .phantom import grid_axes

LATTICE_MM = 5.0
SIGMA_MM = 10.0
Z_APEX, Z_DIA = 45.0, -45.0
SI_PEAK_MM, AP_PEAK_MM = 8.0, 2.0


def s_breath(t):
    return 0.5 * (1.0 - np.cos(2.0 * np.pi * np.asarray(t, dtype=np.float64)))


def _lattice_axes(cfg: Config):
    axes = []
    for n, h in ((cfg.nx, cfg.hx), (cfg.ny, cfg.hy), (cfg.nz, cfg.hz)):
        half = n * h / 2.0 + LATTICE_MM
        m = int(np.ceil(2.0 * half / LATTICE_MM)) + 1
        axes.append(-half + LATTICE_MM * np.arange(m))
    return axes  # x, y, z


def _interp_matrix(src: np.ndarray, dst: np.ndarray) -> np.ndarray:
    """Dense (len(dst) x len(src)) linear-interpolation matrix, clamped at the ends."""
    t = np.clip((dst - src[0]) / (src[1] - src[0]), 0.0, len(src) - 1.0)
    i0 = np.minimum(np.floor(t).astype(np.int64), len(src) - 2)
    w = t - i0
    M = np.zeros((len(dst), len(src)))
    M[np.arange(len(dst)), i0] = 1.0 - w
    M[np.arange(len(dst)), i0 + 1] += w
    return M


@dataclass
class MotionSpec:
    """Perturbation lattices of the nine non-reference phases, already scaled to mm."""
    cfg: Config
    lattices: List[np.ndarray]  # index 0 = phase 0 (zeros), each [3][mz][my][mx]

    def lattice_at_phase(self, phi: float) -> np.ndarray:
        """Perturbation lattice linearly interpolated in phase, periodic, zero at phase 0."""
        n = self.cfg.n_phases
        p = (phi % 1.0) * n
        i0 = int(np.floor(p)) % n
        i1 = (i0 + 1) % n
        w = p - np.floor(p)
        return (1.0 - w) * self.lattices[i0] + w * self.lattices[i1]


def lattice_to_grid(cfg: Config, lat: np.ndarray) -> np.ndarray:
    """Trilinear interpolation of a lattice field at the voxel centres: [3][nz][ny][nx]."""
    lx, ly, lz = _lattice_axes(cfg)
    xs, ys, zs = grid_axes(cfg)
    Mx, My, Mz = _interp_matrix(lx, xs), _interp_matrix(ly, ys), _interp_matrix(lz, zs)
    out = np.empty((3, cfg.nz, cfg.ny, cfg.nx))
    for c in range(3):
        a = np.tensordot(Mz, lat[c], axes=(1, 0))          # [nz][my][mx]
        a = np.tensordot(a, My, axes=(1, 1))               # [nz][mx][ny]
        a = np.tensordot(a, Mx, axes=(1, 1))               # [nz][ny][nx]
        out[c] = a
    return out


def lattice_at_points(cfg: Config, lat: np.ndarray, pts: np.ndarray) -> np.ndarray:
    """Same interpolant evaluated at arbitrary points [n][3] (mm) -> [n][3]."""
    lx, ly, lz = _lattice_axes(cfg)
    pts = np.atleast_2d(np.asarray(pts, dtype=np.float64))
    coords = np.stack([
        np.clip((pts[:, 2] - lz[0]) / LATTICE_MM, 0, len(lz) - 1),
        np.clip((pts[:, 1] - ly[0]) / LATTICE_MM, 0, len(ly) - 1),
        np.clip((pts[:, 0] - lx[0]) / LATTICE_MM, 0, len(lx) - 1),
    ])
    return np.stack([ndimage.map_coordinates(lat[c], coords, order=1, mode="nearest")
                     for c in range(3)], axis=1)


def motion_spec(cfg: Config) -> MotionSpec:
    lx, ly, lz = _lattice_axes(cfg)
    shape = (3, len(lz), len(ly), len(lx))
    lattices = [np.zeros(shape)]
    sig = SIGMA_MM / LATTICE_MM
    for i in range(1, cfg.n_phases):
        rng = np.random.default_rng(1000 + i)
        lat = rng.standard_normal(shape)
        for c in range(3):
            lat[c] = ndimage.gaussian_filter(lat[c], sigma=sig, mode="nearest")
        g = lattice_to_grid(cfg, lat)
        rms = np.sqrt(np.mean(np.sum(g * g, axis=0)))
        lattices.append(lat * (cfg.pert_rms_mm / rms))
    return MotionSpec(cfg, lattices)


def _time_courses(cfg: Config, phi: float):
    s_si = float(s_breath(phi))
    s_ap = float(s_breath(phi - 0.1) - s_breath(-0.1)) if cfg.hysteresis else s_si
    return s_si, s_ap


def sinusoid_at(cfg: Config, x, y, z, phi: float):
    """Analytic SI + AP part at world points (mm); returns (dx, dy, dz)."""
    sx, sy, sz = cfg.scale
    s_si, s_ap = _time_courses(cfg, phi)
    z0 = np.asarray(z, dtype=np.float64) / sz
    y0 = np.asarray(y, dtype=np.float64) / sy
    tau = np.clip((Z_APEX - z0) / (Z_APEX - Z_DIA), 0.0, 1.0)
    dz = SI_PEAK_MM * s_si * tau
    dy = AP_PEAK_MM * s_ap * np.clip((y0 + 40.0) / 80.0, 0.0, 1.0)
    return np.zeros(np.broadcast(x, dy, dz).shape), dy + 0 * dz, dz + 0 * dy


def dvf_grid(cfg: Config, spec: MotionSpec, phi: float, amplitude: float = 1.0) -> np.ndarray:
    """Pull-back DVF on the voxel grid at breathing phase phi: float64 [3][nz][ny][nx]."""
    xs, ys, zs = grid_axes(cfg)
    Z, Y, X = np.meshgrid(zs, ys, xs, indexing="ij")
    dx, dy, dz = sinusoid_at(cfg, X, Y, Z, phi)
    out = lattice_to_grid(cfg, spec.lattice_at_phase(phi))
    out[0] += dx
    out[1] += dy
    out[2] += dz
    return amplitude * out


def dvf_at_points(cfg: Config, spec: MotionSpec, phi: float, amplitude: float, pts) -> np.ndarray:
    pts = np.atleast_2d(np.asarray(pts, dtype=np.float64))
    dx, dy, dz = sinusoid_at(cfg, pts[:, 0], pts[:, 1], pts[:, 2], phi)
    return amplitude * (np.stack([dx, dy, dz], axis=1)
                        + lattice_at_points(cfg, spec.lattice_at_phase(phi), pts))


def training_dvfs(cfg: Config, spec: MotionSpec) -> np.ndarray:
    """The N-1 = 9 training DVFs (phases 1..9) as float32 [9][3][nz][ny][nx]."""
    out = np.empty((cfg.n_phases - 1, 3, cfg.nz, cfg.ny, cfg.nx), dtype=np.float32)
    for i in range(1, cfg.n_phases):
        out[i - 1] = dvf_grid(cfg, spec, i / cfg.n_phases)
    return out


@dataclass(frozen=True)
class Frame:
    index: int
    time_s: float
    angle_rad: float
    phase: float
    amplitude: float


def test_trajectory(cfg: Config) -> List[Frame]:
    """The test rotation: projection i at i/6 s and i * angle_step."""
    n = cfg.n_proj
    if n == 8:  # C0: 8 angles 45 deg apart, phases spread evenly over one cycle
        return [Frame(i, i * 0.5, np.deg2rad(i * cfg.angle_step_deg), i / 8.0, cfg.amplitude)
                for i in range(n)]
    times = np.arange(n) / 6.0
    if not cfg.irregular:
        return [Frame(i, float(t), np.deg2rad(i * cfg.angle_step_deg), float((t / 4.0) % 1.0),
                      cfg.amplitude) for i, t in enumerate(times)]
    rng = np.random.default_rng(2)
    starts, periods, amps = [0.0], [], []
    while starts[-1] <= times[-1]:
        T = rng.uniform(3.0, 5.0)
        periods.append(T)
        amps.append(cfg.amplitude * (1.0 + rng.uniform(-0.2, 0.2)))
        starts.append(starts[-1] + T)
    frames = []
    for i, t in enumerate(times):
        c = int(np.searchsorted(starts, t, side="right") - 1)
        frames.append(Frame(i, float(t), np.deg2rad(i * cfg.angle_step_deg),
                            float((t - starts[c]) / periods[c]), float(amps[c])))
    return frames


test_trajectory.__test__ = False  # not a pytest test


def true_tumour_position(cfg: Config, spec: MotionSpec, frame: Frame, r0_mm) -> np.ndarray:
    """Ground-truth tumour centre: the point r with r + x_test(r) = r0, by a generic
    root finder on the analytic field (accuracy context, not a parity value)."""
    r0 = np.asarray(r0_mm, dtype=np.float64)

    def fun(r):
        return r + dvf_at_points(cfg, spec, frame.phase, frame.amplitude, r[None, :])[0] - r0

    sol = optimize.root(fun, r0, tol=1e-12)
    return sol.x
