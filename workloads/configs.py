"""The five workload configurations of BASELINE.json (`configs[0..4]` = C0..C4).

Shapes follow BASELINE.json; what the configs leave open (organ placement,
scaling between configs, DVF tapers) is fixed here and restated in DESIGN.md.
The paper's own workload (256x256x120 volume, 10 phases,
360 projections over one rotation, 1.5x test amplitude, 40x30 cm imager) is
what these stand in for.
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Tuple


@dataclass(frozen=True)
class Config:
    name: str
    # volume (x fastest), voxel size in mm
    nx: int
    ny: int
    nz: int
    hx: float
    hy: float
    hz: float
    K: int
    # flat detector (u fastest), pitch in mm
    nu: int
    nv: int
    pu: float
    pv: float
    sad: float = 1000.0
    sdd: float = 1500.0
    # phantom: config-0 coordinates are multiplied per axis by `scale`
    scale: Tuple[float, float, float] = (1.0, 1.0, 1.0)
    heart_and_ribs: bool = True
    # motion model
    n_phases: int = 10
    pert_rms_mm: float = 1.0
    hysteresis: bool = False
    # test trajectory
    n_proj: int = 360
    angle_step_deg: float = 1.0
    irregular: bool = False
    amplitude: float = 1.5
    # noise
    noise: str = "gaussian"  # "gaussian" (0.5% of max) or "poisson" (I0 = 1e5)
    # solver
    iterations: int = 10
    batched_linesearch: bool = False

    @property
    def V(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def npix(self) -> int:
        return self.nu * self.nv

    @property
    def h(self) -> Tuple[float, float, float]:
        return (self.hx, self.hy, self.hz)

    @property
    def shape_zyx(self) -> Tuple[int, int, int]:
        return (self.nz, self.ny, self.nx)

    def with_(self, **kw) -> "Config":
        return replace(self, **kw)


def _fov_scale(nx, ny, nz, hx, hy, hz):
    # half field of view per axis / 64 mm (C0's half field of view)
    return (nx * hx / 2.0 / 64.0, ny * hy / 2.0 / 64.0, nz * hz / 2.0 / 64.0)


_C0 = Config(
    name="C0", nx=32, ny=32, nz=32, hx=4.0, hy=4.0, hz=4.0, K=3,
    nu=64, nv=48, pu=2.0, pv=2.0, scale=(1.0, 1.0, 1.0), heart_and_ribs=False,
    pert_rms_mm=0.5, n_proj=8, angle_step_deg=45.0, iterations=30,
)
_C1 = Config(
    name="C1", nx=128, ny=128, nz=64, hx=3.0, hy=3.0, hz=3.0, K=3,
    nu=256, nv=192, pu=1.55, pv=1.55, scale=_fov_scale(128, 128, 64, 3.0, 3.0, 3.0),
)
_C2 = Config(
    name="C2", nx=256, ny=256, nz=128, hx=1.5, hy=1.5, hz=1.5, K=3,
    nu=512, nv=384, pu=0.776, pv=0.776, scale=_fov_scale(256, 256, 128, 1.5, 1.5, 1.5),
    irregular=True, noise="poisson",
)
_C3 = Config(
    name="C3", nx=256, ny=256, nz=256, hx=1.5, hy=1.5, hz=1.5, K=5,
    nu=512, nv=384, pu=0.776, pv=0.776, scale=_fov_scale(256, 256, 256, 1.5, 1.5, 1.5),
    hysteresis=True, batched_linesearch=True,
)
_C4 = Config(
    name="C4", nx=512, ny=512, nz=128, hx=0.98, hy=0.98, hz=0.98, K=3,
    nu=1024, nv=768, pu=0.388, pv=0.388, scale=_fov_scale(512, 512, 128, 0.98, 0.98, 0.98),
)

_ALL = {c.name: c for c in (_C0, _C1, _C2, _C3, _C4)}
CONFIG_NAMES = tuple(_ALL)


def get_config(name: str) -> Config:
    return _ALL[name]


def small_config(name: str, nx: int, ny: int, nz: int, h: float, nu: int, nv: int,
                 pitch: float, K: int = 3, **kw) -> Config:
    """A reduced configuration with the same recipe (used by parity tests that
    need several tiles and a ragged tail but must finish in seconds)."""
    return Config(name=name, nx=nx, ny=ny, nz=nz, hx=h, hy=h, hz=h, K=K, nu=nu, nv=nv,
                  pu=pitch, pv=pitch, scale=_fov_scale(nx, ny, nz, h, h, h), **kw)
