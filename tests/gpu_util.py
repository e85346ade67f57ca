"""Helpers of the `-m gpu` parity tests: build a CUDA model from the same float32 arrays the oracle
consumes.  Imports of torch / the CUDA package happen inside the functions so that collecting the
tests on a CPU box does not need a GPU."""
from __future__ import annotations

import numpy as np

import oracle


def make_model(g: oracle.Geometry, f0, xbar, u, landmarks=None, max_batch=1, max_candidates=1, tile_skipping=1,
               projector=0, ray_step_vox=0.0):
    # tile_skipping=1: the parity grids are too small for the library's default to turn the tile flags on
    import torch
    import paper_1004_0014_b200 as pc
    dev = torch.device("cuda:0")
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(dev)
    return pc.Model(nx=g.nx, ny=g.ny, nz=g.nz, hx=g.hx, hy=g.hy, hz=g.hz, K=g.K, nu=g.nu, nv=g.nv, pu=g.pu,
                    pv=g.pv, f0=t(f0), mean_dvf=t(xbar), eig_dvf=t(u), landmarks_mm=landmarks, sad=g.sad,
                    sdd=g.sdd, off_u=g.off_u, off_v=g.off_v, cx=g.cx, cy=g.cy, cz=g.cz, max_batch=max_batch,
                    max_candidates=max_candidates, tile_skipping=tile_skipping, projector=projector,
                    ray_step_vox=ray_step_vox)


def to_dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to("cuda:0")


def to_host(t) -> np.ndarray:
    return t.detach().cpu().numpy()


def rel_l2(a, b) -> float:
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def oracle_opts(o) -> oracle.Opts:
    """The oracle's options for a paper_1004_0014_b200.Opts."""
    return oracle.Opts(max_iter=o.max_iter, grad_tol=o.grad_tol, armijo_c=o.armijo_c, armijo_beta=o.armijo_beta,
                       max_backtracks=o.max_backtracks, init_step_vox=o.init_step_vox,
                       batched_linesearch=o.batched_linesearch, inv_max_iter=o.inv_max_iter,
                       inv_tol_mm=o.inv_tol_mm)
