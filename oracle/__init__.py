"""ctypes wrapper around the CPU oracle (oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package; the product
(paper_1004_0014_b200) never does.  All results are float64.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

from .build import build as _build


class _Geom(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("hx", C.c_double), ("hy", C.c_double), ("hz", C.c_double),
                ("cx", C.c_double), ("cy", C.c_double), ("cz", C.c_double),
                ("K", C.c_int32), ("nu", C.c_int32), ("nv", C.c_int32),
                ("pu", C.c_double), ("pv", C.c_double), ("sad", C.c_double), ("sdd", C.c_double),
                ("off_u", C.c_double), ("off_v", C.c_double)]


class _Opts(C.Structure):
    _fields_ = [("max_iter", C.c_int32), ("grad_tol", C.c_double), ("armijo_c", C.c_double),
                ("armijo_beta", C.c_double), ("max_backtracks", C.c_int32),
                ("init_step_vox", C.c_double), ("batched_linesearch", C.c_int32),
                ("inv_max_iter", C.c_int32), ("inv_tol_mm", C.c_double)]


class _Result(C.Structure):
    _fields_ = [("iters", C.c_int32), ("status", C.c_int32), ("J0", C.c_double), ("J", C.c_double),
                ("a", C.c_double), ("b", C.c_double)]


@dataclass(frozen=True)
class Geometry:
    nx: int
    ny: int
    nz: int
    hx: float
    hy: float
    hz: float
    K: int
    nu: int
    nv: int
    pu: float
    pv: float
    sad: float = 1000.0
    sdd: float = 1500.0
    off_u: float = 0.0
    off_v: float = 0.0
    cx: float = 0.0
    cy: float = 0.0
    cz: float = 0.0

    @property
    def V(self):
        return self.nx * self.ny * self.nz

    @property
    def vshape(self):
        return (self.nz, self.ny, self.nx)

    @property
    def pshape(self):
        return (self.nv, self.nu)

    def _c(self) -> _Geom:
        # pitches and sizes are what the float32 C-ABI of the GPU path sees: round through float32
        f = lambda v: float(np.float32(v))
        return _Geom(self.nx, self.ny, self.nz, f(self.hx), f(self.hy), f(self.hz),
                     f(self.cx), f(self.cy), f(self.cz), self.K, self.nu, self.nv,
                     f(self.pu), f(self.pv), f(self.sad), f(self.sdd), f(self.off_u), f(self.off_v))


@dataclass
class Opts:
    max_iter: int = 10
    grad_tol: float = 0.0
    armijo_c: float = 1e-4
    armijo_beta: float = 0.5
    max_backtracks: int = 8
    init_step_vox: float = 1.0
    batched_linesearch: int = 0
    inv_max_iter: int = 50
    inv_tol_mm: float = 1e-4

    def _c(self) -> _Opts:
        f = lambda v: float(np.float32(v))
        return _Opts(self.max_iter, f(self.grad_tol), f(self.armijo_c), f(self.armijo_beta),
                     self.max_backtracks, f(self.init_step_vox), self.batched_linesearch,
                     self.inv_max_iter, f(self.inv_tol_mm))


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.orc_cost.restype = C.c_double
    return _lib


def set_threads(n: int) -> None:
    lib().orc_set_threads(int(n))


def max_threads() -> int:
    return int(lib().orc_max_threads())


SIDDON, RAY_MARCHING = 0, 1


def set_projector(kind: int, step_mm: float = 1.0) -> None:
    """Which discretisation of P project / backproject / gradient / solve use from now on: SIDDON (reading
    A3, the default) or RAY_MARCHING with the nominal step `step_mm` (reading C1)."""
    lib().orc_set_projector(int(kind), C.c_double(float(step_mm)))


def get_projector() -> int:
    return int(lib().orc_get_projector())


def _f32(a):
    a = np.ascontiguousarray(a)
    assert a.dtype == np.float32, "oracle inputs are the float32 arrays the GPU path consumes"
    return a


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _angle(theta) -> float:
    # the C-ABI passes the gantry angle as float32
    return float(np.float32(theta))


def warp(g: Geometry, f0, xbar, u, w) -> np.ndarray:
    f0, xbar, u, w = _f32(f0), _f32(xbar), _f32(u), _f64(w)
    out = np.empty(g.vshape, dtype=np.float64)
    gc = g._c()
    lib().orc_warp(C.byref(gc), _p(f0), _p(xbar), _p(u), _p(w), _p(out))
    return out


def warp_grad(g: Geometry, f0, xbar, u, w) -> np.ndarray:
    f0, xbar, u, w = _f32(f0), _f32(xbar), _f32(u), _f64(w)
    out = np.empty((3,) + g.vshape, dtype=np.float64)
    gc = g._c()
    lib().orc_warp_grad(C.byref(gc), _p(f0), _p(xbar), _p(u), _p(w), _p(out))
    return out


def project(g: Geometry, f, theta) -> np.ndarray:
    f = _f64(f)
    assert f.size == g.V
    out = np.empty(g.pshape, dtype=np.float64)
    gc = g._c()
    lib().orc_project(C.byref(gc), _p(f), C.c_double(_angle(theta)), _p(out))
    return out


def backproject(g: Geometry, r, theta) -> np.ndarray:
    r = _f64(r)
    assert r.size == g.nu * g.nv
    out = np.empty(g.vshape, dtype=np.float64)
    gc = g._c()
    lib().orc_backproject(C.byref(gc), _p(r), C.c_double(_angle(theta)), _p(out))
    return out


def traverse(g: Geometry, theta, iu: int, iv: int):
    cap = g.nx + g.ny + g.nz + 8
    ijk = np.zeros((cap, 3), dtype=np.int32)
    ln = np.zeros(cap, dtype=np.float64)
    n = C.c_int32(0)
    gap = C.c_double(0)
    gc = g._c()
    rc = lib().orc_traverse(C.byref(gc), C.c_double(_angle(theta)), int(iu), int(iv), cap, _p(ijk), _p(ln),
                            C.byref(n), C.byref(gap))
    assert rc == 0
    return ijk[:n.value].copy(), ln[:n.value].copy(), gap.value


def lsfit(p, y):
    p, y = _f64(p), _f32(y)
    a, b = C.c_double(0), C.c_double(0)
    rc = lib().orc_lsfit(C.c_int64(p.size), _p(p), _p(y), C.byref(a), C.byref(b))
    return rc, a.value, b.value


def cost(p, y, a, b) -> float:
    p, y = _f64(p), _f32(y)
    return float(lib().orc_cost(C.c_int64(p.size), _p(p), _p(y), C.c_double(a), C.c_double(b)))


def gradient(g: Geometry, f0, xbar, u, w, a, b, p, y, theta) -> np.ndarray:
    f0, xbar, u, w, p, y = _f32(f0), _f32(xbar), _f32(u), _f64(w), _f64(p), _f32(y)
    out = np.empty(g.K, dtype=np.float64)
    gc = g._c()
    lib().orc_gradient(C.byref(gc), _p(f0), _p(xbar), _p(u), _p(w), C.c_double(a), C.c_double(b), _p(p), _p(y),
                       C.c_double(_angle(theta)), _p(out))
    return out


def evaluate(g: Geometry, f0, xbar, u, w, theta):
    """f(w) and p = P f(w)."""
    f = warp(g, f0, xbar, u, w)
    return f, project(g, f, theta)


def invert(g: Geometry, xbar, u, w, r0, max_iter: int = 50, tol_mm: float = 1e-4):
    xbar, u, w = _f32(xbar), _f32(u), _f64(w)
    r0 = _f32(np.atleast_2d(r0))
    M = r0.shape[0]
    out = np.empty((M, 3), dtype=np.float64)
    its = np.zeros(M, dtype=np.int32)
    gc = g._c()
    lib().orc_invert(C.byref(gc), _p(xbar), _p(u), _p(w), M, _p(r0), int(max_iter),
                     C.c_double(float(np.float32(tol_mm))), _p(out), _p(its))
    return out, its


def dvf_at_points(g: Geometry, xbar, u, w, pts) -> np.ndarray:
    xbar, u, w = _f32(xbar), _f32(u), _f64(w)
    pts = _f64(np.atleast_2d(pts))
    out = np.empty_like(pts)
    gc = g._c()
    lib().orc_dvf_at_points(C.byref(gc), _p(xbar), _p(u), _p(w), pts.shape[0], _p(pts), _p(out))
    return out


def solve(g: Geometry, f0, xbar, u, y, theta, w0, opts: Optional[Opts] = None,
          forced_mu: Optional[Sequence[float]] = None, want_volume: bool = True):
    opts = opts or Opts()
    f0, xbar, u, y, w0 = _f32(f0), _f32(xbar), _f32(u), _f32(y), _f64(w0)
    n = opts.max_iter
    w = np.empty(g.K, dtype=np.float64)
    f = np.empty(g.vshape, dtype=np.float64) if want_volume else None
    p = np.empty(g.pshape, dtype=np.float64)
    Jt = np.full(n + 1, np.nan)
    gt = np.full(max(n, 1), np.nan)
    mt = np.full(max(n, 1), np.nan)
    bt = np.full(max(n, 1), -1, dtype=np.int32)
    res = _Result()
    fm = _f64(forced_mu) if forced_mu is not None else None
    if fm is not None:
        assert fm.size >= n
    gc, oc = g._c(), opts._c()
    lib().orc_solve(C.byref(gc), _p(f0), _p(xbar), _p(u), _p(y), C.c_double(_angle(theta)), _p(w0), C.byref(oc),
                    _p(fm) if fm is not None else None, _p(w), _p(f) if f is not None else None, _p(p),
                    C.byref(res), _p(Jt), _p(gt), _p(mt), _p(bt))
    it = res.iters
    return dict(w=w, f=f, p=p, a=res.a, b=res.b, J0=res.J0, J=res.J, iters=it, status=res.status,
                J_trace=Jt[:it + 1], gnorm_trace=gt[:min(it + 1, n)], mu_trace=mt[:it], backtracks=bt[:it])


# ---------------------------------------------------------------- frame stream
#
# PAPER.md:L141 (section 4): "We initialized the PCA coefficients to those at its previous frame";
# PAPER.md:L154 (section 5): "we can also use the predicted PCA coefficients from previous
# histories to serve as the initial guess for optimization".  The paper names no predictor;
# DESIGN.md reading B9 takes the polynomial of degree `order` through the last order + 1 frames
# (order 0 = the previous frame's w, L141), written here as the Lagrange interpolation formula.

def predict_w(times: Sequence[float], ws, t: float, order: int, w0=None) -> np.ndarray:
    """w predicted for time t from the history (times[i], ws[i]), oldest first.

    order < 0: always w0.  No history: w0.  Otherwise the Lagrange polynomial through the last
    m = min(order, len(history) - 1) + 1 frames evaluated at t, in float64:
        w(t) = sum_i w_i prod_{j != i} (t - t_j) / (t_i - t_j).
    If two of those frames share a time stamp the prediction is the last frame's w.
    """
    ws = np.asarray(ws, dtype=np.float64)
    K = ws.shape[1] if ws.ndim == 2 else (len(w0) if w0 is not None else 0)
    base = np.zeros(K) if w0 is None else np.asarray(w0, dtype=np.float64)
    if order < 0 or len(times) == 0:
        return base.copy()
    m = min(order, len(times) - 1) + 1
    ts = [float(x) for x in times[-m:]]
    wm = ws[-m:]
    if len(set(ts)) < m:
        return wm[-1].copy()
    out = np.zeros(K)
    for i in range(m):
        c = 1.0
        for j in range(m):
            if j != i:
                c *= (float(t) - ts[j]) / (ts[i] - ts[j])
        out += c * wm[i]
    return out


def solve_frames(g: Geometry, f0, xbar, u, ys, thetas, times, order: int, opts: Optional[Opts] = None, w0=None,
                 history=None):
    """The per-projection solve over consecutive frames: frame n starts from float32(predict_w(...))
    of the frames before it (w_init crosses the boundary as float32).  `history`, if given, is
    a list of (t, w) the first prediction starts from.  Returns the list of solve() results, each
    with its 'w_init'."""
    hist_t = [h[0] for h in history] if history else []
    hist_w = [np.asarray(h[1], dtype=np.float64) for h in history] if history else []
    out = []
    for y, th, t in zip(ys, thetas, times):
        wi = predict_w(hist_t, np.array(hist_w).reshape(len(hist_w), g.K), t, order, w0).astype(np.float32)
        r = solve(g, f0, xbar, u, y, th, wi, opts, want_volume=False)
        r["w_init"] = wi
        out.append(r)
        hist_t.append(float(t))
        hist_w.append(np.asarray(r["w"], dtype=np.float32).astype(np.float64))   # w leaves a solve as float32
    return out


# ---------------------------------------------------------------- PCA motion model
#
# PAPER.md:L63-69 (section 2.1, Eq. 1): "the DVF ... is approximated by a linear combination of the
# sample mean vector and a few eigenvectors corresponding to the largest eigenvalues";
# the training DVFs of the other phases relative to the reference give xbar, u_1..K.
# Written as the definition: the principal axes of the samples are the right singular vectors of
# the centred data matrix (library SVD, float64).  Reading A12: unit-norm u_k, eigenvalues of the
# scatter matrix (no 1/(N-1)), sign of u_k such that u_k . (D_sign_ref - mean) >= 0; reading B10:
# if that product is exactly 0, the training coefficient of largest magnitude is made positive.

def pca_fit(dvfs, K: int, sign_ref: Optional[int] = None):
    """dvfs [N][...] float32 samples.  Returns dict(mean [...], eig [K][...], eigenvalues [N]
    descending, coeffs [N][K] = u_k . (D_i - mean)), all float64."""
    d32 = np.asarray(dvfs, dtype=np.float32)
    N = d32.shape[0]
    shape = d32.shape[1:]
    D = d32.reshape(N, -1).astype(np.float64)
    if sign_ref is None:
        sign_ref = N // 2
    mean = D.sum(axis=0) / N
    X = D - mean[None, :]
    _, S, Vt = np.linalg.svd(X, full_matrices=False)
    lam = S ** 2
    u = Vt[:K].copy()
    coeffs = X @ u.T
    for k in range(K):
        c = coeffs[sign_ref, k]
        if c < 0 or (c == 0 and coeffs[np.argmax(np.abs(coeffs[:, k])), k] < 0):
            u[k] = -u[k]
            coeffs[:, k] = -coeffs[:, k]
    return dict(mean=mean.reshape(shape), eig=u.reshape((K,) + shape), eigenvalues=lam, coeffs=coeffs)
