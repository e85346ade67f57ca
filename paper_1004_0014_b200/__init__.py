"""Thin Python binding of libpcamm (include/pcamm.h): argument marshalling only.

Every step of the hot path (DVF synthesis + warp, cone-beam projection, intensity fit, fused
adjoint gradient, Armijo loop, tumour localisation; PAPER.md sections 2.1-2.3) runs in the CUDA
kernels behind the C ABI.  PyTorch supplies device memory and the current stream; nothing here
computes.  There is no CPU fallback: importing works without a GPU (so that the symbol table
can be checked), creating a :class:`Model` does not.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass, field
from typing import Optional, Sequence

import numpy as np

from .build import LIB, build as _build

KMAX = 8
MAX_BACKTRACKS = 16

OK, E_INVALID, E_CUDA, E_NOMEM, E_NONFINITE, E_SINGULAR = 0, -1, -2, -3, -4, -5
S_MAXITER, S_GRADTOL, S_LINESEARCH = 1, 2, 3


class pcamm_geometry(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("hx", C.c_float), ("hy", C.c_float), ("hz", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float), ("cz", C.c_float),
                ("K", C.c_int32), ("nu", C.c_int32), ("nv", C.c_int32),
                ("pu", C.c_float), ("pv", C.c_float), ("sad", C.c_float), ("sdd", C.c_float),
                ("off_u", C.c_float), ("off_v", C.c_float),
                ("max_batch", C.c_int32), ("max_candidates", C.c_int32), ("field_storage", C.c_int32), ("tile_skipping", C.c_int32),
                ("projector", C.c_int32), ("ray_step_vox", C.c_float)]


class pcamm_opts(C.Structure):
    _fields_ = [("max_iter", C.c_int32), ("grad_tol", C.c_float), ("armijo_c", C.c_float),
                ("armijo_beta", C.c_float), ("max_backtracks", C.c_int32), ("init_step_vox", C.c_float),
                ("batched_linesearch", C.c_int32), ("inv_max_iter", C.c_int32), ("inv_tol_mm", C.c_float),
                ("loop_mode", C.c_int32)]


class pcamm_info(C.Structure):
    _fields_ = [("iters", C.c_int32), ("status", C.c_int32), ("J0", C.c_double), ("J", C.c_double),
                ("a", C.c_double), ("b", C.c_double),
                ("J_trace", C.POINTER(C.c_double)), ("gnorm_trace", C.POINTER(C.c_double)),
                ("mu_trace", C.POINTER(C.c_double)), ("backtracks_trace", C.POINTER(C.c_int32))]


# every symbol include/pcamm.h declares
SYMBOLS = ("pcamm_default_opts", "pcamm_model_create", "pcamm_model_destroy", "pcamm_model_fields",
           "pcamm_reconstruct",
           "pcamm_reconstruct_host", "pcamm_reconstruct_batch", "pcamm_warp", "pcamm_project",
           "pcamm_backproject", "pcamm_eval", "pcamm_traverse", "pcamm_localise", "pcamm_time_kernel", "pcamm_time_slots",
           "pcamm_tune", "pcamm_tile_counts", "pcamm_timeline", "pcamm_fit_cost_static", "pcamm_launch_count", "pcamm_last_error", "pcamm_pca_fit", "pcamm_predict_w", "pcamm_frames_create",
           "pcamm_frames_destroy", "pcamm_frames_reset", "pcamm_frames_count", "pcamm_frames_predict",
           "pcamm_frames_push")

_lib = None


class PcammError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"pcamm error {code}: {msg}")
        self.code = code


def lib(build_if_missing: bool = True):
    """Load libpcamm.so (compiling it in-tree first if it is missing or stale)."""
    global _lib
    if _lib is None:
        path = _build() if build_if_missing else LIB
        if not os.path.exists(path):
            raise ImportError(f"{path} is missing: run `python -m paper_1004_0014_b200.build` (there is no fallback)")
        L = C.CDLL(path)
        L.pcamm_last_error.restype = C.c_char_p
        L.pcamm_launch_count.restype = C.c_int64
        L.pcamm_model_destroy.restype = None
        L.pcamm_default_opts.restype = None
        L.pcamm_frames_destroy.restype = None
        L.pcamm_frames_count.restype = C.c_int32
        _lib = L
    return _lib


def last_error() -> str:
    return (lib().pcamm_last_error() or b"").decode()


def launch_count(reset: bool = False) -> int:
    return int(lib().pcamm_launch_count(1 if reset else 0))


def tune(name: str, value: int) -> None:
    """pcamm_tune: a measurement knob (set before creating the Model)."""
    _check(lib().pcamm_tune(name.encode(), int(value)))


def _check(rc: int) -> int:
    if rc < 0:
        raise PcammError(rc, last_error())
    return rc


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
    loop_mode: int = 0

    def _c(self) -> pcamm_opts:
        return pcamm_opts(self.max_iter, self.grad_tol, self.armijo_c, self.armijo_beta, self.max_backtracks,
                          self.init_step_vox, self.batched_linesearch, self.inv_max_iter, self.inv_tol_mm,
                          self.loop_mode)


@dataclass
class Result:
    w: np.ndarray
    status: int
    iters: int
    J0: float
    J: float
    a: float
    b: float
    landmarks: Optional[np.ndarray] = None
    J_trace: Optional[np.ndarray] = None
    gnorm_trace: Optional[np.ndarray] = None
    mu_trace: Optional[np.ndarray] = None
    backtracks: Optional[np.ndarray] = None
    w_init: Optional[np.ndarray] = None   # Frames.push: the predicted start


def _torch():
    import torch
    return torch


def _dev_f32(t, n: int, name: str):
    torch = _torch()
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError(f"{name}: expected a contiguous float32 CUDA tensor")
    if t.numel() != n:
        raise ValueError(f"{name}: expected {n} elements, got {t.numel()}")
    return C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(_torch().cuda.current_stream().cuda_stream)


def _host_f32(a, n: int):
    a = np.ascontiguousarray(a, dtype=np.float32).reshape(-1)
    if a.size != n:
        raise ValueError(f"expected {n} values, got {a.size}")
    return a


class Model:
    """pcamm_model_create / pcamm_model_destroy and the calls on a model.

    f0 [nz][ny][nx], mean_dvf [3][nz][ny][nx], eig_dvf [K][3][nz][ny][nx] are float32 CUDA tensors
    (copied by the library); landmarks_mm [M][3] is a host array.
    """

    def __init__(self, *, nx, ny, nz, hx, hy, hz, K, nu, nv, pu, pv, f0, mean_dvf, eig_dvf,
                 landmarks_mm=None, sad=1000.0, sdd=1500.0, off_u=0.0, off_v=0.0, cx=0.0, cy=0.0, cz=0.0,
                 max_batch=1, max_candidates=1, field_storage=0, tile_skipping=0, projector=0, ray_step_vox=0.0):
        torch = _torch()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1004_0014_b200 needs a CUDA device (there is no CPU fallback)")
        self.geo = pcamm_geometry(nx, ny, nz, hx, hy, hz, cx, cy, cz, K, nu, nv, pu, pv, sad, sdd, off_u, off_v,
                                  max_batch, max_candidates, field_storage, tile_skipping, projector, ray_step_vox)
        self.K, self.V, self.npix = K, nx * ny * nz, nu * nv
        self.vshape, self.pshape = (nz, ny, nx), (nv, nu)
        lm = np.zeros((0, 3), np.float32) if landmarks_mm is None else \
            np.ascontiguousarray(np.atleast_2d(landmarks_mm), dtype=np.float32)
        self.M = lm.shape[0]
        self._h = C.c_void_p()
        _check(lib().pcamm_model_create(C.byref(self.geo), _dev_f32(f0, self.V, "f0"),
                                        _dev_f32(mean_dvf, 3 * self.V, "mean_dvf"),
                                        _dev_f32(eig_dvf, 3 * K * self.V, "eig_dvf"), self.M,
                                        lm.ctypes.data_as(C.c_void_p), _stream(), C.byref(self._h)))
        self.device = f0.device

    def fields(self):
        """pcamm_model_fields: (mean_dvf [3][nz][ny][nx], eig_dvf [K][3][nz][ny][nx]) in mm as the solve uses them."""
        torch = _torch()
        mean = torch.empty((3,) + self.vshape, dtype=torch.float32, device=self.device)
        eig = torch.empty((self.K, 3) + self.vshape, dtype=torch.float32, device=self.device)
        _check(lib().pcamm_model_fields(self._h, C.c_void_p(mean.data_ptr()), C.c_void_p(eig.data_ptr()), _stream()))
        return mean, eig

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib().pcamm_model_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the solve

    def _info(self, opts: Opts, B: int, trace: bool):
        infos = (pcamm_info * B)()
        keep = []
        if trace:
            n = max(opts.max_iter, 1)
            for b in range(B):
                Jt = np.full(n + 1, np.nan)
                gt = np.full(n, np.nan)
                mt = np.full(n, np.nan)
                bt = np.full(n, -1, dtype=np.int32)
                infos[b].J_trace = Jt.ctypes.data_as(C.POINTER(C.c_double))
                infos[b].gnorm_trace = gt.ctypes.data_as(C.POINTER(C.c_double))
                infos[b].mu_trace = mt.ctypes.data_as(C.POINTER(C.c_double))
                infos[b].backtracks_trace = bt.ctypes.data_as(C.POINTER(C.c_int32))
                keep.append((Jt, gt, mt, bt))
        return infos, keep

    def _result(self, b, w, lm, infos, keep, max_iter) -> Result:
        I = infos[b]
        r = Result(w=w[b].copy(), status=I.status, iters=I.iters, J0=I.J0, J=I.J, a=I.a, b=I.b,
                   landmarks=lm[b].copy() if lm is not None else None)
        if keep:
            Jt, gt, mt, bt = keep[b]
            it = I.iters
            r.J_trace, r.gnorm_trace = Jt[:it + 1], gt[:min(it + 1, max_iter)]
            r.mu_trace, r.backtracks = mt[:it], bt[:it]
        return r

    def reconstruct(self, y, angle_rad: float, w_init, opts: Optional[Opts] = None, volume_out=None,
                    trace: bool = False, host_y: bool = False) -> Result:
        """pcamm_reconstruct (y: CUDA tensor) or pcamm_reconstruct_host (host_y=True, y: host array)."""
        opts = opts or Opts()
        w0 = _host_f32(w_init, self.K)
        w = np.zeros((1, self.K), np.float32)
        lm = np.zeros((1, self.M, 3), np.float32) if self.M else None
        infos, keep = self._info(opts, 1, trace)
        oc = opts._c()
        vol = _dev_f32(volume_out, self.V, "volume_out") if volume_out is not None else None
        if host_y:
            yh = y if isinstance(y, np.ndarray) else y.numpy()
            assert yh.dtype == np.float32 and yh.flags.c_contiguous and yh.size == self.npix
            fn, yarg = lib().pcamm_reconstruct_host, C.c_void_p(yh.ctypes.data)
        else:
            fn, yarg = lib().pcamm_reconstruct, _dev_f32(y, self.npix, "y")
        _check(fn(self._h, yarg, C.c_float(angle_rad), w0.ctypes.data_as(C.c_void_p), C.byref(oc),
                  w.ctypes.data_as(C.c_void_p), vol, lm.ctypes.data_as(C.c_void_p) if lm is not None else None,
                  infos, _stream()))
        return self._result(0, w, lm, infos, keep, opts.max_iter)

    def reconstruct_batch(self, y, angles_rad, w_init, opts: Optional[Opts] = None, volumes_out=None,
                          trace: bool = False):
        opts = opts or Opts()
        ang = np.ascontiguousarray(angles_rad, dtype=np.float32).reshape(-1)
        B = ang.size
        w0 = _host_f32(w_init, B * self.K)
        w = np.zeros((B, self.K), np.float32)
        lm = np.zeros((B, self.M, 3), np.float32) if self.M else None
        infos, keep = self._info(opts, B, trace)
        oc = opts._c()
        vol = _dev_f32(volumes_out, B * self.V, "volumes_out") if volumes_out is not None else None
        _check(lib().pcamm_reconstruct_batch(self._h, B, _dev_f32(y, B * self.npix, "y"),
                                             ang.ctypes.data_as(C.c_void_p), w0.ctypes.data_as(C.c_void_p),
                                             C.byref(oc), w.ctypes.data_as(C.c_void_p), vol,
                                             lm.ctypes.data_as(C.c_void_p) if lm is not None else None, infos,
                                             _stream()))
        return [self._result(b, w, lm, infos, keep, opts.max_iter) for b in range(B)]

    # ---- function-level hooks

    def _empty(self, shape):
        torch = _torch()
        return torch.empty(shape, dtype=torch.float32, device=self.device)

    def warp(self, w, out=None):
        out = self._empty(self.vshape) if out is None else out
        w = _host_f32(w, self.K)
        _check(lib().pcamm_warp(self._h, w.ctypes.data_as(C.c_void_p), _dev_f32(out, self.V, "out"), _stream()))
        return out

    def project(self, volume, angle_rad: float, out=None):
        out = self._empty(self.pshape) if out is None else out
        _check(lib().pcamm_project(self._h, _dev_f32(volume, self.V, "volume"), C.c_float(angle_rad),
                                   _dev_f32(out, self.npix, "out"), _stream()))
        return out

    def backproject(self, r, angle_rad: float, out=None):
        out = self._empty(self.vshape) if out is None else out
        _check(lib().pcamm_backproject(self._h, _dev_f32(r, self.npix, "r"), C.c_float(angle_rad),
                                       _dev_f32(out, self.V, "out"), _stream()))
        return out

    def eval(self, y, angle_rad: float, w, a: float, b: float, want_proj: bool = True):
        """J, grad [K], (a_fit, b_fit), p at (w, a, b)."""
        w = _host_f32(w, self.K)
        J = C.c_double(0)
        g = np.zeros(self.K, np.float64)
        ab = np.zeros(2, np.float64)
        p = self._empty(self.pshape) if want_proj else None
        _check(lib().pcamm_eval(self._h, _dev_f32(y, self.npix, "y"), C.c_float(angle_rad),
                                w.ctypes.data_as(C.c_void_p), C.c_float(a), C.c_float(b), C.byref(J),
                                g.ctypes.data_as(C.c_void_p), ab.ctypes.data_as(C.c_void_p),
                                _dev_f32(p, self.npix, "p") if p is not None else None, _stream()))
        return J.value, g, (ab[0], ab[1]), p

    def traverse(self, angle_rad: float, iu: int, iv: int):
        cap = self.geo.nx + self.geo.ny + self.geo.nz + 8
        ijk = np.zeros((cap, 3), np.int32)
        ln = np.zeros(cap, np.float32)
        n = C.c_int32(0)
        _check(lib().pcamm_traverse(self._h, C.c_float(angle_rad), int(iu), int(iv), cap,
                                    ijk.ctypes.data_as(C.c_void_p), ln.ctypes.data_as(C.c_void_p), C.byref(n),
                                    _stream()))
        return ijk[:n.value].copy(), ln[:n.value].copy()

    def localise(self, w, inv_max_iter: int = 50, inv_tol_mm: float = 1e-4) -> np.ndarray:
        w = _host_f32(w, self.K)
        out = np.zeros((self.M, 3), np.float32)
        _check(lib().pcamm_localise(self._h, w.ctypes.data_as(C.c_void_p), int(inv_max_iter), C.c_float(inv_tol_mm),
                                    out.ctypes.data_as(C.c_void_p), _stream()))
        return out

    def timeline(self):
        """pcamm_timeline: (kind, start_us, end_us) arrays of the kernels of the last solve (timeline knob)."""
        cap = 2048
        kind = np.zeros(cap, np.int32)
        t0 = np.zeros(cap, np.float64)
        t1 = np.zeros(cap, np.float64)
        n = C.c_int32(0)
        _check(lib().pcamm_timeline(self._h, cap, kind.ctypes.data_as(C.c_void_p), t0.ctypes.data_as(C.c_void_p),
                                    t1.ctypes.data_as(C.c_void_p), C.byref(n), _stream()))
        k = min(n.value, cap)
        return kind[:k].copy(), t0[:k].copy(), t1[:k].copy()

    def tile_counts(self, reset: bool = False):
        """pcamm_tile_counts: (warp tiles loaded, gradient tiles loaded, tiles of the volume, voxels per tile,
        gradient records gathered, gradient records written by the warp kernel)."""
        out = (C.c_int64 * 6)()
        _check(lib().pcamm_tile_counts(self._h, 1 if reset else 0, out, _stream()))
        return tuple(int(v) for v in out)

    def time_slots(self, w) -> None:
        """pcamm_time_slots: the candidate coefficient vectors [n][K] the warp / projection timings run over."""
        w = np.ascontiguousarray(w, np.float32).reshape(-1, self.K)
        _check(lib().pcamm_time_slots(self._h, int(w.shape[0]), w.ctypes.data_as(C.c_void_p), _stream()))

    def time_kernel(self, which: int, reps: int = 20) -> float:
        """Average device milliseconds per launch of kernel 0 warp / 1 project / 2 gradient on the
        inputs left by the last :meth:`eval` (CUDA events on the current stream, inside the library)."""
        ms = C.c_float(0)
        _check(lib().pcamm_time_kernel(self._h, int(which), int(reps), C.byref(ms), _stream()))
        return float(ms.value)


STATIC_MAX_PIXELS = 1 << 22     # PCAMM_STATIC_MAX_PIXELS


def fit_cost_static(p, y, out=None):
    """pcamm_fit_cost_static: the intensity fit (Eq. 4) and cost (Eq. 2) of the projection pair (p, y)
    (float32 CUDA tensors of the same size, at most STATIC_MAX_PIXELS pixels) without a model and
    without any allocation inside the library (its scratch is a static device array; calls that
    overlap on the GPU race on it).  `out`: a float64 CUDA tensor of 8 elements to receive the results
    (allocated here if None; pass one where nothing may allocate).  Asynchronous: returns `out`
    = (a, b, J, sum p, sum y, sum y^2, sum y p, status), valid once the current stream reaches it."""
    torch = _torch()
    n = int(p.numel())
    pp, yy = _dev_f32(p, n, "p"), _dev_f32(y, n, "y")
    if out is None:
        out = torch.empty(8, dtype=torch.float64, device=p.device)
    if not (out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == 8):
        raise TypeError("out: expected a contiguous float64 CUDA tensor of 8 elements")
    _check(lib().pcamm_fit_cost_static(pp, yy, C.c_int64(n), C.c_void_p(out.data_ptr()), _stream()))
    return out


def pca_fit(dvfs, K: int, sign_ref: int = -1, pass_ms: Optional[list] = None):
    """pcamm_pca_fit: the PCA motion model of the training DVFs `dvfs` [N][...] (float32 CUDA tensor).
    Returns (mean [...], eig [K][...]) as CUDA tensors in the layout Model takes, the N eigenvalues of
    the scatter matrix (descending) and the training coefficients [N][K] (float64 host arrays)."""
    torch = _torch()
    if not (dvfs.is_cuda and dvfs.dtype == torch.float32 and dvfs.is_contiguous()):
        raise ValueError("dvfs must be a contiguous float32 CUDA tensor")
    N = int(dvfs.shape[0])
    n = dvfs[0].numel()
    mean = torch.empty(tuple(dvfs.shape[1:]), dtype=torch.float32, device=dvfs.device)
    eig = torch.empty((K,) + tuple(dvfs.shape[1:]), dtype=torch.float32, device=dvfs.device)
    lam = np.zeros(max(N, 1), np.float64)
    coeffs = np.zeros((max(N, 1), max(K, 1)), np.float64)
    ms = (C.c_float * 2)()
    _check(lib().pcamm_pca_fit(C.c_int64(n), N, int(K), C.c_void_p(dvfs.data_ptr()), int(sign_ref),
                               C.c_void_p(mean.data_ptr()), C.c_void_p(eig.data_ptr()), lam.ctypes.data_as(C.c_void_p),
                               coeffs.ctypes.data_as(C.c_void_p), ms if pass_ms is not None else None, _stream()))
    if pass_ms is not None:
        pass_ms[:] = [float(ms[0]), float(ms[1])]
    return mean, eig, lam, coeffs


def predict_w(order: int, times, ws, t: float, w0=None, K: Optional[int] = None) -> np.ndarray:
    """pcamm_predict_w: the start predicted for time t from the history (times[i], ws[i]), oldest first."""
    ws = np.ascontiguousarray(ws, dtype=np.float32)
    ts = np.ascontiguousarray(times, dtype=np.float64).reshape(-1)
    n = ts.size
    K = K or (ws.shape[1] if ws.ndim == 2 and n else len(w0))
    ws = ws.reshape(n, K)
    w0a = _host_f32(w0, K) if w0 is not None else None
    out = np.zeros(K, np.float32)
    _check(lib().pcamm_predict_w(int(order), int(K), int(n), ts.ctypes.data_as(C.c_void_p), ws.ctypes.data_as(C.c_void_p),
                                 w0a.ctypes.data_as(C.c_void_p) if w0a is not None else None, C.c_double(t),
                                 out.ctypes.data_as(C.c_void_p)))
    return out


class Frames:
    """pcamm_frames_*: consecutive projections of one treatment; each solve starts from the
    coefficients predicted from the frames before it (order 0: the previous frame's w, 1: linear,
    2: quadratic extrapolation in the frames' time stamps, -1: always w0)."""

    def __init__(self, model: Model, order: int = 0, w0=None):
        self.model = model                    # keeps the model alive
        self._h = C.c_void_p()
        w0a = _host_f32(w0, model.K) if w0 is not None else None
        _check(lib().pcamm_frames_create(model._h, int(order), w0a.ctypes.data_as(C.c_void_p) if w0a is not None else None,
                                         C.byref(self._h)))

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib().pcamm_frames_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def reset(self) -> None:
        _check(lib().pcamm_frames_reset(self._h))

    def count(self) -> int:
        return int(lib().pcamm_frames_count(self._h))

    def predict(self, t: float) -> np.ndarray:
        w = np.zeros(self.model.K, np.float32)
        _check(lib().pcamm_frames_predict(self._h, C.c_double(t), w.ctypes.data_as(C.c_void_p)))
        return w

    def push(self, y, angle_rad: float, t: float, opts: Optional[Opts] = None, volume_out=None, trace: bool = False,
             host_y: bool = False) -> Result:
        """Solve the frame measured at time t; the result carries the start that was used as w_init."""
        m = self.model
        opts = opts or Opts()
        w = np.zeros((1, m.K), np.float32)
        wi = np.zeros(m.K, np.float32)
        lm = np.zeros((1, m.M, 3), np.float32) if m.M else None
        infos, keep = m._info(opts, 1, trace)
        oc = opts._c()
        vol = _dev_f32(volume_out, m.V, "volume_out") if volume_out is not None else None
        if host_y:
            yh = y if isinstance(y, np.ndarray) else y.numpy()
            assert yh.dtype == np.float32 and yh.flags.c_contiguous and yh.size == m.npix
            yarg = C.c_void_p(yh.ctypes.data)
        else:
            yarg = _dev_f32(y, m.npix, "y")
        _check(lib().pcamm_frames_push(self._h, yarg, 1 if host_y else 0, C.c_float(angle_rad), C.c_double(t),
                                       C.byref(oc), w.ctypes.data_as(C.c_void_p), wi.ctypes.data_as(C.c_void_p), vol,
                                       lm.ctypes.data_as(C.c_void_p) if lm is not None else None, infos, _stream()))
        r = m._result(0, w, lm, infos, keep, opts.max_iter)
        r.w_init = wi
        return r
