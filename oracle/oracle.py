"""ctypes marshalling for oracle/osiv_oracle.c (float64 CPU oracle; test infrastructure only).

No arithmetic of the method is done here: every function forwards to the C routine of the
same name.  Arrays are numpy float64, C-contiguous; images are [ny][nx], sinograms [V_S][C]
(compact: the views of subset m in the order v = m, m+M, ...), counts [V][C].
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "osiv_oracle.c")
_SO = os.path.join(_HERE, "liboracle.so")
_lib = None


class _CGeometry(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("pixel_mm", C.c_double),
                ("n_views", C.c_int32), ("n_channels", C.c_int32), ("sad_mm", C.c_double),
                ("dgamma_rad", C.c_double), ("channel_offset", C.c_double), ("theta0_rad", C.c_double),
                ("model", C.c_int32), ("_pad", C.c_int32)]


class _CParams(C.Structure):
    _fields_ = [("beta", C.c_double), ("n_subsets", C.c_int32), ("n_iters", C.c_int32),
                ("mu0", C.c_double), ("lambda0", C.c_double), ("lambda_up", C.c_double),
                ("lambda_down", C.c_double), ("lambda_min", C.c_double), ("kappa", C.c_double),
                ("tv_eps", C.c_double), ("return_best", C.c_int32), ("monitor_mode", C.c_int32),
                ("forced_lambda", C.POINTER(C.c_double))]


@dataclass
class Geometry:
    nx: int
    ny: int
    pixel_mm: float
    n_views: int
    n_channels: int
    sad_mm: float = 850.0
    dgamma_rad: float = 0.0
    channel_offset: float = 0.0
    theta0_rad: float = 0.0
    model: int = 0                # 0: exact chord length (C2); 1: Joseph's interpolating model (8(f)-2)

    def c(self) -> _CGeometry:
        return _CGeometry(self.nx, self.ny, self.pixel_mm, self.n_views, self.n_channels, self.sad_mm,
                          self.dgamma_rad, self.channel_offset, self.theta0_rad, self.model, 0)


@dataclass
class Params:
    beta: float = 0.005
    n_subsets: int = 1
    n_iters: int = 10
    mu0: float = 0.005            # 0.05 /cm
    lambda0: float = 0.01
    lambda_up: float = 1e-4       # PAPER.md:102 Eq. 4
    lambda_down: float = 2e-4     # PAPER.md:106 Eq. 5
    lambda_min: float = 1e-4
    kappa: float = 100.0
    tv_eps: float = 1e-5
    return_best: int = 0
    monitor_mode: int = 0         # 0: Eq. 4-5 compare with D(n-1) (C10); 1: with D(n-M), the same subset (G3)
    forced_lambda: Optional[np.ndarray] = None


def build(force: bool = False) -> str:
    """Compile osiv_oracle.c with gcc (-O2, OpenMP on the outer loops only)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _SO, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        dp, gp = C.POINTER(C.c_double), C.POINTER(_CGeometry)
        L.oracle_num_threads.restype = C.c_int
        L.oracle_set_num_threads.argtypes = [C.c_int]
        L.oracle_dgamma.restype = C.c_double
        L.oracle_dgamma.argtypes = [gp]
        L.oracle_ray.argtypes = [gp, C.c_int, C.c_int, dp, dp, dp, dp]
        L.oracle_weight.restype = C.c_double
        L.oracle_weight.argtypes = [gp, C.c_int, C.c_int, C.c_int, C.c_int]
        L.oracle_candidate_K.restype = C.c_int
        L.oracle_candidate_K.argtypes = [gp]
        for name in ("oracle_forward", "oracle_forward_brute", "oracle_backward", "oracle_backward_brute"):
            getattr(L, name).argtypes = [gp, dp, dp, C.c_int, C.c_int]
            getattr(L, name).restype = None
        L.oracle_tv_value.restype = C.c_double
        L.oracle_tv_value.argtypes = [dp, C.c_int, C.c_int, C.c_double]
        L.oracle_tv_grad.argtypes = [dp, dp, C.c_int, C.c_int, C.c_double]
        L.oracle_loglik.restype = C.c_double
        L.oracle_loglik.argtypes = [gp, dp, dp, dp, C.c_double, C.c_int, C.c_int]
        L.oracle_residual.restype = C.c_double
        L.oracle_residual.argtypes = [gp, dp, dp, dp, C.c_double, C.c_int, C.c_int, dp]
        L.oracle_tau.restype = C.c_double
        L.oracle_tau.argtypes = [gp, C.c_int, C.c_double]
        L.oracle_tv3_value.restype = C.c_double
        L.oracle_tv3_value.argtypes = [dp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double]
        L.oracle_tv3_grad.argtypes = [dp, dp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double]
        L.oracle_reconstruct_stack.restype = C.c_int
        L.oracle_reconstruct_stack.argtypes = [gp, C.c_int, dp, dp, C.c_double, C.POINTER(_CParams), C.c_int, C.c_double, dp, dp]
        L.oracle_reconstruct.restype = C.c_int
        L.oracle_reconstruct.argtypes = [gp, dp, dp, C.c_double, C.POINTER(_CParams), dp, dp]
        _lib = L
    return _lib


def _dp(a: Optional[np.ndarray]):
    if a is None:
        return None
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _nvs(g: Geometry, subset: int, n_subsets: int) -> int:
    return g.n_views if subset < 0 else g.n_views // n_subsets


def num_threads() -> int:
    return lib().oracle_num_threads()


def set_num_threads(n: int) -> None:
    lib().oracle_set_num_threads(int(n))


def dgamma(g: Geometry) -> float:
    return lib().oracle_dgamma(C.byref(g.c()))


def ray(g: Geometry, v: int, c: int):
    out = [C.c_double() for _ in range(4)]
    lib().oracle_ray(C.byref(g.c()), v, c, *[C.byref(o) for o in out])
    return tuple(o.value for o in out)


def weight(g: Geometry, v: int, c: int, ix: int, iy: int) -> float:
    return lib().oracle_weight(C.byref(g.c()), v, c, ix, iy)


def candidate_K(g: Geometry) -> int:
    return lib().oracle_candidate_K(C.byref(g.c()))


def _proj(name: str, g: Geometry, src: np.ndarray, out_shape, subset: int, n_subsets: int) -> np.ndarray:
    src = _f64(src)
    out = np.zeros(out_shape, dtype=np.float64)
    getattr(lib(), name)(C.byref(g.c()), _dp(src), _dp(out), subset, n_subsets)
    return out


def forward(g: Geometry, img, subset: int = -1, n_subsets: int = 1) -> np.ndarray:
    assert np.shape(img) == (g.ny, g.nx)
    return _proj("oracle_forward", g, img, (_nvs(g, subset, n_subsets), g.n_channels), subset, n_subsets)


def forward_brute(g: Geometry, img, subset: int = -1, n_subsets: int = 1) -> np.ndarray:
    assert np.shape(img) == (g.ny, g.nx)
    return _proj("oracle_forward_brute", g, img, (_nvs(g, subset, n_subsets), g.n_channels), subset, n_subsets)


def backward(g: Geometry, sino, subset: int = -1, n_subsets: int = 1) -> np.ndarray:
    assert np.shape(sino) == (_nvs(g, subset, n_subsets), g.n_channels)
    return _proj("oracle_backward", g, sino, (g.ny, g.nx), subset, n_subsets)


def backward_brute(g: Geometry, sino, subset: int = -1, n_subsets: int = 1) -> np.ndarray:
    assert np.shape(sino) == (_nvs(g, subset, n_subsets), g.n_channels)
    return _proj("oracle_backward_brute", g, sino, (g.ny, g.nx), subset, n_subsets)


def tv_value(mu, eps: float) -> float:
    mu = _f64(mu)
    return lib().oracle_tv_value(_dp(mu), mu.shape[1], mu.shape[0], eps)


def tv_grad(mu, eps: float) -> np.ndarray:
    mu = _f64(mu)
    out = np.zeros_like(mu)
    lib().oracle_tv_grad(_dp(mu), _dp(out), mu.shape[1], mu.shape[0], eps)
    return out


def _blank(blank):
    if np.isscalar(blank):
        return None, float(blank)
    b = _f64(blank)
    return b, 0.0


def loglik(g: Geometry, img, counts, blank, subset: int = -1, n_subsets: int = 1) -> float:
    img, counts = _f64(img), _f64(counts)
    b, bs = _blank(blank)
    return lib().oracle_loglik(C.byref(g.c()), _dp(img), _dp(counts), _dp(b), bs, subset, n_subsets)


def residual(g: Geometry, l, counts, blank, subset: int = -1, n_subsets: int = 1):
    """returns (r [V_S][C], D)"""
    l, counts = _f64(l), _f64(counts)
    b, bs = _blank(blank)
    r = np.zeros_like(l)
    D = lib().oracle_residual(C.byref(g.c()), _dp(l), _dp(counts), _dp(b), bs, subset, n_subsets, _dp(r))
    return r, D


def tau(g: Geometry, n_subsets: int, kappa: float = 100.0) -> float:
    return lib().oracle_tau(C.byref(g.c()), n_subsets, kappa)


def reconstruct(g: Geometry, counts, blank, prm: Params):
    """returns (image [ny][nx] float64, trace [n_iters][2] = (D, lambda), status)"""
    counts = _f64(counts)
    assert counts.shape == (g.n_views, g.n_channels)
    assert g.n_views % prm.n_subsets == 0
    b, bs = _blank(blank)
    forced = None if prm.forced_lambda is None else _f64(prm.forced_lambda)
    if forced is not None:
        assert forced.shape == (prm.n_iters,)
    cp = _CParams(prm.beta, prm.n_subsets, prm.n_iters, prm.mu0, prm.lambda0, prm.lambda_up, prm.lambda_down,
                  prm.lambda_min, prm.kappa, prm.tv_eps, prm.return_best, prm.monitor_mode, _dp(forced))
    img = np.zeros((g.ny, g.nx), dtype=np.float64)
    trace = np.zeros((prm.n_iters, 2), dtype=np.float64)
    status = lib().oracle_reconstruct(C.byref(g.c()), _dp(counts), _dp(b), bs, C.byref(cp), _dp(img), _dp(trace))
    return img, trace, status


def tv3_value(mu, eps: float, wz: float) -> float:
    """3-D smoothed isotropic TV of a stack [S][ny][nx] (reading H2)"""
    mu = _f64(mu)
    return lib().oracle_tv3_value(_dp(mu), mu.shape[2], mu.shape[1], mu.shape[0], eps, wz)


def tv3_grad(mu, eps: float, wz: float):
    mu = _f64(mu)
    out = np.zeros_like(mu)
    lib().oracle_tv3_grad(_dp(mu), _dp(out), mu.shape[2], mu.shape[1], mu.shape[0], eps, wz)
    return out


def reconstruct_stack(g: Geometry, counts, blank, prm: Params, view_shift: int = 0, tv_z: float = 0.0):
    """Stack of S slices (readings H1-H3): counts [S][V][C] -> (images [S][ny][nx], trace [S][n_iters][2], status)"""
    counts = _f64(counts)
    S = counts.shape[0]
    assert counts.shape[1:] == (g.n_views, g.n_channels) and g.n_views % prm.n_subsets == 0
    assert prm.forced_lambda is None and not prm.return_best
    b, bs = _blank(blank)
    cp = _CParams(prm.beta, prm.n_subsets, prm.n_iters, prm.mu0, prm.lambda0, prm.lambda_up, prm.lambda_down,
                  prm.lambda_min, prm.kappa, prm.tv_eps, 0, prm.monitor_mode, None)
    img = np.zeros((S, g.ny, g.nx), dtype=np.float64)
    trace = np.zeros((S, prm.n_iters, 2), dtype=np.float64)
    status = lib().oracle_reconstruct_stack(C.byref(g.c()), S, _dp(counts), _dp(b), bs, C.byref(cp), view_shift, tv_z,
                                            _dp(img), _dp(trace))
    return img, trace, status
