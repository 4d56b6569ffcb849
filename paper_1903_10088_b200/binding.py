"""ctypes binding of include/osiv.h: same names, argument marshalling only (no arithmetic of the method).

Device buffers are torch CUDA tensors (float32, contiguous); work is enqueued on torch's current stream.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np

from . import build as _build

OSIV_OK, OSIV_ERR_INVALID_ARG, OSIV_ERR_CUDA, OSIV_ERR_NOT_FINITE, OSIV_ERR_SCRATCH_LIMIT = 0, -1, -2, -3, -4
STATIC_SCRATCH_BYTES = 4 << 20      # OSIV_STATIC_SCRATCH_BYTES of include/osiv.h

EXPORTED_SYMBOLS = (
    "osiv_version", "osiv_strerror", "osiv_default_params", "osiv_create", "osiv_destroy", "osiv_ray_table", "osiv_get_dgamma",
    "osiv_get_tau", "osiv_launch_count", "osiv_set_symmetry", "osiv_set_overlap", "osiv_set_back_kernel", "osiv_get_back_kernel", "osiv_set_graph", "osiv_graph_replays", "osiv_debug_checks", "osiv_get_plan", "osiv_set_profiling", "osiv_get_profile", "osiv_forward", "osiv_backward", "osiv_tv_gradient", "osiv_tv_gradient_static", "osiv_reconstruct",
    "osiv_reconstruct_host", "osiv_probe_peaks", "osiv_debug_timeline",
)


class OsivError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {strerror(status)} ({status})")


class _CGeometry(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("pixel_mm", C.c_double), ("n_views", C.c_int32),
                ("n_channels", C.c_int32), ("sad_mm", C.c_double), ("sdd_mm", C.c_double), ("dgamma_rad", C.c_double),
                ("channel_offset", C.c_double), ("theta0_rad", C.c_double), ("model", C.c_int32), ("reserved", C.c_int32)]


class _CParams(C.Structure):
    _fields_ = [("beta", C.c_double), ("n_subsets", C.c_int32), ("n_iters", C.c_int32), ("mu0", C.c_double),
                ("lambda0", C.c_double), ("lambda_up", C.c_double), ("lambda_down", C.c_double),
                ("lambda_min", C.c_double), ("kappa", C.c_double), ("tv_eps", C.c_double),
                ("return_best", C.c_int32), ("monitor_mode", C.c_int32), ("view_shift", C.c_int32), ("reserved", C.c_int32),
                ("tv_z", C.c_double), ("forced_lambda", C.POINTER(C.c_double))]


@dataclass
class Geometry:
    nx: int
    ny: int
    pixel_mm: float
    n_views: int
    n_channels: int
    sad_mm: float = 850.0
    sdd_mm: float = 1450.0
    dgamma_rad: float = 0.0
    channel_offset: float = 0.0
    theta0_rad: float = 0.0
    model: int = 0

    def c(self) -> _CGeometry:
        return _CGeometry(self.nx, self.ny, self.pixel_mm, self.n_views, self.n_channels, self.sad_mm, self.sdd_mm,
                          self.dgamma_rad, self.channel_offset, self.theta0_rad, self.model, 0)


@dataclass
class Params:
    beta: float = 0.005
    n_subsets: int = 1
    n_iters: int = 1
    mu0: float = 0.005
    lambda0: float = 0.01
    lambda_up: float = 1e-4
    lambda_down: float = 2e-4
    lambda_min: float = 1e-4
    kappa: float = 100.0
    tv_eps: float = 1e-5
    return_best: int = 0
    monitor_mode: int = 0
    view_shift: int = 0
    tv_z: float = 0.0
    forced_lambda: Optional[np.ndarray] = None


_lib = None


def lib_path() -> str:
    return _build.SO


def lib():
    """Load libosiv.so (building it with nvcc if the sources are newer).  Raises if it cannot be had."""
    global _lib
    if _lib is None:
        # OSIV_TRACE_BUILD=1 selects the timeline build of the same sources (diagnostics; see timeline.py)
        # OSIV_CHECK_BUILD=1 selects the build with device-side index checks (diagnostics; osiv_debug_checks)
        path = _build.build(trace=os.environ.get("OSIV_TRACE_BUILD", "") == "1", check=os.environ.get("OSIV_CHECK_BUILD", "") == "1")
        L = C.CDLL(path)
        vp, ip = C.c_void_p, C.c_int32
        L.osiv_version.restype = C.c_int
        L.osiv_strerror.restype = C.c_char_p
        L.osiv_strerror.argtypes = [C.c_int]
        L.osiv_default_params.argtypes = [C.POINTER(_CParams)]
        L.osiv_create.argtypes = [C.POINTER(_CGeometry), ip, ip, C.POINTER(vp)]
        L.osiv_destroy.argtypes = [vp]
        L.osiv_ray_table.argtypes = [C.POINTER(_CGeometry), vp, vp]
        L.osiv_get_dgamma.argtypes = [vp, C.POINTER(C.c_double)]
        L.osiv_get_tau.argtypes = [vp, ip, C.c_double, C.POINTER(C.c_double)]
        L.osiv_launch_count.restype = C.c_int64
        L.osiv_launch_count.argtypes = [vp]
        L.osiv_set_symmetry.argtypes = [vp, ip]
        L.osiv_set_overlap.argtypes = [vp, ip]
        L.osiv_set_back_kernel.argtypes = [vp, ip]
        L.osiv_set_graph.argtypes = [vp, ip]
        L.osiv_graph_replays.argtypes = [vp]
        L.osiv_graph_replays.restype = C.c_int64
        L.osiv_get_back_kernel.argtypes = [vp, ip, ip, C.POINTER(C.c_int32)]
        L.osiv_get_plan.argtypes = [vp, ip, ip, C.POINTER(C.c_int32)]
        L.osiv_set_profiling.argtypes = [vp, ip]
        L.osiv_get_profile.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_int64), C.POINTER(C.c_double),
                                       C.POINTER(C.c_int64)]
        L.osiv_forward.argtypes = [vp, vp, vp, ip, ip, ip, vp]
        L.osiv_backward.argtypes = [vp, vp, vp, ip, ip, ip, vp]
        L.osiv_tv_gradient.argtypes = [vp, vp, vp, ip, C.c_double, vp]
        L.osiv_tv_gradient_static.argtypes = [vp, vp, vp, ip, C.c_double, vp]
        L.osiv_reconstruct.argtypes = [vp, vp, vp, C.c_float, C.POINTER(_CParams), ip, vp, vp, vp]
        L.osiv_reconstruct_host.argtypes = [vp, vp, vp, C.c_float, C.POINTER(_CParams), ip, vp, vp, vp]
        L.osiv_probe_peaks.argtypes = [ip, C.POINTER(C.c_double)]
        L.osiv_debug_timeline.argtypes = [vp, ip]
        L.osiv_debug_checks.argtypes = [vp]
        _lib = L
    return _lib


def version() -> int:
    return lib().osiv_version()


PROBE_FIELDS = ("ffma_tflops", "ffma2_tflops", "issue_ginst_per_s", "l2_read_gbs", "smem_read_gbs", "l1_read_gbs",
                "l1_read_b32_gbs", "sms")


def debug_checks() -> dict:
    """osiv_debug_checks: {violations, first_site, checks} of the checked build (raises OsivError in the regular build)"""
    out = (C.c_uint64 * 3)()
    _check(lib().osiv_debug_checks(out), "osiv_debug_checks")
    return {"violations": int(out[0]), "first_site": int(out[1]), "checks": int(out[2])}


def probe_peaks(device: int = 0) -> dict:
    """osiv_probe_peaks: measured FP32 / issue / L2 / shared-memory / L1 peaks of `device` (diagnostics)."""
    out = (C.c_double * 8)()
    _check(lib().osiv_probe_peaks(int(device), out), "osiv_probe_peaks")
    return dict(zip(PROBE_FIELDS, (float(v) for v in out)))


def strerror(status: int) -> str:
    return lib().osiv_strerror(int(status)).decode()


def default_params() -> Params:
    cp = _CParams()
    _check(lib().osiv_default_params(C.byref(cp)), "osiv_default_params")
    return Params(beta=cp.beta, n_subsets=cp.n_subsets, n_iters=cp.n_iters, mu0=cp.mu0, lambda0=cp.lambda0,
                  lambda_up=cp.lambda_up, lambda_down=cp.lambda_down, lambda_min=cp.lambda_min, kappa=cp.kappa,
                  tv_eps=cp.tv_eps, return_best=cp.return_best, monitor_mode=cp.monitor_mode,
                  view_shift=cp.view_shift, tv_z=cp.tv_z)


def ray_table(geom: "Geometry"):
    """A0 setup on the host (no GPU): (rays [V][C][4] = {alpha, beta, g0, h}, views [V][2]) float32."""
    rays = np.zeros((geom.n_views, geom.n_channels, 4), dtype=np.float32)
    views = np.zeros((geom.n_views, 2), dtype=np.float32)
    cg = geom.c()
    _check(lib().osiv_ray_table(C.byref(cg), rays.ctypes.data, views.ctypes.data), "osiv_ray_table")
    return rays, views


def _check(status: int, where: str) -> None:
    if status != OSIV_OK:
        raise OsivError(status, where)


def _stream() -> int:
    import torch
    return int(torch.cuda.current_stream().cuda_stream)


def _dev(t, shape, name: str) -> int:
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError(f"{name}: expected a contiguous float32 CUDA tensor")
    if tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: expected shape {tuple(shape)}, got {tuple(t.shape)}")
    return t.data_ptr()


def _cparams(p: Params):
    forced = None
    fptr = None
    if p.forced_lambda is not None:
        forced = np.ascontiguousarray(p.forced_lambda, dtype=np.float64)
        if forced.shape != (p.n_iters,):
            raise ValueError("forced_lambda must have n_iters entries")
        fptr = forced.ctypes.data_as(C.POINTER(C.c_double))
    cp = _CParams(p.beta, p.n_subsets, p.n_iters, p.mu0, p.lambda0, p.lambda_up, p.lambda_down, p.lambda_min,
                  p.kappa, p.tv_eps, p.return_best, p.monitor_mode, p.view_shift, 0, p.tv_z, fptr)
    return cp, forced


class Handle:
    """osiv_handle: geometry tables and workspace on one CUDA device."""

    def __init__(self, geom: Geometry, max_batch: int = 1, device: int = 0):
        self.geom = geom
        self.max_batch = max_batch
        self._h = C.c_void_p()
        cg = geom.c()
        _check(lib().osiv_create(C.byref(cg), max_batch, device, C.byref(self._h)), "osiv_create")
        self.device = device

    def close(self) -> None:
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().osiv_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- small queries --
    def dgamma(self) -> float:
        out = C.c_double()
        _check(lib().osiv_get_dgamma(self._h, C.byref(out)), "osiv_get_dgamma")
        return out.value

    def tau(self, n_subsets: int, kappa: float = 100.0) -> float:
        out = C.c_double()
        _check(lib().osiv_get_tau(self._h, n_subsets, kappa, C.byref(out)), "osiv_get_tau")
        return out.value

    def launch_count(self) -> int:
        return int(lib().osiv_launch_count(self._h))

    def set_symmetry(self, enable: bool) -> None:
        """enable=False forces the general (NS = 1) kernels even where the quarter-turn path applies"""
        _check(lib().osiv_set_symmetry(self._h, 1 if enable else 0), "osiv_set_symmetry")

    def set_overlap(self, enable: bool) -> None:
        """enable=False chains K1 and K2 in plain stream order instead of programmatic dependent launches"""
        _check(lib().osiv_set_overlap(self._h, 1 if enable else 0), "osiv_set_overlap")

    def set_graph(self, enable: bool) -> None:
        """enable=False enqueues every launch of reconstruct from the host instead of replaying a captured CUDA graph"""
        _check(lib().osiv_set_graph(self._h, 1 if enable else 0), "osiv_set_graph")

    def graph_replays(self) -> int:
        return int(lib().osiv_graph_replays(self._h))

    def set_back_kernel(self, general_only: bool = False, staged_rounds: bool = False) -> None:
        """general_only=True forces the general gather K2 where the shared-memory-staged K2 would run; staged_rounds=True
        lets the staged K2 also take subsets that need several staging rounds (by default the general kernel takes those)"""
        _check(lib().osiv_set_back_kernel(self._h, 1 if general_only else 2 if staged_rounds else 0), "osiv_set_back_kernel")

    def back_kernel(self, n_subsets: int = 0, batch: int = 1) -> str:
        """'staged' or 'general': the K2 that reconstruct / backward would run"""
        out = C.c_int32()
        _check(lib().osiv_get_back_kernel(self._h, n_subsets, batch, C.byref(out)), "osiv_get_back_kernel")
        return "staged" if out.value else "general"

    def plan(self, n_subsets: int = 0, batch: int = 1) -> dict:
        out = (C.c_int32 * 8)()
        _check(lib().osiv_get_plan(self._h, n_subsets, batch, out), "osiv_get_plan")
        keys = ("k1_orbit", "k1_split", "k1_blocks", "k1_threads", "k2_orbit", "k2_split", "k2_blocks", "k2_threads")
        return dict(zip(keys, [int(x) for x in out]))

    def set_profiling(self, enable: bool) -> None:
        _check(lib().osiv_set_profiling(self._h, 1 if enable else 0), "osiv_set_profiling")

    def get_profile(self):
        """(ms_forward, n_forward, ms_back, n_back) accumulated by profiled osiv_reconstruct calls"""
        a, b = C.c_double(), C.c_double()
        na, nb = C.c_int64(), C.c_int64()
        _check(lib().osiv_get_profile(self._h, C.byref(a), C.byref(na), C.byref(b), C.byref(nb)), "osiv_get_profile")
        return a.value, na.value, b.value, nb.value

    def n_subset_views(self, subset: int, n_subsets: int) -> int:
        return self.geom.n_views if subset < 0 else self.geom.n_views // n_subsets

    # -- compute calls (device tensors in, device tensors out) --
    def forward(self, img, subset: int = -1, n_subsets: int = 1, out=None):
        import torch
        g = self.geom
        batch = img.shape[0]
        ip = _dev(img, (batch, g.ny, g.nx), "img")
        vs = self.n_subset_views(subset, n_subsets)
        if out is None:
            out = torch.empty((batch, vs, g.n_channels), dtype=torch.float32, device=img.device)
        op = _dev(out, (batch, vs, g.n_channels), "out")
        _check(lib().osiv_forward(self._h, ip, op, batch, subset, n_subsets, _stream()), "osiv_forward")
        return out

    def backward(self, sino, subset: int = -1, n_subsets: int = 1, out=None):
        import torch
        g = self.geom
        batch = sino.shape[0]
        vs = self.n_subset_views(subset, n_subsets)
        sp = _dev(sino, (batch, vs, g.n_channels), "sino")
        if out is None:
            out = torch.empty((batch, g.ny, g.nx), dtype=torch.float32, device=sino.device)
        op = _dev(out, (batch, g.ny, g.nx), "out")
        _check(lib().osiv_backward(self._h, sp, op, batch, subset, n_subsets, _stream()), "osiv_backward")
        return out

    def tv_gradient(self, img, tv_eps: float = 1e-5, out=None):
        import torch
        g = self.geom
        batch = img.shape[0]
        ip = _dev(img, (batch, g.ny, g.nx), "img")
        if out is None:
            out = torch.empty_like(img)
        op = _dev(out, (batch, g.ny, g.nx), "out")
        _check(lib().osiv_tv_gradient(self._h, ip, op, batch, tv_eps, _stream()), "osiv_tv_gradient")
        return out

    def tv_gradient_static(self, img, out, tv_eps: float = 1e-5):
        """osiv_tv_gradient_static: the same gradient with its scratch in the library's fixed device array; nothing is
        allocated, here or in the library, so `out` is required.  Raises OsivError(SCRATCH_LIMIT) beyond
        STATIC_SCRATCH_BYTES.  Calls that overlap on the GPU race on the shared array."""
        g = self.geom
        batch = img.shape[0]
        ip = _dev(img, (batch, g.ny, g.nx), "img")
        op = _dev(out, (batch, g.ny, g.nx), "out")
        _check(lib().osiv_tv_gradient_static(self._h, ip, op, batch, tv_eps, _stream()), "osiv_tv_gradient_static")
        return out

    def reconstruct(self, counts, blank, params: Params, out=None, trace: bool = False):
        """counts [batch][V][C] CUDA float32; blank: python scalar or CUDA float32 [C].
        Returns the image tensor, or (image, trace ndarray [batch][n_iters][2]) when trace=True
        (which synchronises and raises OsivError(NOT_FINITE) if the monitor blew up)."""
        import torch
        g = self.geom
        batch = counts.shape[0]
        cp_ = _dev(counts, (batch, g.n_views, g.n_channels), "counts")
        if isinstance(blank, (int, float)):
            bp, bs = None, float(blank)
        else:
            bp, bs = _dev(blank, (g.n_channels,), "blank"), 0.0
        if out is None:
            out = torch.empty((batch, g.ny, g.nx), dtype=torch.float32, device=counts.device)
        op = _dev(out, (batch, g.ny, g.nx), "out")
        cp, keep = _cparams(params)
        tr = np.zeros((batch, params.n_iters, 2), dtype=np.float64) if trace else None
        tp = tr.ctypes.data if trace else None
        _check(lib().osiv_reconstruct(self._h, cp_, bp, bs, C.byref(cp), batch, op, tp, _stream()), "osiv_reconstruct")
        del keep
        return (out, tr) if trace else out

    def reconstruct_host(self, counts, blank, params: Params, out=None, trace: bool = False):
        """End-to-end call on HOST buffers: counts is a float32 numpy array or CPU (ideally pinned) torch
        tensor [batch][V][C]; the result is written to `out` (same kinds) and the stream is synchronised."""
        import torch
        g = self.geom

        def host_ptr(a, shape, name):
            if isinstance(a, torch.Tensor):
                if a.is_cuda or a.dtype != torch.float32 or not a.is_contiguous() or tuple(a.shape) != tuple(shape):
                    raise TypeError(f"{name}: expected a contiguous float32 CPU tensor of shape {shape}")
                return a.data_ptr()
            if not (isinstance(a, np.ndarray) and a.dtype == np.float32 and a.flags["C_CONTIGUOUS"]
                    and a.shape == tuple(shape)):
                raise TypeError(f"{name}: expected a contiguous float32 array of shape {shape}")
            return a.ctypes.data

        batch = counts.shape[0]
        cp_ = host_ptr(counts, (batch, g.n_views, g.n_channels), "counts")
        if isinstance(blank, (int, float)):
            bp, bs = None, float(blank)
        else:
            bp, bs = host_ptr(blank, (g.n_channels,), "blank"), 0.0
        if out is None:
            out = np.empty((batch, g.ny, g.nx), dtype=np.float32)
        op = host_ptr(out, (batch, g.ny, g.nx), "out")
        cp, keep = _cparams(params)
        tr = np.zeros((batch, params.n_iters, 2), dtype=np.float64) if trace else None
        tp = tr.ctypes.data if trace else None
        _check(lib().osiv_reconstruct_host(self._h, cp_, bp, bs, C.byref(cp), batch, op, tp, _stream()),
               "osiv_reconstruct_host")
        del keep
        return (out, tr) if trace else out
