"""Thin ctypes binding of include/nmf.h -- argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libnmf_b200.so; this
module passes torch device pointers, sizes and the current CUDA stream across
the C-ABI and owns nothing but the plan handle and its workspace tensor.  There
is no CPU fallback: a missing library or a non-CUDA tensor raises.

Names mirror the C entry points: Plan(N,P,K) ~ nmf_plan_create, Plan.fit ~ nmf_fit,
Plan.fit_batched, Plan.project ~ nmf_project, Plan.subtract ~ nmf_subtract,
Plan.objective ~ nmf_objective, Plan.fit_host / Plan.project_subtract_host.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnmf_b200.so")

SYMBOLS = (
    "nmf_plan_create", "nmf_plan_workspace_bytes", "nmf_plan_set_workspace", "nmf_plan_set_stream",
    "nmf_plan_set_variant", "nmf_plan_get_variant", "nmf_plan_destroy", "nmf_plan_staging_bytes", "nmf_plan_set_staging", "nmf_fit", "nmf_fit_batched",
    "nmf_project", "nmf_subtract", "nmf_objective", "nmf_fit_host", "nmf_project_subtract_host",
    "nmf_ref_distance", "nmf_ref_select", "nmf_fit_tol", "nmf_derotate_stack",
    "nmf_plan_launch_count", "nmf_status_string", "nmf_plan_last_cuda_error", "nmf_objective_static",
)

_lib = None
_vp, _ci, _cll, _cf = ctypes.c_void_p, ctypes.c_int, ctypes.c_longlong, ctypes.c_float


class NMFError(RuntimeError):
    def __init__(self, code: int, detail: str = ""):
        self.code = code
        msg = lib().nmf_status_string(code).decode()
        super().__init__(f"{msg}{(' -- ' + detail) if detail else ''}")


def lib():
    """Load libnmf_b200.so (fails loudly when the CUDA extension is missing)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2309_04623_b200.build` "
                              "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        L.nmf_plan_create.argtypes = [ctypes.POINTER(_vp), _ci, _cll, _ci, _ci, _ci]
        L.nmf_plan_workspace_bytes.argtypes = [_vp]; L.nmf_plan_workspace_bytes.restype = ctypes.c_size_t
        L.nmf_plan_set_workspace.argtypes = [_vp, _vp, ctypes.c_size_t]
        L.nmf_plan_staging_bytes.argtypes = [_vp, _ci]; L.nmf_plan_staging_bytes.restype = ctypes.c_size_t
        L.nmf_plan_set_staging.argtypes = [_vp, _vp, ctypes.c_size_t]
        L.nmf_plan_set_stream.argtypes = [_vp, _vp]
        L.nmf_plan_set_variant.argtypes = [_vp, _ci]
        L.nmf_plan_get_variant.argtypes = [_vp]
        L.nmf_plan_destroy.argtypes = [_vp]
        L.nmf_fit.argtypes = [_vp, _vp, _vp, _vp, _vp, _ci]
        L.nmf_fit_batched.argtypes = [_vp, _vp, _vp, _vp, _vp, _ci]
        L.nmf_project.argtypes = [_vp, _vp, _vp, _vp, _vp, _ci, _ci]
        L.nmf_subtract.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _cf, _vp, _ci]
        L.nmf_objective.argtypes = [_vp, _vp, _vp, _vp, _vp, ctypes.POINTER(ctypes.c_double)]
        L.nmf_ref_distance.argtypes = [_vp, _vp, _vp, _vp, _vp, _ci, _vp]
        L.nmf_ref_select.argtypes = [_vp, _vp, _ci, _ci, _vp]
        L.nmf_fit_tol.argtypes = [_vp, _vp, _vp, _vp, _vp, _ci, _ci, ctypes.c_double, ctypes.POINTER(_ci),
                                  ctypes.POINTER(ctypes.c_double)]
        L.nmf_derotate_stack.argtypes = [_vp, _vp, _vp, _vp, _ci, _ci, _cf, _vp, _vp, _ci]
        L.nmf_fit_host.argtypes = [_vp, _vp, _vp, _vp, _vp, _ci]
        L.nmf_project_subtract_host.argtypes = [_vp, _vp, _vp, _vp, _vp, _cf, _vp, _ci, _ci]
        L.nmf_plan_launch_count.argtypes = [_vp]; L.nmf_plan_launch_count.restype = _cll
        L.nmf_status_string.argtypes = [_ci]; L.nmf_status_string.restype = ctypes.c_char_p
        L.nmf_plan_last_cuda_error.argtypes = [_vp]; L.nmf_plan_last_cuda_error.restype = ctypes.c_char_p
        L.nmf_objective_static.argtypes = [_vp, _vp, _vp, _vp, _ci, _cll, _ci, _vp, _vp]
        _lib = L
    return _lib


def _dev(t: torch.Tensor, shape=None) -> int:
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError("expected a contiguous float32 CUDA tensor")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"expected shape {tuple(shape)}, got {tuple(t.shape)}")
    return t.data_ptr()


def _host(t: torch.Tensor, shape=None) -> int:
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError("expected a contiguous float32 host tensor")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"expected shape {tuple(shape)}, got {tuple(t.shape)}")
    return t.data_ptr()


STATIC_MAX_P = 4194304      # NMF_STATIC_MAX_P of include/nmf.h


def objective_static(X, Omega, W, H, out) -> None:
    """nmf_objective_static: the cost of Eq. 2 into `out` (a float64 CUDA tensor of one element), enqueued on torch's
    current stream of the tensors' device.  No plan, no workspace; the library call allocates nothing (its scratch is a
    fixed 256 KB device array, P <= STATIC_MAX_P).  Calls that overlap on the GPU race on that scratch."""
    N, P = X.shape
    K = W.shape[1]
    if not (isinstance(out, torch.Tensor) and out.is_cuda and out.dtype == torch.float64 and out.numel() == 1):
        raise TypeError("expected a float64 CUDA tensor of one element")
    with torch.cuda.device(X.device):
        rc = lib().nmf_objective_static(_dev(X, (N, P)), _dev(Omega, (N, P)), _dev(W, (N, K)), _dev(H, (K, P)), N, P, K,
                                        out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    if rc != 0:
        raise NMFError(rc)


class Plan:
    """nmf_plan for problems of shape (N frames, P pixels, K components)."""

    def __init__(self, N: int, P: int, K: int, batch: int = 1, max_targets: int = 0,
                 device: Optional[torch.device] = None, variant: int = 0):
        self._h = _vp()
        self.N, self.P, self.K, self.batch, self.max_targets = N, P, K, batch, max_targets
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        with torch.cuda.device(self.device):
            rc = lib().nmf_plan_create(ctypes.byref(self._h), N, P, K, batch, max_targets)
        if rc:
            self._h = _vp()
            raise NMFError(rc)
        nbytes = lib().nmf_plan_workspace_bytes(self._h)
        self.workspace = torch.empty(max(nbytes, 16), dtype=torch.uint8, device=self.device)
        self._check(lib().nmf_plan_set_workspace(self._h, self.workspace.data_ptr(), self.workspace.numel()))
        if variant:
            self._check(lib().nmf_plan_set_variant(self._h, variant))

    def use_own_staging(self, M: int = 0):
        """Allocate the staging of fit_host / project_subtract_host as a torch tensor owned by this object and hand it
        to the library (nmf_plan_set_staging), so that the library allocates no device memory on its own."""
        nbytes = lib().nmf_plan_staging_bytes(self._h, max(M, self.max_targets))
        self.staging = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self._check(lib().nmf_plan_set_staging(self._h, self.staging.data_ptr(), nbytes))

    # -- plumbing ---------------------------------------------------------
    def _check(self, rc: int):
        if rc:
            raise NMFError(rc, lib().nmf_plan_last_cuda_error(self._h).decode() if self._h else "")

    def _sync_stream(self):
        """Hand torch's current stream of the plan's device to the plan and make that device current (the library
        checks it: a plan only works with its own device current)."""
        if torch.cuda.current_device() != self.device.index:
            torch.cuda.set_device(self.device)
        self._check(lib().nmf_plan_set_stream(self._h, torch.cuda.current_stream(self.device).cuda_stream))

    @property
    def variant(self) -> int:
        return lib().nmf_plan_get_variant(self._h)

    @property
    def launch_count(self) -> int:
        return int(lib().nmf_plan_launch_count(self._h))

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().nmf_plan_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the calls of include/nmf.h ------------------------------------------
    def fit(self, X, Omega, W, H, iters: int):
        self._sync_stream()
        self._check(lib().nmf_fit(self._h, _dev(X, (self.N, self.P)), _dev(Omega, (self.N, self.P)),
                                  _dev(W, (self.N, self.K)), _dev(H, (self.K, self.P)), iters))

    def fit_tol(self, X, Omega, W, H, max_iters: int, check_every: int, tol: float):
        """nmf_fit_tol: fit with the tolerance stop.  Returns (iterations done, cost at the last check)."""
        done, f = _ci(0), ctypes.c_double(0.0)
        self._sync_stream()
        with torch.cuda.device(self.device):
            self._check(lib().nmf_fit_tol(self._h, _dev(X, (self.N, self.P)), _dev(Omega, (self.N, self.P)),
                                          _dev(W, (self.N, self.K)), _dev(H, (self.K, self.P)), max_iters,
                                          check_every, float(tol), ctypes.byref(done), ctypes.byref(f)))
        return done.value, f.value

    def derotate_stack(self, resid, omega, angle_deg, ny: int, nx: int, fill: float = 0.0, with_count: bool = False):
        """nmf_derotate_stack: rotate the M residual frames by angle_deg [M] and average the valid samples."""
        M = resid.shape[0]
        out = torch.empty(self.P, dtype=torch.float32, device=self.device)
        cnt = torch.empty(self.P, dtype=torch.int32, device=self.device) if with_count else None
        self._sync_stream()
        with torch.cuda.device(self.device):
            self._check(lib().nmf_derotate_stack(self._h, _dev(resid, (M, self.P)),
                                                 None if omega is None else _dev(omega, (M, self.P)),
                                                 _dev(angle_deg, (M,)), ny, nx, float(fill), out.data_ptr(),
                                                 None if cnt is None else cnt.data_ptr(), M))
        return (out, cnt) if with_count else out

    def fit_batched(self, X, Omega, W, H, iters: int):
        B = self.batch
        self._sync_stream()
        self._check(lib().nmf_fit_batched(self._h, _dev(X, (B, self.N, self.P)), _dev(Omega, (B, self.N, self.P)),
                                          _dev(W, (B, self.N, self.K)), _dev(H, (B, self.K, self.P)), iters))

    def project(self, H, target, omega, coef, iters: int):
        M = target.shape[0]
        self._sync_stream()
        self._check(lib().nmf_project(self._h, _dev(H, (self.K, self.P)), _dev(target, (M, self.P)),
                                      None if omega is None else _dev(omega, (M, self.P)),
                                      _dev(coef, (M, self.K)), M, iters))

    def subtract(self, H, target, coef, omega=None, factor=None, fill: float = 0.0, out=None):
        M = target.shape[0]
        if out is None:
            out = torch.empty_like(target)
        self._sync_stream()
        self._check(lib().nmf_subtract(self._h, _dev(H, (self.K, self.P)), _dev(target, (M, self.P)),
                                       _dev(coef, (M, self.K)),
                                       None if omega is None else _dev(omega, (M, self.P)),
                                       None if factor is None else _dev(factor, (M,)),
                                       float(fill), _dev(out, (M, self.P)), M))
        return out

    def ref_distance(self, target, omega_t, X, Omega, out=None):
        """nmf_ref_distance: masked squared Euclidean distances [M,N] (fp32, device) between M targets and X."""
        M = target.shape[0]
        if out is None:
            out = torch.empty((M, self.N), dtype=torch.float32, device=self.device)
        self._sync_stream()
        self._check(lib().nmf_ref_distance(self._h, _dev(target, (M, self.P)),
                                           None if omega_t is None else _dev(omega_t, (M, self.P)),
                                           _dev(X, (self.N, self.P)),
                                           None if Omega is None else _dev(Omega, (self.N, self.P)),
                                           M, _dev(out, (M, self.N))))
        return out

    def ref_select(self, dist, n_sel: int):
        """nmf_ref_select: int32 [M,n_sel] indices of the n_sel closest references per target."""
        M = dist.shape[0]
        idx = torch.empty((M, n_sel), dtype=torch.int32, device=self.device)
        self._sync_stream()
        self._check(lib().nmf_ref_select(self._h, _dev(dist, (M, self.N)), M, int(n_sel), idx.data_ptr()))
        return idx

    def objective(self, X, Omega, W, H) -> float:
        out = ctypes.c_double(0.0)
        self._sync_stream()
        self._check(lib().nmf_objective(self._h, _dev(X, (self.N, self.P)), _dev(Omega, (self.N, self.P)),
                                        _dev(W, (self.N, self.K)), _dev(H, (self.K, self.P)), ctypes.byref(out)))
        return out.value

    def fit_host(self, X, Omega, W, H, iters: int):
        """Host-buffer end-to-end fit (H2D + fit + D2H inside the call; synchronises)."""
        self._sync_stream()
        with torch.cuda.device(self.device):
            self._check(lib().nmf_fit_host(self._h, _host(X, (self.N, self.P)), _host(Omega, (self.N, self.P)),
                                           _host(W, (self.N, self.K)), _host(H, (self.K, self.P)), iters))

    def project_subtract_host(self, H_dev, target, omega, coef, out, iters: int, fill: float = 0.0):
        M = target.shape[0]
        self._sync_stream()
        with torch.cuda.device(self.device):
            self._check(lib().nmf_project_subtract_host(
                self._h, _dev(H_dev, (self.K, self.P)), _host(target, (M, self.P)),
                None if omega is None else _host(omega, (M, self.P)), _host(coef, (M, self.K)),
                float(fill), _host(out, (M, self.P)), M, iters))
