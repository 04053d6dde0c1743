"""ctypes loader for oracle/nmf_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Builds liboracle.so with gcc next to the source on first use (or via
`python -m oracle.nmf_oracle`, which __graft_entry__.build() calls) and exposes
thin numpy wrappers.  fp32 inputs are up-cast exactly; all arithmetic is fp64
(SURVEY.md §8(c)).  See nmf_oracle.c for the passages each function follows.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nmf_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the C oracle (gcc, OpenMP).  Returns the library path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = f"{_LIB}.{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_F = ctypes.POINTER(ctypes.c_float)
_D = ctypes.POINTER(ctypes.c_double)


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_objective.restype = ctypes.c_double
        lib.oracle_objective.argtypes = [ctypes.c_int, ctypes.c_long, ctypes.c_int, _F, _F, _D, _D]
        lib.oracle_h_step.argtypes = [ctypes.c_int, ctypes.c_long, ctypes.c_int, _F, _F, _D, _D]
        lib.oracle_w_step.argtypes = [ctypes.c_int, ctypes.c_long, ctypes.c_int, _F, _F, _D, _D]
        lib.oracle_fit.argtypes = [ctypes.c_int, ctypes.c_long, ctypes.c_int, _F, _F, _D, _D,
                                   ctypes.c_int, _D]
        lib.oracle_project.argtypes = [ctypes.c_int, ctypes.c_long, ctypes.c_int, _D, _F, _F, _D,
                                       ctypes.c_int]
        lib.oracle_subtract.argtypes = [ctypes.c_int, ctypes.c_long, ctypes.c_int, _D, _F, _D, _F,
                                        _D, ctypes.c_double, _D]
        lib.oracle_fit_tol.restype = ctypes.c_int
        lib.oracle_fit_tol.argtypes = [ctypes.c_int, ctypes.c_long, ctypes.c_int, _F, _F, _D, _D,
                                       ctypes.c_int, ctypes.c_int, ctypes.c_double, _D, _D]
        lib.oracle_derotate_stack.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, _F, _F, _D,
                                              ctypes.c_double, _D, ctypes.POINTER(ctypes.c_int)]
        lib.oracle_ref_distance.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_long, _F, _F, _F, _F, _D]
        lib.oracle_ref_select.argtypes = [ctypes.c_int, ctypes.c_int, _D, ctypes.c_int, ctypes.POINTER(ctypes.c_int)]
        _lib = lib
    return _lib


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data_as(_F)


def _f64(a, copy=False):
    a = np.array(a, dtype=np.float64, order="C", copy=True) if copy else np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_D)


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def objective(X, Omega, W, H) -> float:
    """Eq. 2: sum_{Omega>0} Omega*(X-WH)^2, fp64."""
    X, xp = _f32(X); Om, op = _f32(Omega); W, wp = _f64(W); H, hp = _f64(H)
    N, P = X.shape; K = W.shape[1]
    assert Om.shape == (N, P) and W.shape == (N, K) and H.shape == (K, P)
    return float(_load().oracle_objective(N, P, K, xp, op, wp, hp))


def h_step(X, Omega, W, H):
    """One H half-step (Eq. 3 first line).  Returns the new H (fp64)."""
    X, xp = _f32(X); Om, op = _f32(Omega); W, wp = _f64(W); H, hp = _f64(H, copy=True)
    N, P = X.shape; K = W.shape[1]
    _load().oracle_h_step(N, P, K, xp, op, wp, hp)
    return H


def w_step(X, Omega, W, H):
    """One W half-step (Eq. 3 second line).  Returns the new W (fp64)."""
    X, xp = _f32(X); Om, op = _f32(Omega); W, wp = _f64(W, copy=True); H, hp = _f64(H)
    N, P = X.shape; K = W.shape[1]
    _load().oracle_w_step(N, P, K, xp, op, wp, hp)
    return W


def fit(X, Omega, W0, H0, iters: int, trace: bool = False):
    """iters x {H half-step; W half-step} from (W0,H0).  Returns (W, H[, trace])
    with trace = objective at start and after every half-step (2*iters+1)."""
    X, xp = _f32(X); Om, op = _f32(Omega); W, wp = _f64(W0, copy=True); H, hp = _f64(H0, copy=True)
    N, P = X.shape; K = W.shape[1]
    assert Om.shape == (N, P) and W.shape == (N, K) and H.shape == (K, P)
    tr = np.zeros(2 * iters + 1) if trace else None
    tp = tr.ctypes.data_as(_D) if trace else None
    _load().oracle_fit(N, P, K, xp, op, wp, hp, int(iters), tp)
    return (W, H, tr) if trace else (W, H)


def fit_tol(X, Omega, W0, H0, max_iters: int, check_every: int, tol: float):
    """Fit with the tolerance stop of reading G21.  Returns (W, H, iters_done, f_last, trace)
    with trace = [f_0, cost at every check made]."""
    X, xp = _f32(X); Om, op = _f32(Omega); W, wp = _f64(W0, copy=True); H, hp = _f64(H0, copy=True)
    N, P = X.shape; K = W.shape[1]
    assert Om.shape == (N, P) and W.shape == (N, K) and H.shape == (K, P) and check_every >= 1
    tr = np.full(max_iters // check_every + 1, np.nan)
    fl = ctypes.c_double(0.0)
    it = _load().oracle_fit_tol(N, P, K, xp, op, wp, hp, int(max_iters), int(check_every), float(tol),
                                ctypes.byref(fl), tr.ctypes.data_as(_D))
    return W, H, int(it), fl.value, tr[:it // check_every + 1]


def derotate_stack(R, omega, angles_deg, ny: int, nx: int, fill: float = 0.0):
    """Rotate the M frames R [M, ny*nx] by angles_deg (readings G22-G23) and average the valid samples (G24).
    Returns (stack [ny*nx] fp64, count [ny*nx] int32)."""
    R, rp = _f32(R)
    M, P = R.shape
    assert P == ny * nx
    op = None
    if omega is not None:
        om, op = _f32(omega)
    ang, ap = _f64(angles_deg)
    out = np.empty(P, dtype=np.float64)
    cnt = np.empty(P, dtype=np.int32)
    _load().oracle_derotate_stack(M, int(ny), int(nx), rp, op, ap, float(fill), out.ctypes.data_as(_D),
                                  cnt.ctypes.data_as(ctypes.POINTER(ctypes.c_int)))
    return out, cnt


def project(H, T, omega_t, C0, iters: int):
    """Non-negative projection of M frames on fixed H.  Returns C [M,K] fp64."""
    H, hp = _f64(H); T, tp = _f32(T); C, cp = _f64(C0, copy=True)
    M, P = T.shape; K = H.shape[0]
    if omega_t is None:
        op = None
    else:
        om, op = _f32(omega_t)
    _load().oracle_project(M, P, K, hp, tp, op, cp, int(iters))
    return C


def subtract(H, T, C, omega_t=None, factor=None, fill: float = 0.0):
    """out = T - factor*(C H); `fill` where omega_t == 0.  fp64 [M,P]."""
    H, hp = _f64(H); T, tp = _f32(T); C, cp = _f64(C)
    M, P = T.shape; K = H.shape[0]
    op = None
    if omega_t is not None:
        om, op = _f32(omega_t)
    fp = None
    if factor is not None:
        fac, fp = _f64(factor)
    out = np.empty((M, P), dtype=np.float64)
    _load().oracle_subtract(M, P, K, hp, tp, cp, op, fp, float(fill), out.ctypes.data_as(_D))
    return out


def ref_distance(T, omega_t, X, Omega):
    """Masked squared Euclidean distances D[m,n] between targets T [M,P] and references X [N,P] (fp64);
    pixels with omega_t[m,p] == 0 or Omega[n,p] == 0 are skipped."""
    T, tp = _f32(T); X, xp = _f32(X)
    M, P = T.shape; N = X.shape[0]
    otp = op = None
    if omega_t is not None:
        ot, otp = _f32(omega_t)
    if Omega is not None:
        om, op = _f32(Omega)
    D = np.empty((M, N), dtype=np.float64)
    _load().oracle_ref_distance(M, N, P, tp, otp, xp, op, D.ctypes.data_as(_D))
    return D


def ref_select(D, n_sel: int):
    """Indices [M,n_sel] of the n_sel closest references per target, ascending in (distance, index)."""
    D, dp = _f64(D)
    M, N = D.shape
    idx = np.full((M, n_sel), -1, dtype=np.int32)
    _load().oracle_ref_select(M, N, dp, int(n_sel), idx.ctypes.data_as(ctypes.POINTER(ctypes.c_int)))
    return idx


if __name__ == "__main__":
    print(build(force=True))
