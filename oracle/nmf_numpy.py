"""Second, independent fp64 formulation of Eq. 3 -- TEST INFRASTRUCTURE ONLY.

Dense-matrix numpy transcription of PAPER.md:48-50 (Eq. 3) exactly as typeset:
whole-matrix products and Hadamard products, no loops over pixels.  It exists
only to cross-check the C loop oracle at small sizes (pin P12).
Missing data (Omega == 0) is removed with np.where *before* any product so that
NaN/Inf there cannot propagate (reading G5).
"""
from __future__ import annotations

import numpy as np

EPS = 1e-30


def _masked(X, Omega):
    Om = np.asarray(Omega, dtype=np.float64)
    live = Om > 0
    Xc = np.where(live, np.asarray(X, dtype=np.float64), 0.0)
    return np.where(live, Om, 0.0), Xc


def h_step(X, Omega, W, H):
    Om, Xc = _masked(X, Omega)
    num = W.T @ (Om * Xc)            # W^T (V o X)
    den = W.T @ (Om * (W @ H))       # W^T [V o (WH)]
    return H * num / np.maximum(den, EPS)


def w_step(X, Omega, W, H):
    Om, Xc = _masked(X, Omega)
    num = (Om * Xc) @ H.T            # (V o X) H^T
    den = (Om * (W @ H)) @ H.T       # [V o (WH)] H^T
    return W * num / np.maximum(den, EPS)


def objective(X, Omega, W, H):
    Om, Xc = _masked(X, Omega)
    return float(np.sum(Om * (Xc - W @ H) ** 2))


def fit(X, Omega, W0, H0, iters):
    W = np.array(W0, dtype=np.float64)
    H = np.array(H0, dtype=np.float64)
    for _ in range(iters):
        H = h_step(X, Omega, W, H)
        W = w_step(X, Omega, W, H)
    return W, H
