"""Seeded synthetic input generators (numpy only).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds
none of the method's arithmetic: no multiplicative update, no projection, no
objective.  It only synthesises PSF-like reference libraries X, weight/mask
matrices Omega, science frames and the seeded initial factors, with the shapes
and structure of BASELINE.json's five configs (the paper's own
data, §3, is not available and is not reconstructed).

Conventions (SURVEY.md "Notation", BASELINE.json orientation):
  X      [N, P] fp32 >= 0      reference library, P = S*S pixels, row-major
  Omega  [N, P] fp32 >= 0      0 = occulted / bad pixel, else inverse variance
  W0     [N, K] fp32 in [0.1,1)  initial coefficients   ("initialized randomly")
  H0     [K, P] fp32 in [0.1,1)  initial components
  T      [M, P] fp32           science frames; omega_t [M, P] their weights
  C0     [M, K] fp32 in [0.1,1)  initial projection coefficients
"""
from __future__ import annotations

import dataclasses
from typing import Optional

import numpy as np


@dataclasses.dataclass
class Problem:
    """One NMF problem instance: library + science frames + seeded init."""

    name: str
    N: int
    S: int
    K: int
    iters: int
    proj_iters: int
    X: np.ndarray
    Omega: np.ndarray
    W0: np.ndarray
    H0: np.ndarray
    T: np.ndarray
    omega_t: np.ndarray
    C0: np.ndarray

    @property
    def P(self) -> int:
        return self.S * self.S

    @property
    def M(self) -> int:
        return self.T.shape[0]


# --------------------------------------------------------------------------
# small helpers (image geometry, smoothing) -- data synthesis only
# --------------------------------------------------------------------------

def _grid(S: int):
    y, x = np.mgrid[0:S, 0:S]
    return x.astype(np.float64), y.astype(np.float64)


def _smooth_unit_field(rng: np.random.Generator, S: int, sigma_px: float) -> np.ndarray:
    """White unit-variance field, Gaussian-smoothed (periodic, via FFT) and
    re-normalised to unit variance.  'correlation 2 px' in BASELINE.json."""
    w = rng.standard_normal((S, S), dtype=np.float32)
    fy = np.fft.fftfreq(S)[:, None]
    fx = np.fft.rfftfreq(S)[None, :]
    tf = np.exp(-2.0 * (np.pi * sigma_px) ** 2 * (fx * fx + fy * fy)).astype(np.float32)
    g = np.fft.irfft2(np.fft.rfft2(w) * tf, s=(S, S)).astype(np.float32)
    g -= g.mean()
    g /= g.std()
    return g


def _ring(S: int, a_px: float, width_px: float, incl_deg: float, pa_deg: float) -> np.ndarray:
    """Inclined ring with Gaussian radial profile, peak 1, centred on S/2."""
    x, y = _grid(S)
    c = S // 2
    dx, dy = x - c, y - c
    pa = np.deg2rad(pa_deg)
    u = dx * np.cos(pa) + dy * np.sin(pa)
    v = (-dx * np.sin(pa) + dy * np.cos(pa)) / max(np.cos(np.deg2rad(incl_deg)), 1e-3)
    rr = np.sqrt(u * u + v * v)
    return np.exp(-0.5 * ((rr - a_px) / width_px) ** 2)


def _init_factors(rng: np.random.Generator, N: int, K: int, P: int, M: int):
    """Seeded U[0.1,1) init, drawn in fp32."""
    W0 = (0.1 + 0.9 * rng.random((N, K), dtype=np.float32)).astype(np.float32)
    H0 = (0.1 + 0.9 * rng.random((K, P), dtype=np.float32)).astype(np.float32)
    C0 = (0.1 + 0.9 * rng.random((max(M, 1), K), dtype=np.float32)).astype(np.float32)[:M]
    return W0, H0, C0


# --------------------------------------------------------------------------
# config "tiny"
# --------------------------------------------------------------------------

def make_tiny(N: int = 16, S: int = 64, K: int = 5, iters: int = 200, seed: int = 1001,
              noise: float = 0.01, M: int = 1, proj_iters: int = 200) -> Problem:
    """X = W0*H0 + |N(0, noise)|, H0 rows Gaussian blobs, centred r=6 occulter.
    `noise` is the standard deviation; noise=0 gives the exact rank-K library
    used by the recovery pin."""
    rng = np.random.default_rng(seed)
    P = S * S
    x, y = _grid(S)
    Wt = rng.random((N, K))
    Ht = np.empty((K, P))
    for k in range(K):
        sig = rng.uniform(3.0, 10.0) * S / 64.0
        cx, cy = rng.uniform(0, S, size=2)
        Ht[k] = np.exp(-0.5 * ((x - cx) ** 2 + (y - cy) ** 2) / sig ** 2).ravel()
    X = Wt @ Ht
    if noise > 0:
        X = X + np.abs(rng.normal(0.0, noise, size=X.shape))
    c = S // 2
    r_occ = 6.0 * S / 64.0
    mask = ((x - c) ** 2 + (y - c) ** 2 > r_occ ** 2).ravel()
    Omega = np.broadcast_to(mask.astype(np.float32), (N, P)).copy()
    # science frames: fresh mix + faint inclined ring (1 % of the frame peak)
    T = np.empty((M, P))
    for m in range(M):
        w = rng.random(K)
        t = w @ Ht
        if noise > 0:
            t = t + np.abs(rng.normal(0.0, noise, size=P))
        ring = _ring(S, 20.0 * S / 64.0, 2.0 * S / 64.0, 60.0, 30.0).ravel()
        T[m] = t + 0.01 * t.max() * ring
    omega_t = np.broadcast_to(mask.astype(np.float32), (M, P)).copy()
    W0, H0, C0 = _init_factors(rng, N, K, P, M)
    return Problem("tiny", N, S, K, iters, proj_iters, X.astype(np.float32), Omega,
                   W0, H0, T.astype(np.float32), omega_t, C0)


# --------------------------------------------------------------------------
# PSF + speckle generator shared by the MIRI-, STIS- and survey-shaped configs
# --------------------------------------------------------------------------

def _psf_frames(rng: np.random.Generator, n_frames: int, S: int, r0: float, F0: float,
                g_static: np.ndarray, read_var: float = 25.0):
    """I = F0*A*(1+r/r0)^-3 * exp(0.3 g - 0.045), g = sqrt(.8) g_static + sqrt(.2) g_n.
    Returns (noisy clipped frames, noiseless intensity) as fp32 [n, S*S]."""
    x, y = _grid(S)
    c = S // 2
    P = S * S
    Xo = np.empty((n_frames, P), dtype=np.float32)
    Io = np.empty((n_frames, P), dtype=np.float32)
    s8, s2 = np.float32(np.sqrt(0.8)), np.float32(np.sqrt(0.2))
    for n in range(n_frames):
        A = rng.uniform(0.8, 1.2)
        dx, dy = rng.uniform(-0.5, 0.5, size=2)
        r = np.sqrt((x - c - dx) ** 2 + (y - c - dy) ** 2)
        env = (F0 * A * (1.0 + r / r0) ** -3).astype(np.float32)
        g = s8 * g_static + s2 * _smooth_unit_field(rng, S, 2.0)
        I = env * np.exp(np.float32(0.3) * g - np.float32(0.045))
        noise = rng.standard_normal((S, S), dtype=np.float32) * np.sqrt(I + np.float32(read_var))
        Xo[n] = np.maximum(I + noise, 0.0).ravel()
        Io[n] = I.ravel()
    return Xo, Io


def _miri_mask(S: int, r_occ: float) -> np.ndarray:
    """False (masked) on r < r_occ about the un-shifted centre and on the 3-px
    four-quadrant cross |x-c|<=1 or |y-c|<=1."""
    x, y = _grid(S)
    c = S // 2
    m = ((x - c) ** 2 + (y - c) ** 2 >= r_occ ** 2) & (np.abs(x - c) > 1) & (np.abs(y - c) > 1)
    return m.ravel()


def make_miri(N: int = 96, S: int = 256, K: int = 30, iters: int = 500, seed: int = 2002,
              M: int = 8, r_occ: float = 10.0, F0: float = 1e5, r0: float = 4.0,
              proj_iters: int = 200, name: str = "miri") -> Problem:
    rng = np.random.default_rng(seed)
    P = S * S
    g_static = _smooth_unit_field(rng, S, 2.0)
    X, I = _psf_frames(rng, N, S, r0, F0, g_static)
    mask = _miri_mask(S, r_occ)
    Omega = np.where(mask[None, :], 1.0 / (I + 25.0), 0.0).astype(np.float32)
    T, It = _psf_frames(rng, M, S, r0, F0, g_static)
    omega_t = np.where(mask[None, :], 1.0 / (It + 25.0), 0.0).astype(np.float32)
    W0, H0, C0 = _init_factors(rng, N, K, P, M)
    return Problem(name, N, S, K, iters, proj_iters, X, Omega, W0, H0, T, omega_t, C0)


def _stis_mask(rng: np.random.Generator, S: int) -> np.ndarray:
    """False on the vertical occulting band (60 px wide at S=1024, scaled with S)
    and on one fixed 0.5 % random bad-pixel set shared by all frames."""
    x, _ = _grid(S)
    c = S // 2
    half = max(1, int(round(30 * S / 1024)))
    m = ~((x >= c - half) & (x < c + half))
    bad = rng.random((S, S)) < 0.005
    return (m & ~bad).ravel()


def make_stis(N: int = 200, S: int = 1024, K: int = 50, iters: int = 200, seed: int = 3003,
              M: int = 32, init_seed: Optional[int] = None, F0: float = 1e6, r0: float = 8.0,
              proj_iters: int = 200, name: str = "stis") -> Problem:
    """STIS-shaped library.  `init_seed` (3100+K for the component sweep) draws
    the initial factors from its own stream so the library is shared across K."""
    rng = np.random.default_rng(seed)
    P = S * S
    g_static = _smooth_unit_field(rng, S, 2.0)
    mask = _stis_mask(rng, S)
    X, I = _psf_frames(rng, N, S, r0, F0, g_static)
    Omega = np.where(mask[None, :], 1.0 / (I + 25.0), 0.0).astype(np.float32)
    del I
    T, It = _psf_frames(rng, M, S, r0, F0, g_static)
    omega_t = np.where(mask[None, :], 1.0 / (It + 25.0), 0.0).astype(np.float32)
    for m in range(M):
        incl = rng.uniform(30.0, 80.0)
        pa = rng.uniform(0.0, 180.0)
        ring = _ring(S, 150.0 * S / 1024.0, 10.0 * S / 1024.0, incl, pa).ravel()
        T[m] += (1e-4 * F0 * ring).astype(np.float32)
    rng_init = rng if init_seed is None else np.random.default_rng(init_seed)
    W0, H0, C0 = _init_factors(rng_init, N, K, P, M)
    return Problem(name, N, S, K, iters, proj_iters, X, Omega, W0, H0, T, omega_t, C0)


SWEEP_KS = (1, 5, 10, 20, 50, 100)


def make_sweep(K: int, N: int = 200, S: int = 1024, iters: int = 200, M: int = 32) -> Problem:
    """Component sweep: the STIS-shaped library refitted at K, init seed 3100+K."""
    return make_stis(N=N, S=S, K=K, iters=iters, seed=3003, M=M, init_seed=3100 + K,
                     name=f"sweep_K{K}")


def reinit(lib: Problem, K: int, name: str) -> Problem:
    """The sweep problem make_sweep(K) built from an already generated STIS-shaped library `lib` (same N, S, M):
    identical arrays, without regenerating the frames (the library draws do not depend on K)."""
    W0, H0, C0 = _init_factors(np.random.default_rng(3100 + K), lib.N, K, lib.P, lib.M)
    return dataclasses.replace(lib, name=name, K=K, W0=W0, H0=H0, C0=C0)


def make_survey_problem(b: int, N: int = 128, S: int = 256, K: int = 20, iters: int = 300,
                        M: int = 4) -> Problem:
    """Problem b of the survey batch: MIRI generator, seed 5000+b, occulter radius U[6,14]."""
    r_occ = float(np.random.default_rng(5000 + b).uniform(6.0, 14.0))
    return make_miri(N=N, S=S, K=K, iters=iters, seed=5000 + b, M=M, r_occ=r_occ,
                     name=f"survey_{b}")


def make_survey(B: int = 64, **kw):
    """The survey batch as a list of B independent problems of identical shape."""
    return [make_survey_problem(b, **kw) for b in range(B)]


def stack_batch(problems):
    """Stack a list of same-shape problems into [B,N,P], [B,N,K], [B,K,P] arrays."""
    f = lambda a: np.ascontiguousarray(np.stack([getattr(p, a) for p in problems]))
    return f("X"), f("Omega"), f("W0"), f("H0")


CONFIGS = {
    "tiny": make_tiny,
    "miri": make_miri,
    "stis": make_stis,
}
