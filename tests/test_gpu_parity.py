"""T1: CUDA path vs fp64 oracle through the C-ABI, element by element, on the five
BASELINE.json configs (full size where the oracle finishes quickly, otherwise a
reduced size that still spans many tiles and a ragged tail, plus sampled checks at
full size).  Tolerances are BASELINE.json's: rel. Frobenius <= 1e-3, rel. objective <= 1e-5.
"""
import numpy as np
import pytest
import torch

from oracle import nmf_oracle as orc
from paper_2309_04623_b200 import inputs, nmf
from gpu_util import (TOL_FACTOR, check_fit_parity, check_project_subtract_parity, dev, gpu_fit, rel)

pytestmark = pytest.mark.gpu

VARIANTS = [1, 2, 3, 4]   # generic, fused FFMA, fused tensor-core kernel (K <= 64), split tensor-core kernels (K <= 128; the automatic choice except for launch-bound sizes)


@pytest.mark.parametrize("variant", VARIANTS + [5, 6])    # 5 = streaming FP32 kernel (K <= 8), 6 = resident kernel (one launch per fit)
def test_tiny_full(variant):
    p = inputs.make_tiny()
    r = check_fit_parity(p, p.iters, variant)
    check_project_subtract_parity(p, r["H"], r["plan"], p.proj_iters)


@pytest.mark.parametrize("variant", VARIANTS)
def test_miri_full(variant):
    p = inputs.make_miri()
    r = check_fit_parity(p, p.iters, variant)
    # no dead components (G17): column norms of W bounded away from 0
    assert np.linalg.norm(r["W"], axis=0).min() > 1e-20
    check_project_subtract_parity(p, r["H"], r["plan"], 100)


@pytest.mark.parametrize("variant", VARIANTS)
def test_stis_reduced_full_iterations(variant):
    """STIS-shaped generator at 200 frames x 192^2 px (1152 tiles of 32 px, wedge + bad pixels), K=50, 200 it."""
    p = inputs.make_stis(S=192, M=4)
    r = check_fit_parity(p, p.iters, variant)
    check_project_subtract_parity(p, r["H"], r["plan"], 100)


def test_stis_full_size_sampled():
    """Full 200 x 1024^2 x K=50 in bench.py's launch configuration: after 2 iterations every
    sampled H column (column-local update) and the whole W are checked against the oracle
    run on the same full-size inputs."""
    p = inputs.make_stis(M=1)
    Wg, Hg, plan = gpu_fit(p, 2)
    Wo, Ho = orc.fit(p.X, p.Omega, p.W0, p.H0, 2)
    assert rel(Wg, Wo) <= TOL_FACTOR
    rng = np.random.default_rng(0)
    cols = np.concatenate([rng.integers(0, p.P, 4096), np.arange(0, 64), np.arange(p.P - 64, p.P)])
    assert rel(Hg[:, cols], Ho[:, cols]) <= TOL_FACTOR
    assert rel(Hg, Ho) <= TOL_FACTOR
    fo = orc.objective(p.X, p.Omega, Wo, Ho); fg = orc.objective(p.X, p.Omega, Wg, Hg)
    assert abs(fg - fo) / fo <= 1e-5
    # device-side objective agrees with the oracle's
    fd = plan.objective(dev(p.X), dev(p.Omega), dev(Wg), dev(Hg))
    assert abs(fd - fg) / fg <= 1e-6


@pytest.mark.parametrize("K", inputs.SWEEP_KS)
def test_component_sweep_reduced(K):
    """Component sweep K in {1,5,10,20,50,100} on the STIS-shaped library at 200 x 96^2 px, 200 it."""
    p = inputs.make_sweep(K, S=96, M=4)
    r = check_fit_parity(p, p.iters, 0)
    check_project_subtract_parity(p, r["H"], r["plan"], 60)


@pytest.mark.parametrize("variant", VARIANTS)
def test_survey_batch_reduced(variant):
    """Survey batch: 6 independent problems (N=128, 64^2 px, K=20, 300 it) in one batched launch sequence."""
    probs = inputs.make_survey(B=6, S=64)
    X, Om, W0, H0 = inputs.stack_batch(probs)
    B, N, P = X.shape; K = W0.shape[2]
    plan = nmf.Plan(N, P, K, batch=B, variant=variant)
    Xd, Od, Wd, Hd = dev(X), dev(Om), dev(W0), dev(H0)
    plan.fit_batched(Xd, Od, Wd, Hd, probs[0].iters)
    torch.cuda.synchronize()
    Wg, Hg = Wd.cpu().numpy(), Hd.cpu().numpy()
    for b, p in enumerate(probs):
        Wo, Ho = orc.fit(p.X, p.Omega, p.W0, p.H0, p.iters)
        assert rel(Wg[b], Wo) <= TOL_FACTOR and rel(Hg[b], Ho) <= TOL_FACTOR
        fo = orc.objective(p.X, p.Omega, Wo, Ho); fg = orc.objective(p.X, p.Omega, Wg[b], Hg[b])
        assert abs(fg - fo) / fo <= 1e-5
    # a batched fit equals the same problems fitted one at a time (the pixel partitioning, hence the
    # fp32 summation order of the W half-step, depends on the batch size: equal to rounding, not bitwise)
    p = probs[3]
    W1, H1, _ = gpu_fit(p, p.iters, variant)
    assert rel(W1, Wg[3]) <= 1e-4 and rel(H1, Hg[3]) <= 1e-4


def test_objective_kernel_matches_oracle():
    p = inputs.make_miri(N=24, S=64, K=8, M=1)
    plan = nmf.Plan(p.N, p.P, p.K)
    f = plan.objective(dev(p.X), dev(p.Omega), dev(p.W0), dev(p.H0))
    fo = orc.objective(p.X, p.Omega, p.W0, p.H0)
    assert abs(f - fo) / fo <= 1e-12


def test_projection_omega_null_and_factor():
    p = inputs.make_tiny(M=3)
    _, H, plan = gpu_fit(p, 30)
    Hd, T, C = dev(H), dev(p.T), dev(p.C0)
    plan.project(Hd, T, None, C, 50)
    Co = orc.project(H, p.T, None, p.C0, 50)
    assert rel(C.cpu().numpy(), Co) <= TOL_FACTOR
    fac = np.array([0.0, 1.0, 0.5], dtype=np.float32)
    out = plan.subtract(Hd, T, C, None, dev(fac), 0.0).cpu().numpy()
    outo = orc.subtract(H, p.T, C.cpu().numpy(), None, fac)
    assert np.abs(out - outo).max() <= 1e-5 * np.abs(p.T).max()
    assert np.array_equal(out[0], p.T[0])


# ---- closest-frame reference selection ------------------------------------
def _check_ref_selection(T, ot, X, Om, n_sel, K=4):
    M, P = T.shape; N = X.shape[0]
    plan = nmf.Plan(N, P, K)
    d = lambda a: None if a is None else dev(a)
    Dg = plan.ref_distance(d(T), d(ot), d(X), d(Om))
    idx = plan.ref_select(Dg, n_sel)
    torch.cuda.synchronize()
    Dg, idx = Dg.cpu().numpy(), idx.cpu().numpy()
    Do = orc.ref_distance(T, ot, X, Om)
    assert np.all(np.isfinite(Dg))
    assert np.abs(Dg - Do).max() <= 1e-5 * np.abs(Do).max()           # fp32 partials, fp64 fixed-order reduce
    # the selection is an integer decision: bit-exact against the oracle's rule applied to the same fp32 distances
    assert np.array_equal(idx, orc.ref_select(Dg.astype(np.float64), n_sel))
    # and it is a valid answer for the fp64 distances: what it picks is as close as what the oracle picks
    pick = np.take_along_axis(Do, idx.astype(np.int64), axis=1)
    best = np.sort(Do, axis=1)[:, :n_sel]
    assert np.all(np.abs(pick - best) <= 2e-5 * np.abs(Do).max())
    return Dg, idx


@pytest.mark.parametrize("M,N,P", [(1, 1, 4), (5, 9, 36), (33, 130, 1028), (40, 200, 4100), (3, 256, 516)])
def test_ref_selection_ragged(M, N, P):
    rng = np.random.default_rng(M * 100 + N)
    T = (rng.random((M, P)) * 4).astype(np.float32)
    X = (rng.random((N, P)) * 4).astype(np.float32)
    ot = ((rng.random((M, P)) > 0.3) * (0.5 + rng.random((M, P)))).astype(np.float32)
    Om = ((rng.random((N, P)) > 0.2) * (0.5 + rng.random((N, P)))).astype(np.float32)
    if N > 2:
        X[N // 2] = T[0]                                   # the library contains target 0: it must come first
        Om[N // 2] = 1.0
    Dg, idx = _check_ref_selection(T, ot, X, Om, max(1, N // 3))
    if N > 2:
        assert idx[0, 0] == N // 2 and Dg[0, N // 2] == 0.0
    # garbage in masked entries changes nothing, bitwise
    T2, X2 = T.copy(), X.copy()
    T2[ot == 0] = np.nan; X2[Om == 0] = np.inf
    plan = nmf.Plan(N, P, 4)
    D2 = plan.ref_distance(dev(T2), dev(ot), dev(X2), dev(Om)).cpu().numpy()
    assert np.array_equal(D2, Dg)                          # also: run-to-run bitwise equal (fixed-order reduction)
    # NULL masks = all valid
    _check_ref_selection(T, None, X, None, 1)


def test_ref_selection_stis_shaped():
    """Science frames against the STIS-shaped library at 200 frames x 192^2 px: keep the closest 30 %."""
    p = inputs.make_stis(S=192, M=8)
    _check_ref_selection(p.T, p.omega_t, p.X, p.Omega, int(0.3 * p.N), K=p.K)


def test_ref_selection_full_size():
    """Full STIS-shaped library (200 frames x 1024^2 px), 4 science frames: every distance against the oracle."""
    p = inputs.make_stis(M=4)
    _check_ref_selection(p.T, p.omega_t, p.X, p.Omega, 60, K=p.K)
