"""T1 at FULL size and FULL iteration count: the CUDA path (through the binding -> C-ABI) against stored fp64 oracle
results for the configs the oracle cannot recompute inside a test run: STIS-shaped 200 it, every K of the component
sweep (200 it each) and the 64-problem survey batch (300 it).

The stored values (tests/golden/fullsize_*.npz) are written by tests/golden/make_fullsize_goldens.py, which calls only
oracle/ and the seeded generators; nothing in them comes from the CUDA path.  A case whose file has not been generated
is skipped.  Tolerances are BASELINE.json's (gpu_util): rel. Frobenius <= 1e-3 on W, H, coef; rel. objective <= 1e-5
with both objectives evaluated by the oracle in fp64; beside the Frobenius figure every sampled H column is checked
on its own (max-abs difference scaled by the column's norm), so that an error confined to a few pixels cannot hide
in the norm of the whole matrix.
"""
import os

import numpy as np
import pytest
import torch

from oracle import nmf_oracle as orc
from paper_2309_04623_b200 import inputs, nmf
from gpu_util import TOL_FACTOR, TOL_OBJECTIVE, dev, rel

pytestmark = pytest.mark.gpu

GOLD = os.path.join(os.path.dirname(__file__), "golden")
SWEEP_K = (1, 5, 10, 20, 50, 100)


def _load(case):
    path = os.path.join(GOLD, f"fullsize_{case}.npz")
    if not os.path.exists(path):
        pytest.skip(f"{os.path.basename(path)} not generated (python tests/golden/make_fullsize_goldens.py {case})")
    return np.load(path)


@pytest.fixture(scope="module")
def stis_lib():
    return inputs.make_stis()


def _columns_ok(Hg_c, Ho_c):
    """every sampled column on its own: max |dH| over the column <= tol * the column's 2-norm (columns that are
    exactly zero in the oracle -- fully masked pixels, G4 -- must be exactly zero on the device too)"""
    Ho_c = Ho_c.astype(np.float64); Hg_c = Hg_c.astype(np.float64)
    nrm = np.linalg.norm(Ho_c, axis=0)
    err = np.abs(Hg_c - Ho_c).max(axis=0)
    dead = nrm == 0
    assert np.all(Hg_c[:, dead] == 0)
    return float((err[~dead] / nrm[~dead]).max())


def _check_fit(p, g, variant=0):
    plan = nmf.Plan(p.N, p.P, p.K, max_targets=max(p.M, 1), variant=variant)
    X, Om, W, H = dev(p.X), dev(p.Omega), dev(p.W0), dev(p.H0)
    plan.fit(X, Om, W, H, int(g["iters"]))
    torch.cuda.synchronize()
    Wg, Hg = W.cpu().numpy(), H.cpu().numpy()
    assert np.all(np.isfinite(Wg)) and np.all(np.isfinite(Hg)) and Wg.min() >= 0 and Hg.min() >= 0
    cols = g["cols"]
    rw, rh = rel(Wg, g["W"]), rel(Hg[:, cols], g["Hc"])
    rc = _columns_ok(Hg[:, cols], g["Hc"])
    fg = orc.objective(p.X, p.Omega, Wg, Hg)             # fp64 oracle routine on the device's factors
    ro = abs(fg - float(g["f"])) / float(g["f"])
    assert rw <= TOL_FACTOR and rh <= TOL_FACTOR and rc <= TOL_FACTOR, (rw, rh, rc)
    assert ro <= TOL_OBJECTIVE, (ro, fg, float(g["f"]))
    return plan, H, Hg, dict(relW=rw, relH=rh, col=rc, relobj=ro)


def _check_projection(p, g, plan, Hd):
    """the stored science frames projected on the DEVICE's components and subtracted, against the oracle's
    projection on the oracle's components (the difference of the two H, ~1e-6, is part of what is compared)"""
    fr, cols = g["frames"], g["cols"]
    T, om, C = dev(p.T[fr]), dev(p.omega_t[fr]), dev(p.C0[fr])
    plan.project(Hd, T, om, C, int(g["proj_iters"]))
    out = plan.subtract(Hd, T, C, om, None, 0.0)
    torch.cuda.synchronize()
    Cg, outg = C.cpu().numpy(), out.cpu().numpy()
    rc = rel(Cg, g["coef"])
    live = p.omega_t[fr][:, cols] > 0
    dres = np.abs(outg[:, cols] - g["resid"])
    scale = np.abs(p.T[fr]).max()
    assert rc <= TOL_FACTOR, rc
    assert dres[live].max() <= TOL_FACTOR * scale, (dres[live].max(), scale)
    assert np.all(outg[:, cols][~live] == 0.0)
    return dict(relC=rc, resid=float(dres[live].max() / scale))


def test_stis_full_size_full_iterations(stis_lib):
    g = _load("stis")
    plan, Hd, Hg, r = _check_fit(stis_lib, g)
    r.update(_check_projection(stis_lib, g, plan, Hd))
    print("stis full size:", r)


@pytest.mark.parametrize("K", SWEEP_K)
def test_component_sweep_full_size(stis_lib, K):
    g = _load(f"sweep_K{K}")
    p = inputs.reinit(stis_lib, K, f"sweep_K{K}")
    plan, Hd, Hg, r = _check_fit(p, g)
    r.update(_check_projection(p, g, plan, Hd))
    print(f"sweep K={K} full size:", r)


def test_stis_fused_kernel_full_size(stis_lib):
    """the one-kernel-per-iteration tensor-core variant (3) at the metric's shape, same stored oracle result (the
    default is the split kernels, variant 4)"""
    g = _load("stis")
    _, _, _, r = _check_fit(stis_lib, g, variant=3)
    print("stis full size, fused kernel:", r)


def test_survey_batch_full_size():
    """64 problems x (128 frames, 256^2 px, K = 20) x 300 iterations in ONE batched launch sequence"""
    g = _load("survey")
    B = g["W"].shape[0]
    probs = inputs.make_survey(B)
    X, Om, W0, H0 = inputs.stack_batch(probs)
    p0 = probs[0]
    plan = nmf.Plan(p0.N, p0.P, p0.K, batch=B)
    Xd, Od, W, H = dev(X), dev(Om), dev(W0), dev(H0)
    plan.fit_batched(Xd, Od, W, H, int(g["iters"]))
    torch.cuda.synchronize()
    Wg, Hg = W.cpu().numpy(), H.cpu().numpy()
    worst = dict(relW=0.0, relH=0.0, col=0.0, relobj=0.0)
    for b in range(B):
        cols = g["cols"][b]
        fg = orc.objective(probs[b].X, probs[b].Omega, Wg[b], Hg[b])
        r = dict(relW=rel(Wg[b], g["W"][b]), relH=rel(Hg[b][:, cols], g["Hc"][b]),
                 col=_columns_ok(Hg[b][:, cols], g["Hc"][b]), relobj=abs(fg - float(g["f"][b])) / float(g["f"][b]))
        for k in worst:
            worst[k] = max(worst[k], r[k])
    assert worst["relW"] <= TOL_FACTOR and worst["relH"] <= TOL_FACTOR and worst["col"] <= TOL_FACTOR, worst
    assert worst["relobj"] <= TOL_OBJECTIVE, worst
    print("survey batch full size (worst of 64):", worst)
