"""Helpers shared by the GPU parity tests: run the CUDA path through the binding
(C-ABI) and the oracle on the same seeded inputs, and compare with the metrics
BASELINE.json states."""
import numpy as np
import torch

from oracle import nmf_oracle as orc
from paper_2309_04623_b200 import nmf

TOL_FACTOR = 1e-3      # relative Frobenius difference of W, H, coef, residual images (BASELINE.json)
TOL_OBJECTIVE = 1e-5   # relative objective difference, both evaluated in fp64 by the oracle


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def rel(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def gpu_fit(p, iters, variant=0, plan=None):
    plan = plan or nmf.Plan(p.N, p.P, p.K, max_targets=max(p.M, 1), variant=variant)
    X, Om, W, H = dev(p.X), dev(p.Omega), dev(p.W0), dev(p.H0)
    plan.fit(X, Om, W, H, iters)
    torch.cuda.synchronize()
    return W.cpu().numpy(), H.cpu().numpy(), plan


def check_fit_parity(p, iters, variant=0, tol_f=TOL_FACTOR, tol_o=TOL_OBJECTIVE):
    Wg, Hg, plan = gpu_fit(p, iters, variant)
    Wo, Ho = orc.fit(p.X, p.Omega, p.W0, p.H0, iters)
    rw, rh = rel(Wg, Wo), rel(Hg, Ho)
    fo = orc.objective(p.X, p.Omega, Wo, Ho)
    fg = orc.objective(p.X, p.Omega, Wg, Hg)
    ro = abs(fg - fo) / fo
    assert np.all(np.isfinite(Wg)) and np.all(np.isfinite(Hg))
    assert Wg.min() >= 0 and Hg.min() >= 0
    assert rw <= tol_f and rh <= tol_f, (rw, rh)
    assert ro <= tol_o, (ro, fg, fo)
    return dict(relW=rw, relH=rh, relobj=ro, W=Wg, H=Hg, Wo=Wo, Ho=Ho, plan=plan)


def check_project_subtract_parity(p, H32, plan, iters):
    """Projection + subtraction of p.T on fixed (GPU-fitted) components H32."""
    Hd, T, om, C = dev(H32), dev(p.T), dev(p.omega_t), dev(p.C0)
    plan.project(Hd, T, om, C, iters)
    out = plan.subtract(Hd, T, C, om, None, 0.0)
    torch.cuda.synchronize()
    Cg, outg = C.cpu().numpy(), out.cpu().numpy()
    Co = orc.project(H32, p.T, p.omega_t, p.C0, iters)
    outo = orc.subtract(H32, p.T, Co, p.omega_t, None, 0.0)
    live = p.omega_t > 0
    # the model c.H is what is unique when H is rank-deficient on omega>0 (G16): compare it and the residual
    model_g = p.T.astype(np.float64) - outg
    model_o = p.T.astype(np.float64) - outo
    rm = rel(model_g[live], model_o[live])
    rc = rel(Cg, Co)
    assert rm <= TOL_FACTOR, rm
    assert rc <= TOL_FACTOR, rc
    assert np.all(outg[~live] == 0.0)
    # residual images: absolute error relative to the target scale (residual itself is ~noise)
    assert np.abs(outg[live] - outo[live]).max() <= TOL_FACTOR * np.abs(p.T[live]).max()
    return dict(relC=rc, relmodel=rm)
