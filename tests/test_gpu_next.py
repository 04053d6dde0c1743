"""CUDA path vs oracle for the section 8(f) NEXT rows built in round 2: tolerance-based stopping (NEXT-3, PAPER.md:53,
reading G21) and derotate + stack (NEXT-4, readings G22-G24)."""
import numpy as np
import pytest
import torch

from oracle import nmf_oracle as orc
from paper_2309_04623_b200 import inputs, nmf
from gpu_util import TOL_FACTOR, TOL_OBJECTIVE, dev, rel

pytestmark = pytest.mark.gpu


def _robust_tols(trace, m):
    """Tolerances that sit in the middle (geometrically) between two consecutive relative changes of the oracle's
    cost trace, so that the fp32 iterates of the CUDA path cannot flip the decision; returns [(tol, stop_iteration)]."""
    d = np.abs(trace[:-1] - trace[1:]) / trace[:-1]          # d[i]: change seen at check i + 1 (iteration (i + 1) m)
    out = []
    for i in range(1, len(d) - 1):
        # first check whose change falls below tol = sqrt(d[i] d[i+1]) must be i + 1 (changes before it are larger)
        tol = float(np.sqrt(d[i] * d[i + 1]))
        # fp32 iterates move the cost by ~1e-6 relative, i.e. a change d ~ 1e-3 by ~0.2 %: 1.5 % margins are safe
        if d[i + 1] < 0.97 * d[i] and np.all(d[:i + 1] > 1.015 * tol) and d[i + 1] > 2e-4:
            out.append((tol, (i + 2) * m))
    return out


@pytest.mark.parametrize("name,m", [("tiny", 1), ("tiny", 5), ("miri", 10)])
def test_fit_tol_stops_where_the_oracle_stops(name, m):
    p = inputs.make_tiny() if name == "tiny" else inputs.make_miri(S=128, M=1)
    max_iters = 120 if name == "tiny" else 200
    _, _, it0, _, trace = orc.fit_tol(p.X, p.Omega, p.W0, p.H0, max_iters, m, 0.0)
    assert it0 == max_iters
    cands = _robust_tols(trace, m)
    assert len(cands) >= 3
    plan = nmf.Plan(p.N, p.P, p.K)
    for tol, stop in (cands[0], cands[len(cands) // 2], cands[-1]):
        Wo, Ho, ito, fo, _ = orc.fit_tol(p.X, p.Omega, p.W0, p.H0, max_iters, m, tol)
        assert ito == stop
        X, Om, W, H = dev(p.X), dev(p.Omega), dev(p.W0), dev(p.H0)
        itg, fg = plan.fit_tol(X, Om, W, H, max_iters, m, tol)
        assert itg == ito, (tol, itg, ito)
        assert abs(fg - fo) / fo <= TOL_OBJECTIVE
        assert rel(W.cpu().numpy(), Wo) <= TOL_FACTOR and rel(H.cpu().numpy(), Ho) <= TOL_FACTOR
        # same iterates as the fixed-count fit of that many iterations, bitwise; and bitwise repeatable
        W2, H2 = dev(p.W0), dev(p.H0)
        plan.fit(X, Om, W2, H2, itg)
        assert torch.equal(W, W2) and torch.equal(H, H2)
        W3, H3 = dev(p.W0), dev(p.H0)
        assert plan.fit_tol(X, Om, W3, H3, max_iters, m, tol) == (itg, fg)
        assert torch.equal(W, W3) and torch.equal(H, H3)


def test_fit_tol_edge_cases():
    p = inputs.make_tiny()
    plan = nmf.Plan(p.N, p.P, p.K)
    X, Om = dev(p.X), dev(p.Omega)
    f0 = orc.objective(p.X, p.Omega, p.W0, p.H0)
    # tol = 0 never stops: identical to nmf_fit; max_iters not a multiple of check_every; no check at all
    for max_iters, m in ((23, 5), (4, 10), (0, 3)):
        W, H = dev(p.W0), dev(p.H0)
        it, f = plan.fit_tol(X, Om, W, H, max_iters, m, 0.0)
        assert it == max_iters
        W2, H2 = dev(p.W0), dev(p.H0)
        plan.fit(X, Om, W2, H2, max_iters)
        assert torch.equal(W, W2) and torch.equal(H, H2)
        if max_iters < m:
            assert abs(f - f0) / f0 <= 1e-12                  # cost of the initial factors (fp64 on the device)
    # a huge tolerance stops at the first check
    W, H = dev(p.W0), dev(p.H0)
    assert plan.fit_tol(X, Om, W, H, 50, 7, 10.0)[0] == 7
    L = nmf.lib()
    import ctypes
    done = ctypes.c_int(0)
    args = (plan._h, X.data_ptr(), Om.data_ptr(), W.data_ptr(), H.data_ptr())
    assert L.nmf_fit_tol(*args, 10, 0, 0.1, ctypes.byref(done), None) == -1        # check_every < 1
    assert L.nmf_fit_tol(*args, 10, 1, -0.1, ctypes.byref(done), None) == -1       # tol < 0
    assert L.nmf_fit_tol(*args, 10, 1, float("nan"), ctypes.byref(done), None) == -1
    assert L.nmf_fit_tol(*args, 10, 1, 0.1, None, None) == -1


def _check_derotate(R, om, ang, ny, nx, fill):
    M = R.shape[0]
    plan = nmf.Plan(4, ny * nx, 2)
    out, cnt = plan.derotate_stack(dev(R), None if om is None else dev(om), dev(np.asarray(ang, dtype=np.float32)), ny, nx,
                                   fill, with_count=True)
    torch.cuda.synchronize()
    out, cnt = out.cpu().numpy(), cnt.cpu().numpy()
    oo, co = orc.derotate_stack(R, om, np.asarray(ang, dtype=np.float32).astype(np.float64), ny, nx, fill)
    assert np.array_equal(cnt, co)                            # which frames contribute is an integer decision: exact
    live = co > 0
    scale = np.abs(R[np.isfinite(R)]).max()
    assert np.abs(out[live] - oo[live]).max() <= 1e-5 * scale
    assert np.all(out[~live] == np.float32(fill))
    return out, cnt


@pytest.mark.parametrize("ny,nx,M", [(1, 4, 1), (9, 9, 3), (33, 36, 5), (100, 68, 130), (260, 256, 7)])
def test_derotate_stack_ragged(ny, nx, M):
    if (ny * nx) % 4:
        pytest.skip("P % 4 != 0 is rejected at plan creation")
    rng = np.random.default_rng(ny * 100 + nx)
    R = (rng.random((M, ny * nx)) * 20 - 5).astype(np.float32)
    om = (rng.random((M, ny * nx)) > 0.1).astype(np.float32) * (0.5 + rng.random((M, ny * nx))).astype(np.float32)
    ang = rng.uniform(-360, 360, M)
    ang[0] = 90.0
    if M > 2:
        ang[1], ang[2] = 0.0, -180.0
    R[om == 0] = np.nan                                       # masked pixels hold garbage
    _check_derotate(R, om, ang, ny, nx, -3.0)
    Rf = np.nan_to_num(R, nan=1.0)
    _check_derotate(Rf, None, ang, ny, nx, 0.0)


def test_derotate_quarter_turns_exact_on_device():
    """Multiples of 90 degrees move pixels exactly on the device too.  Even side n: the centre is the pixel
    (n/2, n/2) (G22), so +90 degrees gives out[y, x] = in[n - x, y] for x >= 1 and -90 degrees out[y, x] = in[x, n - y]
    for y >= 1; column / row 0 has no source inside the image and is filled (oracle pin P20b)."""
    n = 64
    rng = np.random.default_rng(0)
    R = rng.random((1, n * n)).astype(np.float32)
    plan = nmf.Plan(4, n * n, 2)
    img = R[0].reshape(n, n)
    rot = lambda a: plan.derotate_stack(dev(R), None, dev(np.array([a], dtype=np.float32)), n, n, -1.0).cpu().numpy().reshape(n, n)
    assert np.array_equal(rot(0.0), img) and np.array_equal(rot(360.0), img) and np.array_equal(rot(-720.0), img)
    o = rot(90.0)
    assert np.array_equal(o[:, 1:], np.rot90(img[1:, :], k=-1)) and np.all(o[:, 0] == -1.0)
    o = rot(-90.0)
    assert np.array_equal(o[1:, :], np.rot90(img[:, 1:], k=1)) and np.all(o[0, :] == -1.0)
    o = rot(180.0)
    assert np.array_equal(o[1:, 1:], img[1:, 1:][::-1, ::-1]) and np.all(o[0, :] == -1.0) and np.all(o[:, 0] == -1.0)


def test_derotate_stack_full_size():
    """32 residual frames of 1024 x 1024 (the STIS-shaped science-frame count): every pixel against the oracle."""
    n, M = 1024, 32
    rng = np.random.default_rng(9)
    R = rng.standard_normal((M, n * n), dtype=np.float32) * 30
    om = np.ones((M, n * n), dtype=np.float32)
    om[:, :].reshape(M, n, n)[:, :, n // 2 - 30:n // 2 + 30] = 0     # the occulting band of the STIS-shaped config
    om[rng.random((M, n * n)) < 0.005] = 0
    R[om == 0] = np.inf
    ang = rng.uniform(0, 180, M)
    out, cnt = _check_derotate(R, om, ang, n, n, 0.0)
    assert cnt.max() == M and cnt.min() < M
