"""T2: properties of the CUDA path that hold at any size (no oracle run needed) and the
degenerate / ragged / error cases of the boundary."""
import ctypes

import numpy as np
import pytest
import torch

from oracle import nmf_oracle as orc
from paper_2309_04623_b200 import inputs, nmf
from gpu_util import TOL_FACTOR, check_fit_parity, dev, gpu_fit, rel

pytestmark = pytest.mark.gpu
VARIANTS = [1, 2, 3, 4]   # generic, fused FFMA, fused tensor-core kernel (K <= 64), split tensor-core kernels (K <= 128; the automatic choice except for launch-bound sizes)


@pytest.mark.parametrize("variant", VARIANTS)
def test_bitwise_determinism_and_resume(variant):
    p = inputs.make_miri(N=40, S=96, K=12, M=1)
    W1, H1, plan = gpu_fit(p, 40, variant)
    W2, H2, _ = gpu_fit(p, 40, variant, plan)
    assert np.array_equal(W1, W2) and np.array_equal(H1, H2)
    # checkpoint/resume: 20 + 20 iterations == 40 iterations, bitwise
    X, Om, W, H = dev(p.X), dev(p.Omega), dev(p.W0), dev(p.H0)
    plan.fit(X, Om, W, H, 20); plan.fit(X, Om, W, H, 20)
    torch.cuda.synchronize()
    assert np.array_equal(W.cpu().numpy(), W1) and np.array_equal(H.cpu().numpy(), H1)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("garbage", [np.nan, 1e30, np.inf])
def test_mask_invariance_bitwise(variant, garbage):
    """Entries with Omega == 0 must not influence anything, even NaN/Inf."""
    p = inputs.make_miri(N=32, S=64, K=10, M=2)
    W1, H1, plan = gpu_fit(p, 25, variant)
    q = inputs.make_miri(N=32, S=64, K=10, M=2)
    q.X[q.Omega == 0] = garbage
    W2, H2, _ = gpu_fit(q, 25, variant, plan)
    assert np.array_equal(W1, W2) and np.array_equal(H1, H2)
    q.T[q.omega_t == 0] = garbage
    Hd = dev(H1)
    C1, C2 = dev(p.C0), dev(p.C0)
    plan.project(Hd, dev(p.T), dev(p.omega_t), C1, 20)
    plan.project(Hd, dev(q.T), dev(q.omega_t), C2, 20)
    assert torch.equal(C1, C2)
    out = plan.subtract(Hd, dev(q.T), C2, dev(q.omega_t), None, -1.0)
    assert torch.isfinite(out).all() and bool((out[dev(q.omega_t) == 0] == -1.0).all())


@pytest.mark.parametrize("variant", VARIANTS + [5, 6])
def test_power_of_two_homogeneity_bitwise(variant):
    p = inputs.make_tiny()
    W1, H1, plan = gpu_fit(p, 30, variant)
    q = inputs.make_tiny(); q.X *= np.float32(4); q.W0 *= np.float32(4)
    W2, H2, _ = gpu_fit(q, 30, variant, plan)
    assert np.array_equal(H1, H2) and np.array_equal(W2, W1 * np.float32(4))
    q = inputs.make_tiny(); q.Omega *= np.float32(0.125)
    W3, H3, _ = gpu_fit(q, 30, variant, plan)
    assert np.array_equal(H1, H3) and np.array_equal(W1, W3)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("N,P,K", [(1, 4, 1), (3, 36, 2), (7, 132, 5), (33, 1028, 9), (65, 4100, 17),
                                   (129, 2052, 33), (200, 996, 50), (256, 516, 128), (225, 260, 53)])
def test_ragged_and_extreme_shapes(variant, N, P, K):
    """N, K, P off every tile size; K=1; the compiled maxima N=256, K=128; row-varying zeros in Omega."""
    if variant == 2 and K > 50:
        pytest.skip("the fused FFMA instantiations stop at K = 50")
    rng = np.random.default_rng(N * 1000 + K)
    X = (rng.random((N, P)) * 10).astype(np.float32)
    Om = (rng.random((N, P)) * (rng.random((N, P)) > 0.25)).astype(np.float32)
    Om[:, P // 2] = 0            # one fully masked column
    W0 = (0.1 + 0.9 * rng.random((N, K))).astype(np.float32)
    H0 = (0.1 + 0.9 * rng.random((K, P))).astype(np.float32)
    plan = nmf.Plan(N, P, K, variant=variant)
    if variant in (3, 4) and plan.variant != variant:
        pytest.skip("the fused tensor-core kernel stops at K = 64; the split kernels' operands do not fit shared memory at N = 256, K = 128")
    Xd, Od, Wd, Hd = dev(X), dev(Om), dev(W0), dev(H0)
    plan.fit(Xd, Od, Wd, Hd, 8)
    torch.cuda.synchronize()
    Wo, Ho = orc.fit(X, Om, W0, H0, 8)
    Hg = Hd.cpu().numpy()
    assert rel(Wd.cpu().numpy(), Wo) <= TOL_FACTOR and rel(Hg, Ho) <= TOL_FACTOR
    assert np.all(Hg[:, P // 2] == 0.0)     # G4: fully masked column -> exactly 0


@pytest.mark.parametrize("N,P,K,B", [(1, 4, 1, 1), (3, 36, 2, 1), (7, 132, 5, 1), (33, 1028, 7, 1), (129, 2052, 3, 1),
                                     (200, 32 * 148 * 5 + 20, 5, 1), (256, 32 * 148 * 3 + 8, 8, 1), (200, 32 * 148 * 2, 1, 1),
                                     (24, 2052, 6, 5), (12, 260, 4, 160)])
def test_streaming_kernel_few_components(N, P, K, B):
    """K <= 8 runs the streaming FP32 kernel (variant 5; the automatic choice there): K = 1 .. 8, N = 1 .. 256 (two to
    four stages), ragged last tile, one tile to more tiles per CTA than stages, batched problems (more than SMs);
    garbage where Omega == 0 and a repeated run must give bitwise the same factors."""
    rng = np.random.default_rng(N * 1000 + K + B)
    X = (rng.random((B, N, P)) * 10).astype(np.float32)
    Om = (rng.random((B, N, P)) * (rng.random((B, N, P)) > 0.25)).astype(np.float32)
    Om[:, :, P // 2] = 0         # one fully masked column
    W0 = (0.1 + 0.9 * rng.random((B, N, K))).astype(np.float32)
    H0 = (0.1 + 0.9 * rng.random((B, K, P))).astype(np.float32)
    plan = nmf.Plan(N, P, K, batch=B)
    assert plan.variant == 5 or (P + 127) // 128 * B <= 64       # launch-bound sizes take the fused FFMA kernel
    plan = nmf.Plan(N, P, K, batch=B, variant=5)
    assert plan.variant == 5
    iters = 9 if K <= 2 else 18 if K == 3 else 66                                  # enough for the tile-major copy (and a graph replay)
    res = []
    for garbage in (None, np.nan, 1e30):
        Xg = X.copy()
        if garbage is not None:
            Xg[Om == 0] = garbage
        Xd, Od, Wd, Hd = dev(Xg), dev(Om), dev(W0), dev(H0)
        if B == 1:
            plan.fit(Xd[0], Od[0], Wd[0], Hd[0], iters)
        else:
            plan.fit_batched(Xd, Od, Wd, Hd, iters)
        torch.cuda.synchronize()
        res.append((Wd.cpu().numpy(), Hd.cpu().numpy()))
    for Wg, Hg in res[1:]:
        assert np.array_equal(Wg, res[0][0]) and np.array_equal(Hg, res[0][1])
    # one call of `iters` iterations reads X and Omega from the tile-major copy, calls of 3 read the caller's arrays: same bits
    Xd, Od, Wd, Hd = dev(X), dev(Om), dev(W0), dev(H0)
    for _ in range(iters // 3):
        if B == 1:
            plan.fit(Xd[0], Od[0], Wd[0], Hd[0], 3)
        else:
            plan.fit_batched(Xd, Od, Wd, Hd, 3)
    torch.cuda.synchronize()
    assert np.array_equal(Wd.cpu().numpy(), res[0][0]) and np.array_equal(Hd.cpu().numpy(), res[0][1])
    Wg, Hg = res[0]
    for b in range(0, B, max(1, B // 4)):
        Wo, Ho = orc.fit(X[b], Om[b], W0[b], H0[b], iters)
        assert rel(Wg[b], Wo) <= TOL_FACTOR and rel(Hg[b], Ho) <= TOL_FACTOR, (b, rel(Wg[b], Wo), rel(Hg[b], Ho))
        assert np.all(Hg[b][:, P // 2] == 0.0)


@pytest.mark.parametrize("N,P,K", [(1, 4, 1), (3, 36, 2), (16, 4096, 5), (7, 132, 8), (64, 128 * 148, 3), (33, 128 * 147 + 20, 7)])
def test_resident_kernel_small_problems(N, P, K):
    """K <= 8, N <= 64, at most one 128-pixel tile per SM: the whole fit is ONE cooperative launch (variant 6; the automatic
    choice there) with a grid-wide barrier per iteration: one CTA to all 148, ragged last tile, 1 + 40 + 41 iterations
    against one call of 82 (bitwise), garbage where Omega == 0, oracle parity."""
    rng = np.random.default_rng(N * 1000 + K)
    X = (rng.random((N, P)) * 10).astype(np.float32)
    Om = (rng.random((N, P)) * (rng.random((N, P)) > 0.25)).astype(np.float32)
    Om[:, P // 2] = 0
    W0 = (0.1 + 0.9 * rng.random((N, K))).astype(np.float32)
    H0 = (0.1 + 0.9 * rng.random((K, P))).astype(np.float32)
    plan = nmf.Plan(N, P, K)
    assert plan.variant == 6
    iters = 82
    res = []
    for garbage in (None, np.nan):
        Xg = X.copy()
        if garbage is not None:
            Xg[Om == 0] = garbage
        Xd, Od, Wd, Hd = dev(Xg), dev(Om), dev(W0), dev(H0)
        plan.fit(Xd, Od, Wd, Hd, iters)
        torch.cuda.synchronize()
        res.append((Wd.cpu().numpy(), Hd.cpu().numpy()))
    Xd, Od, Wd, Hd = dev(X), dev(Om), dev(W0), dev(H0)
    for n in (1, 40, 41):
        plan.fit(Xd, Od, Wd, Hd, n)
    torch.cuda.synchronize()
    res.append((Wd.cpu().numpy(), Hd.cpu().numpy()))
    for Wg, Hg in res[1:]:
        assert np.array_equal(Wg, res[0][0]) and np.array_equal(Hg, res[0][1])
    Wo, Ho = orc.fit(X, Om, W0, H0, iters)
    assert rel(res[0][0], Wo) <= TOL_FACTOR and rel(res[0][1], Ho) <= TOL_FACTOR, (rel(res[0][0], Wo), rel(res[0][1], Ho))
    assert np.all(res[0][1][:, P // 2] == 0.0)


def test_zero_entries_stay_zero_and_empty_iters():
    p = inputs.make_tiny()
    p.W0[2, 1] = 0.0; p.H0[3, 77] = 0.0
    W, H, plan = gpu_fit(p, 10)
    assert W[2, 1] == 0.0 and H[3, 77] == 0.0
    W0, H0, _ = gpu_fit(p, 0, plan=plan)
    assert np.array_equal(W0, p.W0) and np.array_equal(H0, p.H0)


def test_objective_monotone_on_gpu_iterates():
    """fp32 iterates still decrease the fp64-evaluated objective every iteration (P1 on the device path)."""
    p = inputs.make_tiny()
    plan = nmf.Plan(p.N, p.P, p.K)
    X, Om, W, H = dev(p.X), dev(p.Omega), dev(p.W0), dev(p.H0)
    prev = plan.objective(X, Om, W, H)
    for _ in range(25):
        plan.fit(X, Om, W, H, 1)
        f = plan.objective(X, Om, W, H)
        assert f <= prev * (1 + 1e-6)
        prev = f


def test_error_codes():
    L = nmf.lib()
    p = inputs.make_tiny()
    plan = nmf.Plan(p.N, p.P, p.K, max_targets=2)
    X, Om, W, H = dev(p.X), dev(p.Omega), dev(p.W0), dev(p.H0)
    h = plan._h
    assert L.nmf_fit(h, None, Om.data_ptr(), W.data_ptr(), H.data_ptr(), 1) == -1
    assert L.nmf_fit(h, X.data_ptr(), Om.data_ptr(), W.data_ptr(), H.data_ptr(), -1) == -1
    assert L.nmf_fit(h, X.data_ptr() + 4, Om.data_ptr(), W.data_ptr(), H.data_ptr(), 1) == -2
    assert L.nmf_project(h, H.data_ptr(), X.data_ptr(), None, W.data_ptr(), 3, 1) == -1    # M > max_targets
    assert L.nmf_plan_set_workspace(h, plan.workspace.data_ptr(), 8) == -4
    h2 = ctypes.c_void_p()
    assert L.nmf_plan_create(ctypes.byref(h2), p.N, p.P, p.K, 1, 0) == 0
    assert L.nmf_fit(h2, X.data_ptr(), Om.data_ptr(), W.data_ptr(), H.data_ptr(), 1) == -4  # no workspace
    assert L.nmf_plan_destroy(h2) == 0
    with pytest.raises(TypeError):
        plan.fit(X.cpu(), Om, W, H, 1)


def test_host_entry_points_match_device_path():
    p = inputs.make_miri(N=24, S=64, K=8, M=3)
    Wd, Hd, plan = gpu_fit(p, 15)
    Wh, Hh = torch.from_numpy(p.W0.copy()), torch.from_numpy(p.H0.copy())
    plan.fit_host(torch.from_numpy(p.X), torch.from_numpy(p.Omega), Wh, Hh, 15)
    assert np.array_equal(Wh.numpy(), Wd) and np.array_equal(Hh.numpy(), Hd)
    C = torch.from_numpy(p.C0.copy()); out = torch.empty(p.M, p.P)
    plan.project_subtract_host(dev(Hd), torch.from_numpy(p.T), torch.from_numpy(p.omega_t), C, out, 30)
    Co = orc.project(Hd, p.T, p.omega_t, p.C0, 30)
    assert rel(C.numpy(), Co) <= TOL_FACTOR
    # the same with staging owned by the caller (nmf_plan_set_staging): bitwise the same results, and a staging buffer
    # that is too small is refused instead of being replaced behind the caller
    plan2 = nmf.Plan(p.N, p.P, p.K, max_targets=p.M)
    plan2.use_own_staging(p.M)
    W2, H2 = torch.from_numpy(p.W0.copy()), torch.from_numpy(p.H0.copy())
    plan2.fit_host(torch.from_numpy(p.X), torch.from_numpy(p.Omega), W2, H2, 15)
    assert np.array_equal(W2.numpy(), Wd) and np.array_equal(H2.numpy(), Hd)
    L = nmf.lib()
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    assert L.nmf_plan_set_staging(plan2._h, small.data_ptr(), 1024) == 0
    assert L.nmf_fit_host(plan2._h, p.X.ctypes.data, p.Omega.ctypes.data, W2.data_ptr(), H2.data_ptr(), 1) == -4
    assert L.nmf_plan_set_staging(plan2._h, None, 0) == 0
    assert L.nmf_plan_set_staging(plan2._h, small.data_ptr(), 0) == -1


@pytest.mark.parametrize("variant", [3, 4])
@pytest.mark.parametrize("N", [64, 96, 128, 200])
def test_tensor_core_path_multi_tile_deterministic(N, variant):
    """Several pixel tiles per persistent CTA (the TMA ring wraps many times) with one and two 128-frame M tiles:
    parity after 2 iterations and bitwise run-to-run equality (a ring slot released before its values were
    consumed once showed up here as a 1e-4, run-dependent error in W)."""
    K, P = 32, 128 * 148 * 2 + 36
    rng = np.random.default_rng(N)
    X = (rng.random((N, P)) * 10).astype(np.float32)
    Om = (rng.random((N, P)) * (rng.random((N, P)) > 0.25)).astype(np.float32)
    W0 = (0.1 + 0.9 * rng.random((N, K))).astype(np.float32)
    H0 = (0.1 + 0.9 * rng.random((K, P))).astype(np.float32)
    plan = nmf.Plan(N, P, K, variant=variant)
    res = []
    for _ in range(2):
        Wd, Hd = dev(W0), dev(H0)
        plan.fit(dev(X), dev(Om), Wd, Hd, 2)
        torch.cuda.synchronize()
        res.append((Wd.cpu().numpy(), Hd.cpu().numpy()))
    assert np.array_equal(res[0][0], res[1][0]) and np.array_equal(res[0][1], res[1][1])
    Wo, Ho = orc.fit(X, Om, W0, H0, 2)
    assert rel(res[0][0], Wo) <= 1e-5 and rel(res[0][1], Ho) <= 1e-5


@pytest.mark.parametrize("N,K,tiles", [(200, 100, 2), (200, 112, 3), (224, 100, 2), (240, 128, 2), (128, 100, 5), (200, 81, 4)])
def test_split_kernels_small_rings(N, K, tiles):
    """Large K with many frames leaves the split kernels two or three ring slots, and several tiles per persistent CTA
    on all 148 SMs.  (N, K) = (200, 100) had three slots: a group that ran ahead of a late TMA load tested the mbarrier
    parity of the slot's use before last, read a slot that had not landed and corrupted the transaction count --
    launch failure, only with two or more tiles per CTA.)  Parity after 2 iterations, bitwise run-to-run equality."""
    P = 128 * 148 * tiles
    rng = np.random.default_rng(N + K)
    X = (rng.random((N, P)) * 10).astype(np.float32)
    Om = (rng.random((N, P)) * (rng.random((N, P)) > 0.25)).astype(np.float32)
    W0 = (0.1 + 0.9 * rng.random((N, K))).astype(np.float32)
    H0 = (0.1 + 0.9 * rng.random((K, P))).astype(np.float32)
    plan = nmf.Plan(N, P, K)
    if plan.variant != 4:
        pytest.skip("the operands of this shape do not fit the split kernels' shared memory")
    res = []
    for _ in range(2):
        Wd, Hd = dev(W0), dev(H0)
        plan.fit(dev(X), dev(Om), Wd, Hd, 2)
        torch.cuda.synchronize()
        res.append((Wd.cpu().numpy(), Hd.cpu().numpy()))
    assert np.array_equal(res[0][0], res[1][0]) and np.array_equal(res[0][1], res[1][1])
    Wo, Ho = orc.fit(X, Om, W0, H0, 2)
    assert rel(res[0][0], Wo) <= TOL_FACTOR and rel(res[0][1], Ho) <= TOL_FACTOR


@pytest.mark.parametrize("variant", [3, 4])
def test_projection_many_targets(variant):
    """M = 300 science frames: the tensor-core projection handles them 256 at a time (two passes)."""
    N, P, K, M = 12, 2052, 9, 300
    rng = np.random.default_rng(7)
    H = (rng.random((K, P)) + 0.05).astype(np.float32)
    T = (rng.random((M, P)) * 5).astype(np.float32)
    om = (rng.random((M, P)) * (rng.random((M, P)) > 0.2)).astype(np.float32)
    C0 = (0.1 + 0.9 * rng.random((M, K))).astype(np.float32)
    plan = nmf.Plan(N, P, K, max_targets=M, variant=variant)
    C = dev(C0)
    plan.project(dev(H), dev(T), dev(om), C, 25)
    Co = orc.project(H, T, om, C0, 25)
    assert rel(C.cpu().numpy(), Co) <= TOL_FACTOR
    out = plan.subtract(dev(H), dev(T), C, dev(om), None, 0.0).cpu().numpy()
    outo = orc.subtract(H, T, Co, om, None, 0.0)
    assert np.abs(out - outo).max() <= TOL_FACTOR * np.abs(T).max()


@pytest.mark.parametrize("M,P,K,iters", [
    (1, 4, 1, 5), (31, 132, 16, 5), (33, 1028, 17, 5), (64, 4100, 33, 5), (32, 128 * 148 * 2 + 68, 50, 4),
    (7, 128 * 148 * 3, 64, 3), (4, 128 * 148 * 17 + 192, 5, 3), (40, 128 * 148 * 33 + 64, 20, 2)])
def test_projection_pipelined_kernel_shapes(M, P, K, iters):
    """Projections of up to 64 frames with K <= 64 run the pipelined W kernel (k_tc_wp: H pieces double-buffered and
    landed 64 pixels at a time, S' of the next tile queued behind AB): one tile, one to three tiles per CTA, ragged last
    tile, more than 16 and more than 32 tiles per CTA (one and two accumulator flushes), every 16-component block count,
    1 to 64 frames (one or two lane quadrants); twice, bitwise equal."""
    rng = np.random.default_rng(100 * M + K)
    H = (rng.random((K, P)) + 0.05).astype(np.float32)
    T = (rng.random((M, P)) * 5).astype(np.float32)
    om = (rng.random((M, P)) * (rng.random((M, P)) > 0.2)).astype(np.float32)
    C0 = (0.1 + 0.9 * rng.random((M, K))).astype(np.float32)
    plan = nmf.Plan(8, P, K, max_targets=M, variant=4)
    Hd, Td, od = dev(H), dev(T), dev(om)
    res = []
    for _ in range(2):
        C = dev(C0)
        plan.project(Hd, Td, od, C, iters)
        torch.cuda.synchronize()
        res.append(C.cpu().numpy())
    assert np.array_equal(res[0], res[1])
    Co = orc.project(H, T, om, C0, iters)
    assert rel(res[0], Co) <= TOL_FACTOR, rel(res[0], Co)


@pytest.mark.parametrize("K,M", [(1, 600), (5, 4096), (13, 600), (13, 4096)])
def test_generic_projection_many_targets_no_weights(K, M):
    """omega == NULL projection runs the generic FFMA W half-step.  For K <= 13 its geometry allowed up to 1024 frames per
    CTA and asked for up to 296 KB of shared memory (launch failure, coef overwritten from an unwritten slab): the frames
    per CTA are now capped by the opt-in shared memory.  M up to the plan maximum of 4096."""
    N, P = 8, 516
    rng = np.random.default_rng(1000 * K + M)
    H = (rng.random((K, P)) + 0.05).astype(np.float32)
    T = (rng.random((M, P)) * 5).astype(np.float32)
    C0 = (0.1 + 0.9 * rng.random((M, K))).astype(np.float32)
    plan = nmf.Plan(N, P, K, max_targets=M)
    C = dev(C0)
    plan.project(dev(H), dev(T), None, C, 10)
    torch.cuda.synchronize()
    Co = orc.project(H, T, None, C0, 10)
    assert rel(C.cpu().numpy(), Co) <= TOL_FACTOR
    # the same through the generic family with weights (variant 1)
    om = (rng.random((M, P)) * (rng.random((M, P)) > 0.2)).astype(np.float32)
    plan1 = nmf.Plan(N, P, K, max_targets=M, variant=1)
    C1 = dev(C0)
    plan1.project(dev(H), dev(T), dev(om), C1, 10)
    torch.cuda.synchronize()
    assert rel(C1.cpu().numpy(), orc.project(H, T, om, C0, 10)) <= TOL_FACTOR


@pytest.mark.parametrize("variant", [3, 4])
def test_batched_more_problems_than_sms(variant):
    """160 independent small problems in one batched launch sequence (grid.y > number of SMs: the persistent
    CTAs of different problems are not co-resident and must not depend on one another)."""
    B, N, P, K = 160, 8, 260, 3
    rng = np.random.default_rng(11)
    X = (rng.random((B, N, P)) * 10).astype(np.float32)
    Om = (rng.random((B, N, P)) * (rng.random((B, N, P)) > 0.2)).astype(np.float32)
    W0 = (0.1 + 0.9 * rng.random((B, N, K))).astype(np.float32)
    H0 = (0.1 + 0.9 * rng.random((B, K, P))).astype(np.float32)
    plan = nmf.Plan(N, P, K, batch=B, variant=variant)
    Wd, Hd = dev(W0), dev(H0)
    plan.fit_batched(dev(X), dev(Om), Wd, Hd, 6)
    torch.cuda.synchronize()
    Wg, Hg = Wd.cpu().numpy(), Hd.cpu().numpy()
    for b in (0, 1, 77, 147, 148, 159):
        Wo, Ho = orc.fit(X[b], Om[b], W0[b], H0[b], 6)
        assert rel(Wg[b], Wo) <= 1e-5 and rel(Hg[b], Ho) <= 1e-5, b


def test_automatic_family_selection():
    """variant 0: the split tensor-core kernels wherever they fit, the streaming kernel for K <= 8, the resident kernel for
    problems that stay on chip, the fused FFMA kernel for other launch-bound sizes (at most 64 pixel tiles in all), the
    generic kernels where nothing else covers the shape"""
    assert nmf.Plan(200, 1 << 20, 50).variant == 4
    assert nmf.Plan(200, 1 << 20, 100).variant == 4
    assert nmf.Plan(128, 65536, 20, batch=64).variant == 4
    assert nmf.Plan(200, 1 << 20, 5).variant == 5
    assert nmf.Plan(16, 4096, 5).variant == 6
    assert nmf.Plan(16, 4096, 5, batch=2).variant == 2   # the resident kernel takes one problem
    assert nmf.Plan(16, 4096, 12).variant == 2           # ... of at most 8 components
    assert nmf.Plan(16, 4096, 60).variant == 4          # no fused FFMA instantiation beyond K = 50
    assert nmf.Plan(256, 1 << 16, 128).variant == 1
