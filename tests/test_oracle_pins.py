"""T0: pins for the CPU oracle.  No GPU.

Every check here ties oracle/ to something other than itself: the paper's cost
and update definitions worked by hand (golden fixtures), closed forms, library
routines (SVD, least squares) on special cases, brute-force NNLS, and invariants
that a dropped term / wrong index / transposed operand would break.
"""
import itertools
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import nmf_oracle as orc
from oracle import nmf_numpy as onp
from paper_2309_04623_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _parse_rows(s):
    return np.array([[float(Fraction(t)) for t in row.split()] for row in s.split(" / ")])


def _load_p4():
    d = {}
    for line in open(os.path.join(GOLD, "p4_worked_example.txt")):
        if line.startswith("#") or not line.strip():
            continue
        key, rest = line.split(None, 1)
        d[key] = _parse_rows(rest.strip())
    return d


@pytest.fixture(scope="module")
def tiny():
    return inputs.make_tiny()


# ---- P4: exact-rational worked example -------------------------------------
def test_p4_worked_example():
    g = _load_p4()
    X, Om, W0, H0 = g["X"], g["Omega"], g["W0"], g["H0"]
    assert orc.objective(X, Om, W0, H0) == pytest.approx(46.0, rel=1e-14)
    H1 = orc.h_step(X, Om, W0, H0)
    np.testing.assert_allclose(H1, g["H1"], rtol=1e-14, atol=0)
    assert orc.objective(X, Om, W0, H1) == pytest.approx(g["f_H1"][0, 0], rel=1e-13)
    W1 = orc.w_step(X, Om, W0, H1)
    np.testing.assert_allclose(W1, g["W1"], rtol=1e-13)
    assert orc.objective(X, Om, W1, H1) == pytest.approx(g["f_W1"][0, 0], rel=2e-9)
    W2, H2, tr = orc.fit(X, Om, W0, H0, 2, trace=True)
    np.testing.assert_allclose(tr, [46.0, g["f_H1"][0, 0], g["f_W1"][0, 0], g["f_H2"][0, 0], g["f_W2"][0, 0]],
                               rtol=2e-9)
    np.testing.assert_allclose(W2, g["W2"], rtol=2e-9)
    np.testing.assert_allclose(H2, g["H2"], rtol=2e-9, atol=0)
    assert np.all(H2[:, 2] == 0.0)     # fully masked column -> exactly 0 (G4)


def test_p4b_k1_hand_example():
    X = np.array([[1.0, 2.0], [3.0, 4.0]])
    w0 = np.ones((2, 1)); h0 = np.ones((1, 2))
    for line in open(os.path.join(GOLD, "p4b_k1_example.txt")):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        Om = np.ones((2, 2)) if t[0] == "case_full" else np.array([[1.0, 0.0], [1.0, 1.0]])
        h1 = [float(Fraction(v)) for v in t[2:4]]
        w1 = [float(Fraction(v)) for v in t[5:7]]
        f = [float(Fraction(v)) for v in t[8:11]]
        W, H, tr = orc.fit(X, Om, w0, h0, 1, trace=True)
        np.testing.assert_allclose(H.ravel(), h1, rtol=1e-15)
        np.testing.assert_allclose(W.ravel(), w1, rtol=1e-15)
        np.testing.assert_allclose(tr, f, rtol=1e-13)


# ---- P1 + P2: monotone objective on both half-steps, non-negativity ----------
def test_p1_p2_monotone_nonneg(tiny):
    p = tiny
    W, H, tr = orc.fit(p.X, p.Omega, p.W0, p.H0, 200, trace=True)
    assert np.all(tr[1:] <= tr[:-1] * (1 + 1e-12)), "objective increased on a half-step"
    assert tr[-1] < 1e-3 * tr[0]
    assert np.all(W >= 0) and np.all(H >= 0) and np.all(np.isfinite(W)) and np.all(np.isfinite(H))
    # step-by-step API agrees with the fused loop, and zeros stay zeros
    W0z = p.W0.astype(np.float64).copy(); W0z[3, 2] = 0.0
    H0z = p.H0.astype(np.float64).copy(); H0z[1, 100] = 0.0
    Wz, Hz = orc.fit(p.X, p.Omega, W0z, H0z, 5)
    assert Wz[3, 2] == 0.0 and Hz[1, 100] == 0.0


def test_p1_monotone_weighted_rowvarying():
    """Heteroscedastic, row-varying zeros (the general Omega of Eq. 2)."""
    rng = np.random.default_rng(7)
    N, P, K = 9, 157, 4
    X = rng.random((N, P)).astype(np.float32) * 10
    Om = (rng.random((N, P)) * (rng.random((N, P)) > 0.3)).astype(np.float32)
    W0 = 0.1 + rng.random((N, K)); H0 = 0.1 + rng.random((K, P))
    _, _, tr = orc.fit(X, Om, W0, H0, 60, trace=True)
    assert np.all(tr[1:] <= tr[:-1] * (1 + 1e-12))


# ---- P3: mask invariance, bitwise ------------------------------------------
@pytest.mark.parametrize("garbage", [1e30, np.nan, np.inf, -5.0])
def test_p3_mask_invariance(tiny, garbage):
    p = tiny
    W, H = orc.fit(p.X, p.Omega, p.W0, p.H0, 20)
    Xg = p.X.copy(); Xg[p.Omega == 0] = garbage
    Wg, Hg = orc.fit(Xg, p.Omega, p.W0, p.H0, 20)
    assert np.array_equal(W, Wg) and np.array_equal(H, Hg)
    assert orc.objective(Xg, p.Omega, W, H) == orc.objective(p.X, p.Omega, W, H)
    Tg = p.T.copy(); Tg[p.omega_t == 0] = garbage
    assert np.array_equal(orc.project(H, Tg, p.omega_t, p.C0, 10), orc.project(H, p.T, p.omega_t, p.C0, 10))


# ---- P5: noise-free rank-K recovery ----------------------------------------
def test_p5_rank_k_recovery():
    p = inputs.make_tiny(noise=0.0)
    norm = float(np.sum(p.Omega.astype(np.float64) * p.X.astype(np.float64) ** 2))
    _, _, tr = orc.fit(p.X, p.Omega, p.W0, p.H0, 2000, trace=True)
    assert np.all(tr[1:] <= tr[:-1] * (1 + 1e-12))
    assert tr[400] / norm <= 1e-3      # after 200 iterations
    assert tr[-1] / norm <= 1e-5       # after 2000 iterations


# ---- P6: fixed point -------------------------------------------------------
def test_p6_fixed_point():
    rng = np.random.default_rng(3)
    N, P, K = 7, 93, 3
    Ws = 0.2 + rng.random((N, K)); Hs = 0.2 + rng.random((K, P))
    X = (Ws @ Hs)
    X32 = X.astype(np.float32)
    # make X exactly representable so that X == Ws Hs holds for the fp32 input
    Ws = np.round(Ws * 64) / 64; Hs = np.round(Hs * 64) / 64
    X32 = (Ws @ Hs).astype(np.float32)
    assert np.array_equal(X32.astype(np.float64), Ws @ Hs)
    Om = (rng.random((N, P)) > 0.2).astype(np.float32) * 0.5
    W, H = orc.fit(X32, Om, Ws, Hs, 100)
    live = Om.max(axis=0) > 0
    np.testing.assert_allclose(W, Ws, rtol=1e-12)
    np.testing.assert_allclose(H[:, live], Hs[:, live], rtol=1e-12)


# ---- P7: K=1 closed form + dominant singular pair --------------------------
def test_p7_k1_closed_form_and_svd():
    rng = np.random.default_rng(11)
    N, P = 12, 200
    X = rng.random((N, P)).astype(np.float32) + 0.05
    Om = (rng.random((N, P)) * (rng.random((N, P)) > 0.25)).astype(np.float32)
    w = 0.1 + rng.random((N, 1)); h = 0.1 + rng.random((1, P))
    Xd, Od = X.astype(np.float64), Om.astype(np.float64)
    # K=1: the update does not depend on the old value (weighted rank-1 ALS)
    h1 = orc.h_step(X, Om, w, h)
    np.testing.assert_allclose(h1[0], (Od * Xd * w).sum(0) / (Od * w * w).sum(0), rtol=1e-12)
    w1 = orc.w_step(X, Om, w, h1)
    np.testing.assert_allclose(w1[:, 0], (Od * Xd * h1).sum(1) / (Od * h1 * h1).sum(1), rtol=1e-12)
    # Omega == 1: converges to the dominant singular pair (Perron-Frobenius)
    ones = np.ones_like(X)
    W, H, tr = orc.fit(X, ones, w, h, 60, trace=True)
    s = np.linalg.svd(Xd, compute_uv=False)
    assert tr[-1] == pytest.approx((Xd ** 2).sum() - s[0] ** 2, rel=1e-10)


# ---- P8: homogeneity, bitwise ----------------------------------------------
def test_p8_power_of_two_homogeneity(tiny):
    p = tiny
    W, H = orc.fit(p.X, p.Omega, p.W0, p.H0, 15)
    W8, H8 = orc.fit(p.X * np.float32(8), p.Omega, p.W0 * np.float32(8), p.H0, 15)
    assert np.array_equal(H8, H) and np.array_equal(W8, W * 8)
    Wo, Ho = orc.fit(p.X, p.Omega * np.float32(0.25), p.W0, p.H0, 15)
    assert np.array_equal(Ho, H) and np.array_equal(Wo, W)


# ---- P9: permutation equivariance ------------------------------------------
def test_p9_equivariance():
    rng = np.random.default_rng(5)
    N, P, K = 8, 120, 4
    X = rng.random((N, P)).astype(np.float32)
    Om = (rng.random((N, P)) * (rng.random((N, P)) > 0.2)).astype(np.float32)
    W0 = 0.1 + rng.random((N, K)); H0 = 0.1 + rng.random((K, P))
    W, H = orc.fit(X, Om, W0, H0, 12)
    pn, pp, pk = rng.permutation(N), rng.permutation(P), rng.permutation(K)
    Wn, Hn = orc.fit(X[pn], Om[pn], W0[pn], H0, 12)
    np.testing.assert_allclose(Wn, W[pn], rtol=1e-12); np.testing.assert_allclose(Hn, H, rtol=1e-12)
    Wp, Hp = orc.fit(X[:, pp], Om[:, pp], W0, H0[:, pp], 12)
    np.testing.assert_allclose(Wp, W, rtol=1e-12); np.testing.assert_allclose(Hp, H[:, pp], rtol=1e-12)
    Wk, Hk = orc.fit(X, Om, W0[:, pk], H0[pk], 12)
    np.testing.assert_allclose(Wk, W[:, pk], rtol=1e-12); np.testing.assert_allclose(Hk, H[pk], rtol=1e-12)


# ---- P10 + P11: projection = NNLS (brute force) and KKT ---------------------
def _nnls_bruteforce(Hm, t, om):
    """min_{c>=0} sum om (t - c H)^2 by enumerating all 2^K supports."""
    K = Hm.shape[0]
    sw = np.sqrt(om)
    A = (Hm * sw).T; b = t * sw
    best, best_c = np.inf, None
    for r in range(K + 1):
        for sup in itertools.combinations(range(K), r):
            c = np.zeros(K)
            if sup:
                sol = np.linalg.lstsq(A[:, sup], b, rcond=None)[0]
                if np.any(sol < 0):
                    continue
                c[list(sup)] = sol
            f = float(np.sum((A @ c - b) ** 2))
            if f < best:
                best, best_c = f, c
    return best, best_c


def test_p10_p11_projection_nnls_kkt(tiny):
    p = tiny
    _, H = orc.fit(p.X, p.Omega, p.W0, p.H0, 50)
    t = p.T[0].astype(np.float64); om = p.omega_t[0].astype(np.float64)
    f_star, c_star = _nnls_bruteforce(H, t, om)
    c = orc.project(H, p.T, p.omega_t, p.C0, 3000)[0]
    f = float(np.sum(om * (t - c @ H) ** 2))
    assert f == pytest.approx(f_star, rel=1e-10)
    np.testing.assert_allclose(c, c_star, rtol=1e-6, atol=1e-8 * np.abs(c_star).max())
    # KKT residual (P11)
    g = (om * (c @ H - t)) @ H.T
    active = c <= 1e-9 * c.max()          # MU approaches an active bound geometrically, never exactly
    kkt = np.where(active, np.minimum(g, 0.0), np.abs(g))
    assert np.abs(kkt).max() / np.abs((om * t) @ H.T).max() < 1e-9
    # with an active constraint: a target anti-correlated with one component
    t2 = np.maximum(t - 3.0 * H[0] * t.max() / H[0].max(), 0).astype(np.float32)[None]
    f2, c2 = _nnls_bruteforce(H, t2[0].astype(np.float64), om)
    c2m = orc.project(H, t2, p.omega_t, p.C0, 20000)[0]
    assert float(np.sum(om * (t2[0] - c2m @ H) ** 2)) == pytest.approx(f2, rel=1e-8)


def test_projection_omega_none_and_rows_independent(tiny):
    p = inputs.make_tiny(M=3)
    _, H = orc.fit(p.X, p.Omega, p.W0, p.H0, 10)
    ones = np.ones_like(p.T)
    assert np.array_equal(orc.project(H, p.T, None, p.C0, 7), orc.project(H, p.T, ones, p.C0, 7))
    call = orc.project(H, p.T, p.omega_t, p.C0, 7)
    for m in range(3):
        assert np.array_equal(call[m:m + 1], orc.project(H, p.T[m:m + 1], p.omega_t[m:m + 1], p.C0[m:m + 1], 7))


# ---- P12: two independent oracles -------------------------------------------
def test_p12_two_oracles_tiny(tiny):
    p = tiny
    W, H = orc.fit(p.X, p.Omega, p.W0, p.H0, 200)
    W2, H2 = onp.fit(p.X, p.Omega, p.W0, p.H0, 200)
    assert np.linalg.norm(W - W2) / np.linalg.norm(W) < 1e-12
    assert np.linalg.norm(H - H2) / np.linalg.norm(H) < 1e-12
    assert orc.objective(p.X, p.Omega, W, H) == pytest.approx(onp.objective(p.X, p.Omega, W, H), rel=1e-12)


def test_p12_two_oracles_miri_reduced():
    p = inputs.make_miri(N=24, S=64, K=8, M=2)
    W, H = orc.fit(p.X, p.Omega, p.W0, p.H0, 50)
    W2, H2 = onp.fit(p.X, p.Omega, p.W0, p.H0, 50)
    assert np.linalg.norm(W - W2) / np.linalg.norm(W) < 1e-12
    assert np.linalg.norm(H - H2) / np.linalg.norm(H) < 1e-12


# ---- subtraction --------------------------------------------------------------
def test_subtract_definition_and_special_cases():
    rng = np.random.default_rng(2)
    M, P, K = 3, 50, 4
    H = np.round(rng.random((K, P)) * 16); C = np.round(rng.random((M, K)) * 8)
    T = (C @ H).astype(np.float32)                       # exactly representable model
    om = (rng.random((M, P)) > 0.3).astype(np.float32)
    out = orc.subtract(H, T, C, om, None, fill=-7.0)
    assert np.all(out[om > 0] == 0.0) and np.all(out[om == 0] == -7.0)
    assert np.array_equal(orc.subtract(H, T, C * 0, None, None), T.astype(np.float64))
    fac = np.array([0.0, 1.0, 2.0])
    out = orc.subtract(H, T, C, None, fac)
    np.testing.assert_array_equal(out, T - fac[:, None] * (C @ H))
    Tn = T.copy(); Tn[om == 0] = np.nan
    assert np.all(np.isfinite(orc.subtract(H, Tn, C, om, None, fill=0.0)))


# ---- generators: structure facts stated in DESIGN.md / SURVEY §8(d) ----------
def test_generator_structure():
    p = inputs.make_tiny()
    assert p.X.shape == (16, 4096) and p.X.dtype == np.float32 and int((p.Omega[0] == 0).sum()) == 113
    assert p.W0.min() >= 0.1 and p.W0.max() < 1.0 and p.H0.dtype == np.float32
    q = inputs.make_miri(N=4, M=1)
    assert int((q.Omega[0] == 0).sum()) == 1727 and q.X.min() >= 0
    assert np.array_equal(q.Omega[0] == 0, q.Omega[3] == 0)
    p2 = inputs.make_tiny()
    assert np.array_equal(p.X, p2.X) and np.array_equal(p.H0, p2.H0)    # seeded
    s = inputs.make_stis(N=3, S=128, K=4, M=1)
    frac = float((s.Omega[0] == 0).mean())
    assert 0.05 < frac < 0.08


# ---------------------------------------------------------------------------------------------
# P13-P16: closest-frame reference selection (readings G19/G20)
# ---------------------------------------------------------------------------------------------
def _ref_case(M=5, N=9, P=37, seed=0, masks=True):
    rng = np.random.default_rng(seed)
    T = (rng.random((M, P)) * 4).astype(np.float32)
    X = (rng.random((N, P)) * 4).astype(np.float32)
    ot = (rng.random((M, P)) > 0.3).astype(np.float32) * (0.5 + rng.random((M, P))).astype(np.float32) if masks else None
    Om = (rng.random((N, P)) > 0.2).astype(np.float32) * (0.5 + rng.random((N, P))).astype(np.float32) if masks else None
    return T, ot, X, Om


def test_p13_ref_distance_brute_force_and_expansion():
    """D against (a) pure-Python loops on a tiny case and (b) the expanded form
    sum a b t^2 - 2 sum (a t)(b x) + sum a b x^2 (three matrix products with the 0/1 masks a, b)."""
    T, ot, X, Om = _ref_case()
    D = orc.ref_distance(T, ot, X, Om)
    M, N, P = T.shape[0], X.shape[0], T.shape[1]
    for m in range(M):
        for n in range(N):
            s = 0.0
            for p in range(P):
                if ot[m, p] > 0 and Om[n, p] > 0:
                    s += (float(T[m, p]) - float(X[n, p])) ** 2
            assert abs(D[m, n] - s) <= 1e-12 * max(s, 1.0)
    a, b = (ot > 0).astype(np.float64), (Om > 0).astype(np.float64)
    t, x = T.astype(np.float64), X.astype(np.float64)
    E = (a * t * t) @ b.T - 2.0 * (a * t) @ (b * x).T + a @ (b * x * x).T
    assert np.abs(D - E).max() <= 1e-10 * np.abs(E).max()


def test_p14_ref_distance_identities():
    T, ot, X, Om = _ref_case(M=4, N=6, P=50, seed=3)
    X[2] = T[1]                                    # a reference equal to a target: distance 0 on any mask
    D = orc.ref_distance(T, ot, X, Om)
    assert D[1, 2] == 0.0 and (D >= 0).all()
    # symmetry: swapping the roles transposes D
    assert np.array_equal(orc.ref_distance(X, Om, T, ot), D.T)
    # no masks: the plain squared Euclidean norm; NULL == all-ones masks
    Dn = orc.ref_distance(T, None, X, None)
    assert np.allclose(Dn, ((T[:, None, :].astype(np.float64) - X[None].astype(np.float64)) ** 2).sum(-1), rtol=1e-13)
    assert np.array_equal(Dn, orc.ref_distance(T, np.ones_like(T), X, np.ones_like(X)))
    # scaling both by s scales D by s^2; a common offset leaves it unchanged (exact in fp64 for powers of two)
    assert np.array_equal(orc.ref_distance(T * np.float32(4), ot, X * np.float32(4), Om), D * 16.0)
    # every masked pair contributes nothing: masking a pixel can only lower D
    ot2 = ot.copy(); ot2[:, ::3] = 0
    assert (orc.ref_distance(T, ot2, X, Om) <= D + 1e-15).all()


def test_p15_ref_distance_mask_invariance():
    """Masked entries may hold NaN / Inf / 1e30: bitwise the same distances."""
    T, ot, X, Om = _ref_case(seed=5)
    D = orc.ref_distance(T, ot, X, Om)
    for g in (np.nan, np.inf, 1e30):
        T2, X2 = T.copy(), X.copy()
        T2[ot == 0] = g; X2[Om == 0] = g
        assert np.array_equal(orc.ref_distance(T2, ot, X2, Om), D)


def test_p16_ref_select_order_and_ties():
    rng = np.random.default_rng(9)
    D = rng.random((6, 40))
    D[2, 7] = D[2, 31] = D[2].min() / 2            # an exact tie for first place: lower index first
    D[4] = 1.0                                     # all equal: identity order
    for n_sel in (1, 5, 40):
        idx = orc.ref_select(D, n_sel)
        ref = np.argsort(D, axis=1, kind="stable")[:, :n_sel]
        assert np.array_equal(idx, ref)
    assert list(orc.ref_select(D, 2)[2]) == [7, 31]
    assert list(orc.ref_select(D, 3)[4]) == [0, 1, 2]
    # selecting the closest frames of a library that contains the target itself returns it first
    T, ot, X, Om = _ref_case(M=3, N=8, P=64, seed=1)
    X[5] = T[0]; X[1] = T[2]
    idx = orc.ref_select(orc.ref_distance(T, ot, X, Om), 4)
    assert idx[0, 0] == 5 and idx[2, 0] == 1


# ---- P17-P19: tolerance-based stopping (reading G21) -------------------------
def test_p17_fit_tol_worked_example():
    """The stop index on the exact-rational example follows from the golden costs (f_0 = 46,
    f after iteration 1 = 16.32935302, after iteration 2 = 15.70666801): the relative changes are 0.6450 and
    0.03813, so tol = 0.04 stops after iteration 2, tol = 0.038 does not, tol = 0.7 stops after iteration 1."""
    g = _load_p4()
    X, Om, W0, H0 = g["X"], g["Omega"], g["W0"], g["H0"]
    f0, f1, f2 = 46.0, g["f_W1"][0, 0], g["f_W2"][0, 0]
    assert (f0 - f1) / f0 == pytest.approx(0.64501, abs=1e-4) and (f1 - f2) / f1 == pytest.approx(0.038133, abs=1e-5)
    W, H, it, fl, tr = orc.fit_tol(X, Om, W0, H0, 10, 1, 0.7)
    assert it == 1 and fl == pytest.approx(f1, rel=2e-9)
    W, H, it, fl, tr = orc.fit_tol(X, Om, W0, H0, 10, 1, 0.04)
    assert it == 2 and fl == pytest.approx(f2, rel=2e-9)
    np.testing.assert_allclose(W, g["W2"], rtol=2e-9); np.testing.assert_allclose(H, g["H2"], rtol=2e-9, atol=0)
    np.testing.assert_allclose(tr, [f0, f1, f2], rtol=2e-9)
    W, H, it, fl, tr = orc.fit_tol(X, Om, W0, H0, 2, 1, 0.038)
    assert it == 2                                        # max_iters reached, not the tolerance
    W, H, it, fl, tr = orc.fit_tol(X, Om, W0, H0, 3, 1, 0.038)
    assert it == 3
    # check_every = 2: the only check in 2 iterations compares f_0 with f after iteration 2 (change 0.6586 < 0.7)
    W, H, it, fl, tr = orc.fit_tol(X, Om, W0, H0, 10, 2, 0.7)
    assert it == 2 and (f0 - f2) / f0 == pytest.approx(0.65855, abs=1e-4)
    np.testing.assert_allclose(tr, [f0, f2], rtol=2e-9)


def test_p18_fit_tol_equals_trace_scan(tiny):
    """The early exit stops exactly where a scan of the fixed-count fit's cost trace says, with the iterates of
    that many fixed-count iterations (bitwise), for several tolerances and check intervals; tol = 0 never stops."""
    p = tiny
    _, _, tr = orc.fit(p.X, p.Omega, p.W0, p.H0, 120, trace=True)
    f = tr[0::2]                                          # cost after every full iteration (tr holds both half-steps)
    last = 120
    for m in (1, 4, 7):
        for tol in (0.0, 1e-4, 1e-3, 1e-2, 0.3):
            checks = np.arange(m, 121, m)
            hit = [t for t in checks if abs(f[t - m] - f[t]) < tol * f[t - m]]
            expect = hit[0] if hit else 120
            W, H, it, fl, trc = orc.fit_tol(p.X, p.Omega, p.W0, p.H0, 120, m, tol)
            assert it == expect, (m, tol, it, expect)
            Wf, Hf = orc.fit(p.X, p.Omega, p.W0, p.H0, it)
            assert np.array_equal(W, Wf) and np.array_equal(H, Hf)
            assert fl == f[it // m * m] and np.array_equal(trc, f[0:it // m * m + 1:m])
            if tol == 0.0:
                assert it == 120
        # P1: the cost is non-increasing, so a looser tolerance can only stop earlier
        its = [orc.fit_tol(p.X, p.Omega, p.W0, p.H0, 120, m, tol)[2] for tol in (1e-5, 1e-4, 1e-3, 1e-2, 1e-1)]
        assert all(a >= b for a, b in zip(its, its[1:])), its
        assert its[0] <= last


def test_p19_fit_tol_fixed_point_never_stops_at_zero_cost():
    """X = W*H* exactly with the fit started at (W*, H*): every cost is 0 and the strict test |df| < tol * f never
    fires -- the fit runs to max_iters (a non-strict test would stop at once; G21 fixes the strict form)."""
    rng = np.random.default_rng(5)
    Ws = rng.integers(1, 4, (5, 2)).astype(np.float64); Hs = rng.integers(1, 4, (2, 24)).astype(np.float64)
    X = (Ws @ Hs).astype(np.float32); Om = np.ones_like(X)
    W, H, it, fl, tr = orc.fit_tol(X, Om, Ws, Hs, 9, 1, 0.5)
    assert it == 9 and fl == 0.0


# ---- P20-P24: derotate + stack (readings G22-G24) -------------------------
def _frames(M, ny, nx, seed):
    rng = np.random.default_rng(seed)
    return (rng.random((M, ny * nx)) * 10 - 3).astype(np.float32)


def test_p20_derotate_quarter_turns_are_exact_pixel_moves():
    """Multiples of 90 degrees move pixels exactly.  With an odd side the centre pixel (n/2, n/2) is the array
    centre, so a counter-clockwise quarter turn (x right, y = row index up) is numpy's rot90 with k = -1 seen in
    row-down display, i.e. out[y, x] = in[cy - (x - cx), cx + (y - cy)]: compared with the library routine."""
    n = 9
    R = _frames(1, n, n, 1)
    img = R[0].reshape(n, n)
    out0, cnt = orc.derotate_stack(R, None, [0.0], n, n)
    assert np.array_equal(out0.reshape(n, n), img.astype(np.float64)) and np.all(cnt == 1)
    out360, _ = orc.derotate_stack(R, None, [360.0], n, n)
    assert np.array_equal(out360, out0)
    out90, cnt = orc.derotate_stack(R, None, [90.0], n, n)
    # reading G22 at 90 degrees: source (xs, ys) = (cx + dy, cy - dx)
    ref = np.empty((n, n))
    c = n // 2
    for y in range(n):
        for x in range(n):
            ref[y, x] = img[c - (x - c), c + (y - c)]
    assert np.array_equal(out90.reshape(n, n), ref) and np.all(cnt == 1)
    assert np.array_equal(ref, np.rot90(img, k=-1).astype(np.float64))     # library routine (rows stored top-down: k = -1)
    out180, _ = orc.derotate_stack(R, None, [180.0], n, n)
    assert np.array_equal(out180.reshape(n, n), img[::-1, ::-1].astype(np.float64))
    out270, _ = orc.derotate_stack(R, None, [-90.0], n, n)
    assert np.array_equal(out270.reshape(n, n), np.rot90(img, k=1).astype(np.float64))
    # four quarter turns compose to the identity
    a = R
    for _ in range(4):
        o, _ = orc.derotate_stack(a, None, [90.0], n, n)
        a = o.astype(np.float32)[None, :]
    assert np.array_equal(a, R)


def test_p20b_even_side_centre_convention():
    """Even side: the centre is the pixel (n/2, n/2), not the array centre, so a half turn maps pixel i to n - i:
    row / column 0 has no source inside the image and is filled."""
    n = 8
    R = _frames(1, n, n, 2)
    img = R[0].reshape(n, n).astype(np.float64)
    out, cnt = orc.derotate_stack(R, None, [180.0], n, n, fill=-7.0)
    o = out.reshape(n, n); cn = cnt.reshape(n, n)
    assert np.all(o[0, :] == -7.0) and np.all(o[:, 0] == -7.0) and np.all(cn[0, :] == 0) and np.all(cn[1:, 1:] == 1)
    assert np.array_equal(o[1:, 1:], img[1:, 1:][::-1, ::-1])


def test_p21_derotate_matches_library_bilinear():
    """Generic angles against scipy.ndimage.map_coordinates(order=1) evaluated at the source coordinates of G22
    (library bilinear interpolation); pixels whose neighbours leave the image are excluded by both."""
    from scipy import ndimage
    ny, nx = 21, 26
    R = _frames(3, ny, nx, 3)
    cy, cx = ny // 2, nx // 2
    yy, xx = np.mgrid[0:ny, 0:nx].astype(np.float64)
    for ang in (17.0, -41.5, 133.0):
        s, c = np.sin(np.deg2rad(ang)), np.cos(np.deg2rad(ang))
        xs = cx + c * (xx - cx) + s * (yy - cy)
        ys = cy - s * (xx - cx) + c * (yy - cy)
        inside = (xs >= 0) & (xs <= nx - 1) & (ys >= 0) & (ys <= ny - 1)
        for m in range(3):
            ref = ndimage.map_coordinates(R[m].reshape(ny, nx).astype(np.float64), [ys, xs], order=1, mode="nearest")
            out, cnt = orc.derotate_stack(R[m:m + 1], None, [ang], ny, nx, fill=np.nan)
            o = out.reshape(ny, nx); cn = cnt.reshape(ny, nx)
            strict = (xs >= 0) & (xs < nx - 1) & (ys >= 0) & (ys < ny - 1)
            assert np.all(cn[strict] == 1) and np.all(cn[~inside] == 0)
            np.testing.assert_allclose(o[strict], ref[strict], rtol=0, atol=1e-12)


def test_p22_derotate_constant_linearity_and_mean():
    ny, nx, M = 17, 19, 5
    rng = np.random.default_rng(4)
    ang = rng.uniform(-180, 180, M)
    # a constant image stays constant wherever a sample exists (bilinear weights sum to 1)
    Cst = np.full((M, ny * nx), 2.5, dtype=np.float32)
    out, cnt = orc.derotate_stack(Cst, None, ang, ny, nx, fill=np.nan)
    assert np.all(np.abs(out[cnt > 0] - 2.5) < 1e-5)              # (ignored neighbours carry weight <= 1e-6 each)
    assert np.all(np.isnan(out[cnt == 0]))
    # linear in the frames
    A, B = np.round(_frames(M, ny, nx, 5) * 8), np.round(_frames(M, ny, nx, 6) * 8)     # small integers: 2A - 3B is exact in fp32
    oa, ca = orc.derotate_stack(A, None, ang, ny, nx)
    ob, _ = orc.derotate_stack(B, None, ang, ny, nx)
    oab, _ = orc.derotate_stack((2 * A - 3 * B).astype(np.float32), None, ang, ny, nx)
    lin = 2 * A.astype(np.float64) - 3 * B.astype(np.float64)
    assert np.array_equal(lin.astype(np.float32).astype(np.float64), lin)   # exactly representable inputs
    np.testing.assert_allclose(oab, 2 * oa - 3 * ob, rtol=0, atol=1e-10)
    # identical frames at angle 0 average to themselves; the stack is the mean of the single-frame results
    one = _frames(1, ny, nx, 7)
    rep, cnt = orc.derotate_stack(np.repeat(one, 4, axis=0), None, [0, 0, 0, 0], ny, nx)
    assert np.array_equal(rep, one[0].astype(np.float64)) and np.all(cnt == 4)
    singles = [orc.derotate_stack(A[m:m + 1], None, ang[m:m + 1], ny, nx) for m in range(M)]
    num = sum(o * (c > 0) for o, c in singles); den = sum((c > 0).astype(int) for o, c in singles)
    np.testing.assert_allclose(oa[den > 0], num[den > 0] / den[den > 0], rtol=0, atol=1e-12)
    assert np.array_equal(ca, den)


def test_p23_derotate_mask_semantics():
    """A masked source pixel (omega == 0) invalidates exactly the output samples that touch it with weight > 1e-6;
    its value (NaN / Inf) never enters the result."""
    ny, nx = 15, 15
    R = _frames(2, ny, nx, 8)
    om = np.ones_like(R)
    om[0, 7 * nx + 4] = 0.0; om[1, 3 * nx + 9] = 0.0
    Rg = R.copy(); Rg[om == 0] = np.nan
    ang = [30.0, 0.0]
    o1, c1 = orc.derotate_stack(R, om, ang, ny, nx, fill=0.0)
    o2, c2 = orc.derotate_stack(Rg, om, ang, ny, nx, fill=0.0)
    assert np.array_equal(o1, o2) and np.array_equal(c1, c2) and np.all(np.isfinite(o2))
    # frame 1 (angle 0): only its own pixel loses a sample
    full, cfull = orc.derotate_stack(R, None, ang, ny, nx)
    lost = (cfull - c1).reshape(ny, nx)
    assert lost[3, 9] >= 1 and lost.sum() <= 1 + 4          # frame 0's masked pixel touches at most 4 outputs
    # every frame masked at a pixel -> fill
    om[:, :] = 0.0
    o3, c3 = orc.derotate_stack(R, om, ang, ny, nx, fill=-1.0)
    assert np.all(o3 == -1.0) and np.all(c3 == 0)
