"""Writes tests/golden/fullsize_*.npz: fp64 ORACLE results of the full-size, full-iteration configs that are too
slow to recompute inside a test run (STIS-shaped 200 it; component sweep K in {1,5,10,20,50,100}, 200 it each;
survey batch 64 problems x 300 it).  TEST INFRASTRUCTURE: calls only oracle/ and the seeded generators
(paper_2309_04623_b200/inputs.py holds none of the method's arithmetic); nothing here touches the CUDA path.

    python tests/golden/make_fullsize_goldens.py [case ...]      # cases: stis sweep_K100 ... survey ; default all

Each file holds, for its case (BASELINE.json configs; readings DESIGN.md section 3):
    W        [N,K] fp64      oracle coefficients after the config's iteration count (Eq. 3)
    f        ()    fp64      oracle objective, Eq. 2, at (W, H)
    cols     [C]   int64     sampled pixel columns: first / last 64, the occulting-wedge edges, seeded random ones
    Hc       [K,C] fp32      oracle H at those columns (fp64 result rounded once to fp32: 6e-8, tolerance is 1e-3)
    frames   [4]   int64     science frames projected on the oracle's H ...
    coef     [4,K] fp64      ... their coefficients after `proj_iters` projection iterations
    resid    [4,C] fp64      ... and target - coef.H at the sampled columns (0 where omega == 0)
    iters, proj_iters, seconds, threads
The survey file stacks the 64 problems along a leading axis (512 sampled columns per problem, no projection).
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import nmf_oracle as orc                      # noqa: E402
from paper_2309_04623_b200 import inputs                  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
PROJ_ITERS = 100
FRAMES = np.array([0, 9, 18, 31])


def sample_cols(S: int, n_random: int, seed: int = 0) -> np.ndarray:
    """first / last 64 pixels, both edges of the occulting band of inputs._stis_mask on 8 rows, seeded random ones"""
    P = S * S
    c, half = S // 2, max(1, int(round(30 * S / 1024)))
    rows = np.linspace(0, S - 1, 8).astype(np.int64)
    xs = np.array([c - half - 2, c - half - 1, c - half, c - half + 1, c + half - 2, c + half - 1, c + half, c + half + 1])
    edge = (rows[:, None] * S + xs[None, :]).ravel()
    rnd = np.random.default_rng(seed).integers(0, P, n_random)
    return np.unique(np.concatenate([np.arange(64), np.arange(P - 64, P), edge, rnd])).astype(np.int64)


def fit_case(p, with_projection: bool, n_random: int):
    t0 = time.time()
    W, H = orc.fit(p.X, p.Omega, p.W0, p.H0, p.iters)
    f = orc.objective(p.X, p.Omega, W, H)
    cols = sample_cols(p.S, n_random)
    out = dict(W=W, f=np.float64(f), cols=cols, Hc=H[:, cols].astype(np.float32), iters=p.iters)
    if with_projection:
        fr = FRAMES[FRAMES < p.M]
        C = orc.project(H, p.T[fr], p.omega_t[fr], p.C0[fr], PROJ_ITERS)
        R = orc.subtract(H, p.T[fr], C, p.omega_t[fr], None, 0.0)
        out.update(frames=fr, coef=C, resid=R[:, cols], proj_iters=PROJ_ITERS)
    out.update(seconds=time.time() - t0, threads=orc.num_threads())
    return out


def main(argv):
    cases = argv or ["stis", "sweep_K100", "sweep_K1", "sweep_K5", "sweep_K10", "sweep_K20", "survey", "sweep_K50"]
    lib = None
    for case in cases:
        path = os.path.join(HERE, f"fullsize_{case}.npz")
        if os.path.exists(path):
            print(f"{case}: exists, skipped", flush=True)
            continue
        t0 = time.time()
        if case == "survey":
            res = []
            for b in range(64):
                r = fit_case(inputs.make_survey_problem(b), False, 384)
                res.append(r)
                print(f"  survey problem {b}: {r['seconds']:.0f} s", flush=True)
            out = {k: np.stack([r[k] for r in res]) for k in ("W", "f", "cols", "Hc")}
            out.update(iters=res[0]["iters"], seconds=time.time() - t0, threads=res[0]["threads"])
        else:
            if lib is None:
                lib = inputs.make_stis()                   # library + science frames, shared by every sweep K
            if case == "stis":
                p = lib
            else:
                p = inputs.reinit(lib, int(case.split("K")[1]), case)
            out = fit_case(p, True, 4096)
        tmp = path + ".tmp.npz"
        np.savez_compressed(tmp, **out)
        os.replace(tmp, path)
        print(f"{case}: {time.time() - t0:.0f} s, f = {float(np.sum(out['f'])):.10e} -> {os.path.basename(path)}", flush=True)


if __name__ == "__main__":
    main(sys.argv[1:])
