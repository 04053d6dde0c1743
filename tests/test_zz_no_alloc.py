"""nmf_objective_static (include/nmf.h): the cost of Eq. 2 for callers that may not allocate -- no plan, no workspace,
scratch in a fixed device array inside the library.  Checked against the existing path (nmf_objective through a plan)
on two calls in a row, the second on a smaller problem so that the shared scratch still holds partial sums of the
first call beyond what the second one writes.  Collected last on purpose (file name): the suite runs with pytest -x.
"""
import ctypes

import numpy as np
import pytest
import torch

from paper_2309_04623_b200 import nmf
from gpu_util import TOL_OBJECTIVE, dev

pytestmark = pytest.mark.gpu


def _problem(N, P, K, seed):
    rng = np.random.default_rng(seed)
    X = (rng.random((N, P)) * 10).astype(np.float32)
    Om = (rng.random((N, P)) * (rng.random((N, P)) > 0.2)).astype(np.float32)
    W = (0.1 + 0.9 * rng.random((N, K))).astype(np.float32)
    H = (0.1 + 0.9 * rng.random((K, P))).astype(np.float32)
    return dev(X), dev(Om), dev(W), dev(H)


def test_objective_static_matches_plan_objective_twice():
    shapes = [(200, 128 * 300 + 36, 50, 1), (33, 1028, 17, 2)]       # 301 blocks, then 9 blocks (ragged last block)
    cases = [(s, _problem(*s)) for s in shapes]
    want = []
    for (N, P, K, _), (X, Om, W, H) in cases:                          # the existing path: plan + workspace
        want.append(nmf.Plan(N, P, K).objective(X, Om, W, H))
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    free_before = None
    for i, (_, (X, Om, W, H)) in enumerate(cases):                     # two calls in a row, no synchronisation between
        if i == 1:
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info()[0]
        nmf.objective_static(X, Om, W, H, out[i:i + 1])
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    got = out.cpu().numpy()
    for g, w in zip(got, want):
        assert np.isfinite(g) and abs(g - w) <= TOL_OBJECTIVE * abs(w), (g, w)
        assert g == w                                                  # same kernels, same fixed summation order
    assert free_after >= free_before                                   # the second call took no device memory
    # and again in the other order: the scratch now holds the small problem's partials
    for i, (_, (X, Om, W, H)) in reversed(list(enumerate(cases))):
        out.zero_()
        nmf.objective_static(X, Om, W, H, out[i:i + 1])
        torch.cuda.synchronize()
        assert out[i].item() == want[i]


def test_objective_static_rejects_sizes_beyond_its_scratch():
    L = nmf.lib()
    X, Om, W, H = _problem(4, 64, 2, 3)
    out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    args = (X.data_ptr(), Om.data_ptr(), W.data_ptr(), H.data_ptr())
    STATIC_LIMIT = -7
    # P beyond NMF_STATIC_MAX_P: rejected before anything is launched or read
    assert L.nmf_objective_static(*args, 4, nmf.STATIC_MAX_P + 4, 2, out.data_ptr(), None) == STATIC_LIMIT
    assert L.nmf_objective_static(*args, 4, 1 << 40, 2, out.data_ptr(), None) == STATIC_LIMIT
    assert b"nmf_objective_static" in L.nmf_status_string(STATIC_LIMIT)
    assert L.nmf_objective_static(*args, 0, 64, 2, out.data_ptr(), None) == -1
    assert L.nmf_objective_static(*args, 4, 64, 2, None, None) == -1
    assert L.nmf_objective_static(*args, 4, 64, 129, out.data_ptr(), None) == -3
    torch.cuda.synchronize()
    assert out.item() == -1.0
    # the limit itself is accepted (shape only: 2048^2 pixels, one frame, one component)
    P = nmf.STATIC_MAX_P
    Xb = torch.full((1, P), 2.0, device="cuda"); Ob = torch.ones(1, P, device="cuda")
    Wb = torch.ones(1, 1, device="cuda"); Hb = torch.ones(1, P, device="cuda")
    nmf.objective_static(Xb, Ob, Wb, Hb, out)
    torch.cuda.synchronize()
    assert out.item() == float(P)                                      # sum of 1 * (2 - 1)^2
