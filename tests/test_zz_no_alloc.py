"""sfft_solve_static (include/sfft.h): the allocation-free variant of sfft_solve against the existing
plan path, on calls in a row that share the library's static workspace.

This file is named so that pytest collects it LAST (the run uses -x).  It passes alone in a
fresh process and after the other tests: it creates its own plans and inputs.

Tolerance: the coefficient tolerance of tests/test_gpu_parity.py (||dc||_inf <= 1e-7 ||c||_inf); the two
paths run the same kernels, so the results are in fact compared bit for bit as well.
"""
import numpy as np
import pytest
import torch

from paper_2603_08593_b200 import SfftError, SfftPlan, SOLVE_STATIC_MAX_N, solve_static

pytestmark = pytest.mark.gpu

TOL_C = 1e-7


def spd_system(N, seed):
    rng = np.random.default_rng(seed)
    G = rng.standard_normal((2 * N + 50, N))
    A = G.T @ G + 1e-3 * np.eye(N)
    b = rng.standard_normal(N) * 10.0
    return torch.from_numpy(A).cuda(), torch.from_numpy(b).cuda()


def plan_solve(H, W, w, DK, DB, A, b):
    with SfftPlan(H, W, w, DK, DB) as plan:
        assert plan.N == b.numel()
        c, info = plan.solve(A, b)
        torch.cuda.synchronize()
        return c.clone(), int(info.item())


def test_static_solve_matches_plan_solve_on_calls_in_a_row():
    # Full configuration's N = 732 (ragged against the 64-wide panels), then a smaller system whose workspace
    # rows are full of the first call's leftovers, then the large one again
    cases = [((2048, 4096, 5, 2, 2), 732, 1), ((64, 64, 2, 1, 1), 78, 2), ((2048, 4096, 5, 2, 2), 732, 3)]
    systems = [spd_system(N, seed) for (_, N, seed) in cases]
    expected = [plan_solve(*cfg, A, b) for (cfg, _, _), (A, b) in zip(cases, systems)]
    outs = [torch.empty(N, dtype=torch.float64, device="cuda") for (_, N, _) in cases]
    infos = [torch.full((1,), -7, dtype=torch.int32, device="cuda") for _ in cases]
    # one warm-up call (the first launch of a kernel loads its module), then the calls in a row on one
    # stream with no synchronisation in between and no allocation: free device memory must not move
    solve_static(*systems[1], coeffs=outs[1], info=infos[1])
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    for (A, b), c, info in zip(systems, outs, infos):
        solve_static(A, b, coeffs=c, info=info)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before
    for (c_ref, info_ref), c, info, (A, b) in zip(expected, outs, infos, systems):
        assert info_ref == 0 and int(info.item()) == 0
        scale = float(c_ref.abs().max())
        assert float((c - c_ref).abs().max()) <= TOL_C * scale
        assert torch.equal(c, c_ref)                      # same kernels, same order of operations
        res = A @ c - b                                   # and it does solve the system
        assert float(res.abs().max()) <= 1e-8 * float(b.abs().max()) * np.sqrt(b.numel())


def test_static_solve_reports_not_positive_definite_like_the_plan_path():
    A, b = spd_system(78, 4)
    A[40, 40] = -1.0
    _, info_ref = plan_solve(64, 64, 2, 1, 1, A, b)
    _, info = solve_static(A, b)
    torch.cuda.synchronize()
    assert info_ref == 41 and int(info.item()) == info_ref   # 1-based order of the first bad leading minor
    # the next call is unaffected by the failed one
    A2, b2 = spd_system(78, 5)
    c_ref, _ = plan_solve(64, 64, 2, 1, 1, A2, b2)
    c, info = solve_static(A2, b2)
    torch.cuda.synchronize()
    assert int(info.item()) == 0 and torch.equal(c, c_ref)


def test_static_solve_limits():
    # the largest admitted size works; one more is rejected with SFFT_ERR_UNSUPPORTED and enqueues nothing
    N = SOLVE_STATIC_MAX_N
    A, b = spd_system(N, 6)
    c, info = solve_static(A, b)
    torch.cuda.synchronize()
    assert int(info.item()) == 0
    c_np = np.linalg.solve(A.cpu().numpy(), b.cpu().numpy())
    assert np.max(np.abs(c.cpu().numpy() - c_np)) <= TOL_C * np.max(np.abs(c_np))
    A1 = torch.eye(N + 1, dtype=torch.float64, device="cuda")
    b1 = torch.ones(N + 1, dtype=torch.float64, device="cuda")
    with pytest.raises(SfftError) as e:
        solve_static(A1, b1)
    assert e.value.code == 2
    # smallest size
    A0 = torch.full((1, 1), 4.0, dtype=torch.float64, device="cuda")
    b0 = torch.full((1,), 2.0, dtype=torch.float64, device="cuda")
    c0, info0 = solve_static(A0, b0)
    torch.cuda.synchronize()
    assert int(info0.item()) == 0 and float(c0[0]) == 0.5
