"""sfft_solve_static (include/sfft.h): the allocation-free variant of step a4, whose scratch is a file-scope
`static __device__` array, against the existing plan path (sfft_solve) on the same systems, calls back to back.

Collected last on purpose (the suite runs with pytest -x).  Passes alone in a fresh process and after the other
tests: it owns its plans and touches no state of theirs; the static array is shared by every call in the process
and carries the previous call's contents, which is exactly what the back-to-back calls below exercise.
Bar: the coefficient tolerance of tests/test_gpu_parity.py (north_star: max|dc| <= 1e-8 max|c| per block).
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2509_18544_b200 import SfftError, SfftPlan, sfft, solve_static, starfield

pytestmark = pytest.mark.gpu

TOL_C = 1e-8


def assert_coeffs(c, c0, nker):
    assert np.max(np.abs(c - c0)[:nker]) <= TOL_C * np.max(np.abs(c0[:nker]))
    assert np.max(np.abs(c - c0)[nker:]) <= TOL_C * np.max(np.abs(c0[nker:]))


def plan_system(nx, ny, L, DK, DB, seed):
    """G, h (device) and the coefficients of the existing path for one seeded synthetic pair."""
    S, R = starfield.random_pair(nx, ny, seed=seed)
    p = SfftPlan(nx, ny, L, DK, DB)
    dS, dR = torch.from_numpy(S).cuda(), torch.from_numpy(R).cuda()
    p.build_system(dS, dR)
    G, h = p.get_system()
    p.solve()
    _, c = p.subtract()
    p.sync_status()
    nker = L * L * (DK + 1) * (DK + 2) // 2
    return G, h, c.cpu().numpy(), nker


def test_static_solve_matches_plan_path_on_calls_in_a_row():
    # n = 732 (12 blocks, last one 28 wide: the headline system size) and n = 153 (3 blocks, last one 25 wide)
    big = plan_system(420, 400, 11, 2, 2, seed=5)
    small = plan_system(330, 300, 5, 2, 1, seed=6)
    assert big[0].shape[0] == 732 and small[0].shape[0] == 153
    results = []
    for G, h, c_plan, nker in (big, small, big, small):          # back to back, the scratch keeps the last call's contents
        G_before, h_before = G.clone(), h.clone()
        c = torch.full_like(h, float("nan"))
        solve_static(G, h, c)
        assert torch.equal(G, G_before) and torch.equal(h, h_before)   # inputs are not modified
        c = c.cpu().numpy()
        assert np.all(np.isfinite(c))
        assert_coeffs(c, c_plan, nker)
        assert_coeffs(c, oracle.solve(G.cpu().numpy(), h.cpu().numpy()), nker)
        results.append(c)
    # the same system gives the same bits whatever the scratch held before
    assert np.array_equal(results[0], results[2]) and np.array_equal(results[1], results[3])


def test_static_solve_on_a_side_stream():
    G, h, c_plan, nker = plan_system(330, 300, 5, 1, 0, seed=7)
    st = torch.cuda.Stream()
    torch.cuda.synchronize()
    c = torch.empty_like(h)
    solve_static(G, h, c, stream=st)                              # blocks until the solve is done
    assert_coeffs(c.cpu().numpy(), c_plan, nker)


def test_static_solve_limits_and_errors():
    assert sfft.SOLVE_STATIC_MAX_N == 1024
    n = sfft.SOLVE_STATIC_MAX_N + 1
    G = torch.eye(n, dtype=torch.float64, device="cuda")
    h = torch.ones(n, dtype=torch.float64, device="cuda")
    c = torch.zeros(n, dtype=torch.float64, device="cuda")
    with pytest.raises(SfftError) as ei:
        solve_static(G, h, c)
    assert ei.value.code == -1 and "1024" in str(ei.value) and "SFFT_SOLVE_STATIC_MAX_N" in str(ei.value)
    assert torch.count_nonzero(c).item() == 0                     # rejected before any work
    lib = sfft.load_library()
    assert lib.sfft_solve_static(G.data_ptr(), h.data_ptr(), c.data_ptr(), 0, None) == -1
    assert lib.sfft_solve_static(None, h.data_ptr(), c.data_ptr(), 4, None) == -1
    # the largest size the array takes: a diagonally dominant SPD matrix with a known solution
    n = sfft.SOLVE_STATIC_MAX_N
    rng = np.random.default_rng(11)
    A = rng.standard_normal((n, n)) * 0.01
    Gh = A @ A.T + np.diag(rng.uniform(1.0, 4.0, n))
    x = rng.standard_normal(n)
    c = torch.empty(n, dtype=torch.float64, device="cuda")
    solve_static(torch.from_numpy(Gh).cuda(), torch.from_numpy(Gh @ x).cuda(), c)
    assert np.max(np.abs(c.cpu().numpy() - x)) <= 1e-10 * np.max(np.abs(x))
    # not positive definite: reported, and the next call works
    Gbad = torch.from_numpy(Gh.copy()).cuda()
    Gbad[100, 100] = -1.0
    with pytest.raises(SfftError) as ei:
        solve_static(Gbad, torch.from_numpy(Gh @ x).cuda(), c)
    assert ei.value.code == -5
    solve_static(torch.from_numpy(Gh).cuda(), torch.from_numpy(Gh @ x).cuda(), c)
    assert np.max(np.abs(c.cpu().numpy() - x)) <= 1e-10 * np.max(np.abs(x))
