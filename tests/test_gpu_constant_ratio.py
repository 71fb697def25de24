"""f4 parity: the constant-photometric-ratio solve through the C ABI against oracle/constant_ratio.py (reading R1 of
DESIGN.md section 15).  Bars as for the free solve (BASELINE.json north_star): coefficients 1e-8 relative (norm-wise),
D within 1e-6 x noise RMS; the constraint itself to rounding."""
import numpy as np
import pytest
import torch

import oracle
from oracle import constant_ratio as cr
from paper_2509_18544_b200 import SfftPlan, starfield

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("nx,ny,L,DK,DB", [(100, 72, 5, 1, 1), (128, 64, 3, 2, 0), (90, 110, 7, 3, 2), (64, 64, 5, 0, 1)])
def test_constant_ratio_parity(nx, ny, L, DK, DB):
    S, R = starfield.random_pair(nx, ny, seed=nx + L)
    p = SfftPlan(nx, ny, L, DK, DB)
    p.build_system(dev(S), dev(R))
    p.solve_constant_ratio()
    D, c = p.subtract(); p.sync_status()
    c, D = c.cpu().numpy(), D.cpu().numpy()
    G0, h0 = oracle.build_system(S, R, None, L, DK, DB)
    c0 = cr.solve_constant_ratio(G0, h0, L, DK, DB)
    assert np.max(np.abs(c - c0)) <= 1e-8 * np.max(np.abs(c0))
    LL, NK = L * L, oracle.num_poly(DK)
    for t in range(1, NK):
        assert abs(c[t * LL:(t + 1) * LL].sum()) <= 1e-11 * np.abs(c[:NK * LL]).sum()
    D0 = oracle.subtract(S, R, L, DK, DB, c0)
    assert np.max(np.abs(D - D0)) <= 1e-6 * 20.0
    # and a second call on the same plan (workspace reuse), after a free solve in between
    p.solve()
    cf = p.subtract()[1].cpu().numpy()
    assert np.max(np.abs(cf - oracle.solve(G0, h0))) <= 1e-8 * np.max(np.abs(c0))
    p.solve_constant_ratio()
    c2 = p.subtract()[1].cpu().numpy()
    assert np.max(np.abs(c2 - c)) <= 1e-12 * np.max(np.abs(c))
    p.destroy()


def test_constant_ratio_config1_like_1024():
    """configs[1] recipe (1024 x 1024, L = 11, DK = 2, DB = 1, n = 729): five constraints on the full-size system."""
    cfg = starfield.make_pair(1)
    S, R = cfg["S"], cfg["R"]
    L, DK, DB = 11, 2, 1
    p = SfftPlan(1024, 1024, L, DK, DB)
    p.build_system(dev(S), dev(R))
    p.solve_constant_ratio()
    D, c = p.subtract(); p.sync_status()
    c = c.cpu().numpy()
    G0, h0 = oracle.build_system(S, R, None, L, DK, DB)          # direct pixel sums: seconds at this size
    c0 = cr.solve_constant_ratio(G0, h0, L, DK, DB)
    assert np.max(np.abs(c - c0)) <= 1e-8 * np.max(np.abs(c0))
    rng = np.random.default_rng(2)
    xs, ys = rng.integers(0, 1024, 200), rng.integers(0, 1024, 200)
    Ds = oracle.subtract_at(S, R, L, DK, DB, c0, xs, ys)
    assert np.max(np.abs(D.cpu().numpy()[ys, xs] - Ds)) <= 1e-6 * cfg["noise_rms"]
    p.destroy()
