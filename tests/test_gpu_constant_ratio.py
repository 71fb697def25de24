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


def test_constant_ratio_as_plan_mode_single_and_batched():
    """sfft_set_constant_ratio: the auxiliary solves ride behind the factorisation (factor stream) and every solve is
    corrected: the single-pair path, the pipelined batched path (groups of 4 + a ragged group) and the host path, each
    image against the oracle's constrained solution; switching the mode off restores the free solution."""
    nx, ny, L, DK, DB = 100, 72, 5, 2, 1
    _, R = starfield.random_pair(nx, ny, seed=200)
    Ss = [starfield.random_pair(nx, ny, seed=201 + b)[0] for b in range(6)]
    G0, _ = oracle.build_system(Ss[0], R, None, L, DK, DB)
    c0s, cfree = [], []
    for S in Ss:
        _, h0 = oracle.build_system(S, R, None, L, DK, DB)
        c0s.append(cr.solve_constant_ratio(G0, h0, L, DK, DB)); cfree.append(oracle.solve(G0, h0))
    p = SfftPlan(nx, ny, L, DK, DB)
    p.set_constant_ratio(True)
    # single pair, twice (the factor and its auxiliary solves are redone per build_system)
    for b in (0, 1):
        p.build_system(dev(Ss[b]), dev(R)); p.solve()
        D, c = p.subtract(); p.sync_status()
        assert np.max(np.abs(c.cpu().numpy() - c0s[b])) <= 1e-8 * np.max(np.abs(c0s[b]))
        assert np.max(np.abs(D.cpu().numpy() - oracle.subtract(Ss[b], R, L, DK, DB, c0s[b]))) <= 1e-6 * 20.0
    # batched
    p.set_template(dev(R))
    Ds, cs = p.subtract_batch([dev(s) for s in Ss]); p.sync_status()
    cs = cs.cpu().numpy()
    for b in range(6):
        assert np.max(np.abs(cs[b] - c0s[b])) <= 1e-8 * np.max(np.abs(c0s[b])), b
        assert np.max(np.abs(Ds[b].cpu().numpy() - oracle.subtract(Ss[b], R, L, DK, DB, c0s[b]))) <= 1e-6 * 20.0, b
    # host path
    Dh, ch = p.difference_host(torch.from_numpy(Ss[2]).pin_memory(), torch.from_numpy(R).pin_memory())
    assert np.max(np.abs(ch.numpy() - c0s[2])) <= 1e-8 * np.max(np.abs(c0s[2]))
    # mode switched on only after set_template (auxiliary solves made lazily), then off again
    q = SfftPlan(nx, ny, L, DK, DB)
    q.set_template(dev(R))
    q.set_constant_ratio(True)
    _, cq = q.subtract_batch([dev(Ss[3]), dev(Ss[4])]); q.sync_status()
    assert np.max(np.abs(cq.cpu().numpy()[1] - c0s[4])) <= 1e-8 * np.max(np.abs(c0s[4]))
    q.set_constant_ratio(False)
    _, cq = q.subtract_batch([dev(Ss[3]), dev(Ss[4])]); q.sync_status()
    assert np.max(np.abs(cq.cpu().numpy()[0] - cfree[3])) <= 1e-8 * np.max(np.abs(cfree[3]))
    p.destroy(); q.destroy()
