"""f1 parity: the decorrelation kernel through the C ABI against oracle/decorrelation.py (readings
D1-D5 of DESIGN.md section 13).  Bars: local kernel 1e-14 x sum |a|; stamp
1e-13 x max W^ (rounding of an N^2-term sum scaled by the largest Fourier weight); decorrelated image
1e-6 x noise RMS like D itself (BASELINE.json north_star)."""
import numpy as np
import pytest
import torch

import oracle
from oracle import decorrelation as deco
from paper_2509_18544_b200 import SfftPlan, starfield
from paper_2509_18544_b200.sfft import SfftError

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _stamp(P, seed, sigma):
    rng = np.random.default_rng(seed)
    w = (P - 1) // 2
    yy, xx = np.mgrid[-w:w + 1, -w:w + 1]
    st = np.exp(-0.5 * (((xx - 0.3) / sigma) ** 2 + ((yy + 0.2) / (1.2 * sigma)) ** 2)) + 0.003 * rng.random((P, P))
    return st / st.sum()


def _wmax(K, PS, PR, vS, vR, N):
    F = deco.noise_power(K, PS, PR, vS, vR, N)
    return float(np.sqrt(F[0, 0] / F.min()))


@pytest.mark.parametrize("L,DK,DB,x,y", [(5, 0, 0, 3.0, 4.0), (7, 1, 0, 0.0, 71.0), (11, 2, 2, 50.5, 36.0),
                                         (5, 3, 1, 99.0, 0.0)])
def test_local_kernel_parity(L, DK, DB, x, y):
    nx, ny = 100, 72
    p = SfftPlan(nx, ny, L, DK, DB)
    c = np.random.default_rng(L + DK).standard_normal(p.n)
    K = p.local_kernel(x, y, coeffs=dev(c)).cpu().numpy()
    K0 = deco.local_kernel(c, L, DK, x, y, nx, ny)
    assert np.max(np.abs(K - K0)) <= 1e-14 * np.abs(c).sum()
    p.destroy()


def test_local_kernel_defaults_to_the_plan_solution():
    nx, ny, L, DK, DB = 100, 72, 5, 1, 1
    S, R = starfield.random_pair(nx, ny, seed=5)
    p = SfftPlan(nx, ny, L, DK, DB)
    with pytest.raises(SfftError):
        p.local_kernel(10, 10)                       # nothing solved yet
    p.build_system(dev(S), dev(R)); p.solve()
    D, c = p.subtract(); p.sync_status()
    K = p.local_kernel(20, 30).cpu().numpy()
    K0 = deco.local_kernel(c.cpu().numpy(), L, DK, 20, 30, nx, ny)
    assert np.max(np.abs(K - K0)) <= 1e-14 * np.abs(c.cpu().numpy()).sum()
    p.destroy()


@pytest.mark.parametrize("Ld,Lk,Lp,N,vS,vR", [
    (11, 11, 11, 64, 25.0, 25.0 / 9),    # Roman-like: template three times deeper (configs[2])
    (21, 11, 15, 96, 64.0, 7.0),         # N not a power of two, PSF stamp larger than the kernel
    (5, 3, 3, 5, 1.0, 1.0),              # the smallest admissible grid: N = Lk + Lp - 1 = L
    (7, 21, 9, 128, 4.0, 0.0),           # var_R = 0: only the science noise, W^ = |P_R^(0)| / |P_R^|
    (1, 1, 1, 8, 2.0, 3.0),              # single taps: F constant, W = delta
    (21, 11, 11, 257, 30.0, 10.0),       # odd prime N, the largest stamp a plan takes (L = 21)
])
def test_decorrelation_stamp_parity(Ld, Lk, Lp, N, vS, vR):
    K = _stamp(Lk, 1, 0.8) * 1.1 if Lk > 1 else np.array([[1.3]])
    PS = _stamp(Lp, 2, 0.9) if Lp > 1 else np.array([[1.0]])
    PR = _stamp(Lp, 3, 0.8) if Lp > 1 else np.array([[0.9]])
    p = SfftPlan(max(64, 2 * Ld), max(64, 2 * Ld) + (N * N) // 32, Ld, 0, 0)  # tall enough for the N x N scratch
    W = p.decorrelation_stamp(dev(K), dev(PS), dev(PR), vS, vR, N).cpu().numpy()
    W0 = deco.decorrelation_stamp(K, PS, PR, vS, vR, N, Ld)
    assert np.max(np.abs(W - W0)) <= 1e-13 * _wmax(K, PS, PR, vS, vR, N)
    p.destroy()


def test_decorrelate_difference_image_end_to_end():
    """Steps 5-7 on one plan: cross-convolve, subtract, local kernel at the frame centre,
    decorrelation stamp, and the stamp applied to D and to the cross-convolved science image."""
    nx, ny, L, DK, DB, N = 100, 72, 7, 1, 1, 48
    S, R = starfield.random_pair(nx, ny, seed=21)
    psfS, psfR = _stamp(L, 4, 0.9), _stamp(L, 5, 0.8)
    vS, vR = 400.0, 400.0
    p = SfftPlan(nx, ny, L, DK, DB)
    Sc, Rc = p.cross_convolve(dev(S), dev(R), dev(psfS), dev(psfR))
    p.build_system(Sc, Rc); p.solve()
    D, c = p.subtract(); p.sync_status()
    K = p.local_kernel((nx - 1) / 2, (ny - 1) / 2)
    W = p.decorrelation_stamp(K, dev(psfS), dev(psfR), vS, vR, N)
    Dd = p.convolve_stamp(D, W).cpu().numpy()
    Sd = p.convolve_stamp(Sc, W).cpu().numpy()
    # oracle chain on the same inputs
    Sc0, Rc0 = oracle.convolve_stamp(S, psfR), oracle.convolve_stamp(R, psfS)
    G0, h0 = oracle.build_system(Sc0, Rc0, None, L, DK, DB)
    c0 = oracle.solve(G0, h0)
    D0 = oracle.subtract(Sc0, Rc0, L, DK, DB, c0)
    K0 = deco.local_kernel(c0, L, DK, (nx - 1) / 2, (ny - 1) / 2, nx, ny)
    W0 = deco.decorrelation_stamp(K0, psfS, psfR, vS, vR, N, L)
    rms = 20.0
    assert np.max(np.abs(W.cpu().numpy() - W0)) <= 1e-8 * _wmax(K0, psfS, psfR, vS, vR, N)   # carries the 1e-8 of c
    assert np.max(np.abs(Dd - oracle.convolve_stamp(D0, W0))) <= 1e-6 * rms
    assert np.max(np.abs(Sd - oracle.convolve_stamp(Sc0, W0))) <= 1e-6 * rms
    p.destroy()


def test_decorrelation_stamp_errors():
    p = SfftPlan(64, 64, 5, 0, 0)
    d3 = torch.zeros((3, 3), dtype=torch.float64, device="cuda"); d3[1, 1] = 1.0
    box = torch.zeros((3, 3), dtype=torch.float64, device="cuda"); box[1, 0] = box[1, 1] = 0.5
    with pytest.raises(SfftError):
        p.decorrelation_stamp(d3, box, box, 1.0, 1.0, 8)        # P^ vanishes at kx = N/2
    with pytest.raises(SfftError):
        p.decorrelation_stamp(d3, d3, d3, 1.0, 1.0, 4)          # N < Lk + Lp - 1
    with pytest.raises(SfftError):
        p.decorrelation_stamp(d3, d3, d3, 0.0, 0.0, 8)          # both variances zero
    with pytest.raises(SfftError):
        p.decorrelation_stamp(d3, d3, d3, 1.0, 1.0, 1024)       # scratch too small on this plan
    even = torch.zeros((4, 4), dtype=torch.float64, device="cuda")
    with pytest.raises(SfftError):
        p.decorrelation_stamp(even, d3, d3, 1.0, 1.0, 8)        # even stamp
    W = p.decorrelation_stamp(d3, d3, d3, 1.0, 1.0, 8).cpu().numpy()   # the plan still works afterwards
    ref = np.zeros((5, 5)); ref[2, 2] = 1.0
    assert np.max(np.abs(W - ref)) < 1e-15
    p.destroy()


def test_decorrelated_science_psf_on_a_small_plan():
    """"Also apply the decorrelation kernel to the science PSF": a 25 x 25 PSF stamp convolved with the
    11 x 11 decorrelation stamp on a plan of the stamp's size (circular at 25 x 25, like any frame: reading C6)."""
    P, L, N = 25, 11, 64
    yy, xx = np.mgrid[0:P, 0:P] - (P - 1) / 2.0
    psf_img = np.exp(-0.5 * ((xx / 1.1) ** 2 + (yy / 1.3) ** 2)); psf_img /= psf_img.sum()
    K, PS, PR = _stamp(L, 7, 0.7), _stamp(L, 8, 0.9), _stamp(L, 9, 0.8)
    big = SfftPlan(128, 128, L, 0, 0)          # the stamp is built once on the frame's plan (its scratch holds N x N) ...
    W = big.decorrelation_stamp(dev(K), dev(PS), dev(PR), 9.0, 1.0, N)
    p = SfftPlan(P, P, L, 0, 0)                # ... and applied to the PSF on a plan of the PSF stamp's size
    W2 = p.decorrelation_stamp(dev(K), dev(PS), dev(PR), 9.0, 1.0, N)   # (every plan's scratch holds a 64 x 64 grid: the FFT
    assert torch.equal(W, W2)                                            #  grid is at least 1024 x 512)
    out = p.convolve_stamp(dev(psf_img), W).cpu().numpy()
    W0 = deco.decorrelation_stamp(K, PS, PR, 9.0, 1.0, N, L)
    ref = oracle.convolve_stamp(psf_img, W0)
    assert np.max(np.abs(out - ref)) <= 1e-12 * np.abs(W0).sum() * psf_img.max()
    assert abs(out.sum() - W0.sum()) <= 1e-12 * np.abs(W0).sum()     # a unit-flux PSF keeps the stamp's flux scale
    p.destroy(); big.destroy()
