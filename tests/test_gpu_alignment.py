"""f3 parity: affine resampling through the C ABI against oracle/alignment.py (readings A1-A4 of
DESIGN.md section 14).  Bars: nearest and masks bit-exact (index work; the source position is evaluated in the same
FP64 operations on both sides); the fill pattern identical; interpolated pixels within 1e-12 x max|img| (a 36-term
weighted sum with weights of order 1, each within a few ulp: DESIGN.md section 14)."""
import numpy as np
import pytest
import torch

from oracle import alignment as al
from paper_2509_18544_b200 import SfftPlan, starfield
from paper_2509_18544_b200.sfft import SfftError

pytestmark = pytest.mark.gpu

TOL_RS = 1e-12


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _rot(theta, sx, sy, tx, ty, nx, ny):
    """Rotation by theta about the frame centre with scales and a translation."""
    cx, cy = (nx - 1) / 2.0, (ny - 1) / 2.0
    c, s = np.cos(theta), np.sin(theta)
    M0, M1, M3, M4 = sx * c, -sy * s, sx * s, sy * c
    return [M0, M1, cx - M0 * cx - M1 * cy + tx, M3, M4, cy - M3 * cx - M4 * cy + ty]


def _check(img, M, method, fill=np.nan):
    ny, nx = img.shape
    p = SfftPlan(nx, ny, 3, 0, 0)
    out = p.resample_affine(dev(img), M, method=method, fill=fill).cpu().numpy()
    ref = al.resample_affine(img, M, method, fill)
    p.destroy()
    assert np.array_equal(np.isnan(out), np.isnan(ref))              # the same pixels are filled
    ok = ~np.isnan(ref)
    if method == al.NEAREST:
        assert np.array_equal(out[ok], ref[ok])
    elif ok.any():
        assert np.max(np.abs(out[ok] - ref[ok])) <= TOL_RS * np.max(np.abs(img))
    return ok.mean()


@pytest.mark.parametrize("method", [al.NEAREST, al.BILINEAR, al.LANCZOS3])
@pytest.mark.parametrize("nx,ny,M", [
    (128, 64, [1, 0, 0, 0, 1, 0]),                                   # identity
    (100, 72, [1, 0, 3, 0, 1, -2]),                                  # integer shift: exact integer decisions
    (100, 72, [1, 0, 0.5, 0, 1, 0.5]),                               # half-pixel: ties of floor(xs + 0.5)
    (61, 67, _rot(0.03, 1.002, 0.998, 1.37, -2.21, 61, 67)),         # small rotation + scale + shift, odd sizes
    (257, 33, _rot(-0.4, 0.9, 1.1, 0.0, 0.0, 257, 33)),              # ragged tails of the 32 x 8 tiles, large rotation
    (64, 64, [0, 1, 0, -1, 0, 63]),                                  # quarter turn
    (40, 40, [1, 0, 100, 0, 1, 0]),                                  # everything outside: all fill
])
def test_resample_parity(nx, ny, M, method):
    _, R = starfield.random_pair(nx, ny, seed=nx + ny)
    _check(R, M, method)


def test_resample_fill_value_and_zero_fill():
    _, R = starfield.random_pair(90, 50, seed=3)
    p = SfftPlan(90, 50, 3, 0, 0)
    M = [1, 0, 4.25, 0, 1, -3.5]
    out = p.resample_affine(dev(R), M, method=3, fill=-1.5).cpu().numpy()
    ref = al.resample_affine(R, M, 3, -1.5)
    assert np.array_equal(out == -1.5, ref == -1.5)
    assert np.max(np.abs(out - ref)) <= TOL_RS * np.max(np.abs(R))
    p.destroy()


@pytest.mark.parametrize("M", [[1, 0, 2.4, 0, 1, -1.6], _rot(0.1, 1.0, 1.0, 0.3, 0.2, 100, 72), [1, 0, 0.5, 0, 1, 0.5]])
def test_mask_parity_bit_exact(M):
    rng = np.random.default_rng(8)
    m = (rng.random((72, 100)) > 0.3).astype(np.uint8) * 3
    p = SfftPlan(100, 72, 3, 0, 0)
    out = p.resample_affine_mask(dev(m), M, fill=7).cpu().numpy()
    assert np.array_equal(out, al.resample_affine_mask(m, M, fill=7))
    p.destroy()


def test_align_then_subtract_on_one_plan():
    """Pipeline order: the template is aligned onto the science grid, then subtracted, on one plan."""
    import oracle
    nx, ny, L, DK, DB = 100, 72, 5, 1, 1
    S, R = starfield.random_pair(nx, ny, seed=31)
    M = _rot(0.01, 1.0, 1.0, 0.4, -0.3, nx, ny)
    sky = float(np.median(R))
    p = SfftPlan(nx, ny, L, DK, DB)
    Ra = p.resample_affine(dev(R), M, method=3, fill=sky)
    p.build_system(dev(S), Ra); p.solve()
    D, c = p.subtract(); p.sync_status()
    Ra0 = al.resample_affine(R, M, 3, sky)
    assert np.max(np.abs(Ra.cpu().numpy() - Ra0)) <= TOL_RS * np.max(np.abs(R))
    G0, h0 = oracle.build_system(S, Ra0, None, L, DK, DB)
    c0 = oracle.solve(G0, h0)
    D0 = oracle.subtract(S, Ra0, L, DK, DB, c0)
    assert np.max(np.abs(c.cpu().numpy() - c0)) <= 1e-8 * np.max(np.abs(c0))
    assert np.max(np.abs(D.cpu().numpy() - D0)) <= 1e-6 * 20.0
    p.destroy()


def test_resample_errors():
    p = SfftPlan(64, 64, 3, 0, 0)
    img = torch.zeros((64, 64), dtype=torch.float64, device="cuda")
    with pytest.raises(SfftError):
        p.resample_affine(img, [1, 0, 0, 0, 1, 0], out=img)                  # aliased
    with pytest.raises(SfftError):
        p.resample_affine(img, [1, 0, float("nan"), 0, 1, 0])                # non-finite matrix
    with pytest.raises(SfftError):
        p.resample_affine(img, [1, 0, 0, 0, 1, 0], method=2)                 # unknown interpolant
    m = torch.zeros((64, 64), dtype=torch.uint8, device="cuda")
    with pytest.raises(SfftError):
        p.resample_affine_mask(m, [1, 0, 0, 0, 1, 0], fill=300)
    p.destroy()


def test_psf_stamp_is_resampled_on_a_plan_of_its_own_size():
    """Reading A4: the reference PSF (a 25 x 25 stamp) is aligned like an image, on a plan of the stamp's size."""
    P = 25
    yy, xx = np.mgrid[0:P, 0:P] - (P - 1) / 2.0
    psf = np.exp(-0.5 * ((xx / 1.6) ** 2 + (yy / 2.1) ** 2)); psf /= psf.sum()
    M = _rot(0.3, 1.0, 1.0, 0.25, -0.4, P, P)
    p = SfftPlan(P, P, 1, 0, 0)
    for method in (al.BILINEAR, al.LANCZOS3):
        out = p.resample_affine(dev(psf), M, method=method, fill=0.0).cpu().numpy()
        ref = al.resample_affine(psf, M, method, 0.0)
        assert np.array_equal(out == 0.0, ref == 0.0)
        assert np.max(np.abs(out - ref)) <= TOL_RS * psf.max()
    p.destroy()
