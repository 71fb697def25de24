"""Pins of oracle/alignment.py (f3; readings A1-A4 of DESIGN.md section 14) -- CPU only.

The paper prints no value for this step; the pins are exact special cases (identity, integer shifts, a quarter
turn), scipy.ndimage's own interpolation for the bilinear case, closed-form Lanczos-3 weights at half-pixel
offsets, exact reproduction of constants, and the accuracy of Lanczos-3 on a band-limited image.
"""
import numpy as np
import pytest
from scipy import ndimage

from oracle import alignment as al

IDENT = [1, 0, 0, 0, 1, 0]


def _img(nx, ny, seed):
    return np.random.default_rng(seed).standard_normal((ny, nx)) * 10.0 + 50.0


@pytest.mark.parametrize("method,a", [(al.NEAREST, 0), (al.BILINEAR, 1), (al.LANCZOS3, 3)])
def test_identity_returns_the_image_inside_the_footprint_rule(method, a):
    img = _img(23, 17, 1)
    out = al.resample_affine(img, IDENT, method, fill=-7.0)
    lo = max(a - 1, 0)
    hi_x, hi_y = 23 - a, 17 - a
    if method == al.NEAREST:
        assert np.array_equal(out, img)
        return
    assert np.max(np.abs(out[lo:hi_y, lo:hi_x] - img[lo:hi_y, lo:hi_x])) < 1e-13
    border = np.ones_like(img, dtype=bool); border[lo:hi_y, lo:hi_x] = False
    assert np.all(out[border] == -7.0)                       # A3: incomplete footprint -> fill


@pytest.mark.parametrize("method", [al.NEAREST, al.BILINEAR, al.LANCZOS3])
def test_integer_shift_moves_pixels(method):
    """xs = x + 3, ys = y - 2: out[y, x] = img[y - 2, x + 3] wherever the footprint fits (index arithmetic here)."""
    img = _img(31, 29, 2)
    out = al.resample_affine(img, [1, 0, 3, 0, 1, -2], method, fill=np.nan)
    for (x, y) in [(5, 7), (10, 20), (20, 9), (24, 25)]:
        assert abs(out[y, x] - img[y - 2, x + 3]) < 1e-13
    assert np.isnan(out[0, 5]) and np.isnan(out[5, 30])      # source row -2 / source column 33 are outside


def test_quarter_turn_is_a_pixel_permutation():
    """xs = y, ys = (n-1) - x on a square frame is an exact quarter turn: out[y, x] = img[n-1-x, y].  A transposed or
    mis-ordered matrix fails this."""
    n = 16
    img = _img(n, n, 3)
    out = al.resample_affine(img, [0, 1, 0, -1, 0, n - 1], al.NEAREST)
    ref = np.empty_like(img)
    for y in range(n):
        for x in range(n):
            ref[y, x] = img[n - 1 - x, y]
    assert np.array_equal(out, ref)
    assert np.array_equal(ref, np.rot90(img, -1))


def test_bilinear_against_scipy_map_coordinates():
    nx, ny = 40, 33
    img = _img(nx, ny, 4)
    th = 0.05
    M = [1.01 * np.cos(th), -np.sin(th), 1.7, np.sin(th), 0.99 * np.cos(th), -0.6]
    out = al.resample_affine(img, M, al.BILINEAR, fill=np.nan)
    xs, ys = al.source_coords(M, nx, ny)
    ref = ndimage.map_coordinates(img, [ys, xs], order=1, mode="constant", cval=np.nan)
    ok = ~np.isnan(out)
    assert ok.sum() > 0.7 * nx * ny
    assert np.max(np.abs(out[ok] - ref[ok])) < 1e-12
    # and the affine geometry itself against scipy's own affine_transform ((row, col) convention)
    ref2 = ndimage.affine_transform(img, np.array([[M[4], M[3]], [M[1], M[0]]]), offset=[M[5], M[2]], order=1,
                                    mode="constant", cval=np.nan)
    assert np.max(np.abs(out[ok] - ref2[ok])) < 1e-12


def test_lanczos3_half_pixel_closed_form_weights():
    """At a half-pixel shift in x the six weights are 6/(25 pi^2), -4/(3 pi^2), 6/pi^2 and mirror, normalised by their
    sum 736/(75 pi^2)."""
    nx, ny = 20, 9
    img = _img(nx, ny, 5)
    out = al.resample_affine(img, [1, 0, 0.5, 0, 1, 0], al.LANCZOS3, fill=np.nan)
    p2 = np.pi ** 2
    wts = np.array([6 / (25 * p2), -4 / (3 * p2), 6 / p2, 6 / p2, -4 / (3 * p2), 6 / (25 * p2)])
    assert abs(wts.sum() - 736 / (75 * p2)) < 1e-15
    wts /= wts.sum()
    for (x, y) in [(2, 2), (9, 4), (16, 5)]:
        ref = float(np.dot(wts, img[y, x - 2:x + 4]))        # xs = x + 0.5: taps x-2 .. x+3
        assert abs(out[y, x] - ref) < 1e-12
    assert np.isnan(out[2, 1]) and np.isnan(out[2, 17])      # tap x-2 = -1 / tap x+3 = 20 outside


@pytest.mark.parametrize("method", [al.BILINEAR, al.LANCZOS3])
def test_constants_are_reproduced(method):
    img = np.full((25, 30), 3.25)
    out = al.resample_affine(img, [0.97, 0.02, 1.3, -0.03, 1.02, 0.4], method, fill=np.nan)
    ok = ~np.isnan(out)
    assert ok.sum() > 300 and np.max(np.abs(out[ok] - 3.25)) < 1e-14


def test_lanczos3_on_a_band_limited_image():
    """A slow sinusoid shifted by a fraction of a pixel: Lanczos-3 must reproduce the analytically shifted image to its
    known accuracy (a sign error of the shift or an off-by-one tap gives errors of order 0.1)."""
    nx, ny = 64, 48
    y, x = np.mgrid[0:ny, 0:nx].astype(np.float64)
    f = lambda xx, yy: np.sin(2 * np.pi * xx / 16.0) * np.cos(2 * np.pi * yy / 12.0)
    dx, dy = 0.3, -0.4
    out = al.resample_affine(f(x, y), [1, 0, dx, 0, 1, dy], al.LANCZOS3, fill=np.nan)
    ok = ~np.isnan(out)
    assert np.max(np.abs(out[ok] - f(x + dx, y + dy)[ok])) < 1e-2
    wrong = f(x - dx, y - dy)
    assert np.max(np.abs(out[ok] - wrong[ok])) > 0.1


def test_mask_nearest():
    rng = np.random.default_rng(6)
    m = (rng.random((21, 26)) > 0.5).astype(np.uint8)
    out = al.resample_affine_mask(m, [1, 0, 2.4, 0, 1, -1.6], fill=9)
    for (x, y) in [(3, 5), (10, 10), (20, 19)]:
        assert out[y, x] == m[y - 2, x + 2]                  # round(x + 2.4) = x + 2, round(y - 1.6) = y - 2
    assert out[0, 0] == 9 and out[5, 25] == 9
    as_float = al.resample_affine(m.astype(np.float64), [1, 0, 2.4, 0, 1, -1.6], al.NEAREST, fill=9.0)
    assert np.array_equal(out, as_float.astype(np.uint8))
