"""Oracle for f3, alignment / resampling onto the science grid (pipeline step 4: "Align the
reference image, reference PSF, and reference detection mask to the science image") -- TEST
INFRASTRUCTURE, plain numpy FP64.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module; it shares no
code with the CUDA path.

PAPER.md gives neither the geometric model nor the interpolant; the readings:

A1  Geometry: an affine map from OUTPUT (science-grid) pixel (x, y) to SOURCE pixel coordinates,
        xs = (M[0] x + M[1] y) + M[2],   ys = (M[3] x + M[4] y) + M[5]
    (pixel centres at integers; evaluated in FP64 in exactly this order, no fused multiply-add).
A2  Interpolants, all separable, footprint half-width a, i0 = floor(xs), taps i = i0-a+1 .. i0+a:
      method 0  nearest:  out = img[floor(ys + 0.5), floor(xs + 0.5)]
      method 1  bilinear: a = 1, k(t) = 1 - |t|
      method 3  Lanczos-3: a = 3, k(t) = sinc(t) sinc(t/3) for |t| < 3 (sinc(t) = sin(pi t)/(pi t)),
                weights divided by their sum along each axis (constants are reproduced exactly).
A3  Boundary: an output pixel whose footprint (all 2a x 2a taps; the one pixel for nearest) is not entirely
    inside the source frame gets the value `fill`.
A4  Masks (uint8) are resampled with method 0 only.
"""
from __future__ import annotations

import numpy as np

NEAREST, BILINEAR, LANCZOS3 = 0, 1, 3


def source_coords(M, nx: int, ny: int):
    """A1 on the whole output grid: (xs, ys), each (ny, nx)."""
    M = [float(m) for m in M]
    x = np.arange(nx, dtype=np.float64)[None, :]
    y = np.arange(ny, dtype=np.float64)[:, None]
    xs = (M[0] * x + M[1] * y) + M[2]
    ys = (M[3] * x + M[4] * y) + M[5]
    return xs, ys


def tap_weight(t, method: int):
    """A2: k(t) of the interpolant."""
    t = np.asarray(t, dtype=np.float64)
    if method == BILINEAR:
        return np.where(np.abs(t) < 1.0, 1.0 - np.abs(t), 0.0)
    if method == LANCZOS3:
        return np.where(np.abs(t) < 3.0, np.sinc(t) * np.sinc(t / 3.0), 0.0)
    raise ValueError("method must be 1 (bilinear) or 3 (Lanczos-3)")


def resample_affine(img, M, method: int, fill: float = 0.0):
    """out(x, y) = sum_{i,j} wx_i wy_j img[j, i] / (sum wx sum wy) over the footprint of (xs, ys); A1-A3."""
    img = np.ascontiguousarray(img, dtype=np.float64)
    ny, nx = img.shape
    xs, ys = source_coords(M, nx, ny)
    if method == NEAREST:
        ix = np.floor(xs + 0.5).astype(np.int64)
        iy = np.floor(ys + 0.5).astype(np.int64)
        inside = (ix >= 0) & (ix < nx) & (iy >= 0) & (iy < ny)
        out = np.full((ny, nx), float(fill))
        out[inside] = img[iy[inside], ix[inside]]
        return out
    a = 1 if method == BILINEAR else 3
    i0 = np.floor(xs).astype(np.int64)
    j0 = np.floor(ys).astype(np.int64)
    inside = (i0 - a + 1 >= 0) & (i0 + a <= nx - 1) & (j0 - a + 1 >= 0) & (j0 + a <= ny - 1)
    acc = np.zeros((ny, nx))
    sx = np.zeros((ny, nx))
    sy = np.zeros((ny, nx))
    for dj in range(-a + 1, a + 1):
        sy += tap_weight(ys - (j0 + dj), method)
    for di in range(-a + 1, a + 1):
        sx += tap_weight(xs - (i0 + di), method)
    for dj in range(-a + 1, a + 1):
        wy = tap_weight(ys - (j0 + dj), method)
        jj = np.clip(j0 + dj, 0, ny - 1)
        row = np.zeros((ny, nx))
        for di in range(-a + 1, a + 1):
            wx = tap_weight(xs - (i0 + di), method)
            ii = np.clip(i0 + di, 0, nx - 1)
            row += wx * img[jj, ii]
        acc += wy * row
    out = acc / (sx * sy)
    return np.where(inside, out, float(fill))


def resample_affine_mask(mask, M, fill: int = 0):
    """A4: nearest-neighbour resampling of a uint8 mask."""
    mask = np.ascontiguousarray(mask, dtype=np.uint8)
    ny, nx = mask.shape
    xs, ys = source_coords(M, nx, ny)
    ix = np.floor(xs + 0.5).astype(np.int64)
    iy = np.floor(ys + 0.5).astype(np.int64)
    inside = (ix >= 0) & (ix < nx) & (iy >= 0) & (iy < ny)
    out = np.full((ny, nx), np.uint8(fill), dtype=np.uint8)
    out[inside] = mask[iy[inside], ix[inside]]
    return out
