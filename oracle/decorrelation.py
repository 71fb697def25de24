"""Oracle for f1, the decorrelation kernel (pipeline step 7: "Fit and apply the
decorrelation kernel to the difference image.  Also apply the decorrelation kernel to the science PSF
and cross-convolved science image") -- TEST INFRASTRUCTURE, plain numpy FP64.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module; it shares no
code with the CUDA path.

PAPER.md gives no formula for the kernel; the readings below (D1-D5) fix one, and
the pins in tests/test_oracle_pins_decorrelation.py tie this file to what those readings mean:

D1  The difference image of the pipeline is D = S (*) P_R - (R (*) P_S) (*) K - B (steps 5 and 6,
    PAPER.md:86-87).  With independent white pixel noise of variance var_S in S and var_R in R, the noise of
    D has the power spectrum
        F(k) = var_S |P_R^(k)|^2 + var_R |P_S^(k)|^2 |K^(k)|^2.
D2  K is the LOCAL matching kernel K(u, v; x, y) = sum_t a_{t,u,v} xt(x)^i yt(y)^j at one chosen pixel (one
    kernel per frame or per stamp).
D3  The decorrelation kernel W is the real, even kernel with W^(k) = sqrt(F(0) / F(k)) on an N x N
    periodic grid: it whitens the noise of D and keeps its flux scale (W^(0) = 1, i.e. sum W = 1).
D4  What is applied to the images is the central Ld x Ld crop of W (taps |u|, |v| <= (Ld-1)/2), NOT
    renormalised, by the same circular convolution as f2 (oracle.sfft_oracle.convolve_stamp).
D5  Tap layout of every stamp: stamp[(v + w) * P + (u + w)], like the kernel coefficients.
"""
from __future__ import annotations

import numpy as np


def poly_exponents(deg: int):
    """(i, j) of the basis x^i y^j in coefficient order: total degree ascending, then j ascending
    (SURVEY.md section 8(b) "Coefficient layout")."""
    return [(d - j, j) for d in range(deg + 1) for j in range(d + 1)]


def coord(x: float, n: int) -> float:
    """Centred pixel coordinate, reading C3: xt = (2 x + 1 - n) / n."""
    return (2.0 * x + 1.0 - n) / n


def local_kernel(c, L: int, DK: int, x: float, y: float, nx: int, ny: int):
    """D2: K[(v + w), (u + w)] = sum_t a_{t,u,v} xt(x)^i yt(y)^j, a_{t,u,v} = c[t L^2 + (v+w) L + (u+w)]."""
    c = np.asarray(c, dtype=np.float64)
    K = np.zeros((L, L))
    xt, yt = coord(x, nx), coord(y, ny)
    for t, (i, j) in enumerate(poly_exponents(DK)):
        K += c[t * L * L:(t + 1) * L * L].reshape(L, L) * (xt ** i) * (yt ** j)
    return K


def embed(stamp, N: int):
    """P x P stamp (taps -w..w) on the N x N periodic grid with tap (u, v) at [v mod N, u mod N]."""
    stamp = np.asarray(stamp, dtype=np.float64)
    P = stamp.shape[0]
    if stamp.ndim != 2 or stamp.shape[1] != P or P % 2 != 1 or P > N:
        raise ValueError("stamp must be P x P, P odd, P <= N")
    w = (P - 1) // 2
    g = np.zeros((N, N))
    for v in range(-w, w + 1):
        for u in range(-w, w + 1):
            g[v % N, u % N] = stamp[v + w, u + w]
    return g


def noise_power(K, psf_S, psf_R, var_S: float, var_R: float, N: int):
    """D1: F[ky, kx] on the N x N grid (np.fft.fft2 as the library DFT step)."""
    Kh = np.fft.fft2(embed(K, N))
    PSh = np.fft.fft2(embed(psf_S, N))
    PRh = np.fft.fft2(embed(psf_R, N))
    return var_S * np.abs(PRh) ** 2 + var_R * np.abs(PSh) ** 2 * np.abs(Kh) ** 2


def decorrelation_kernel(K, psf_S, psf_R, var_S: float, var_R: float, N: int):
    """D3: the full N x N kernel W, tap (u, v) at [v mod N, u mod N]."""
    F = noise_power(K, psf_S, psf_R, var_S, var_R, N)
    if not np.all(F > 0.0):
        raise ValueError("noise power spectrum has a zero: the decorrelation kernel is undefined")
    What = np.sqrt(F[0, 0] / F)
    return np.fft.ifft2(What).real


def decorrelation_stamp(K, psf_S, psf_R, var_S: float, var_R: float, N: int, Ld: int):
    """D4: the central Ld x Ld crop of W in the stamp tap layout (D5)."""
    if Ld % 2 != 1 or Ld > N:
        raise ValueError("Ld must be odd and <= N")
    W = decorrelation_kernel(K, psf_S, psf_R, var_S, var_R, N)
    wd = (Ld - 1) // 2
    out = np.empty((Ld, Ld))
    for v in range(-wd, wd + 1):
        for u in range(-wd, wd + 1):
            out[v + wd, u + wd] = W[v % N, u % N]
    return out
