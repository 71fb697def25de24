"""Pins of oracle/decorrelation.py (f1; readings D1-D5 of DESIGN.md section 13) -- CPU only.

The paper prints no formula or value for the decorrelation kernel, so the pins are what the readings mean:
the kernel must WHITEN the noise covariance of D built tap by tap in real space (no FFT), keep the flux scale,
reduce to a delta when nothing correlates the noise, and agree with a brute-force DFT written as loops.
"""
import numpy as np
import pytest

import oracle
from oracle import decorrelation as deco


def _stamp(P, seed, sigma=1.2):
    rng = np.random.default_rng(seed)
    w = (P - 1) // 2
    yy, xx = np.mgrid[-w:w + 1, -w:w + 1]
    st = np.exp(-0.5 * (((xx - 0.2) / sigma) ** 2 + ((yy + 0.1) / (1.3 * sigma)) ** 2)) + 0.01 * rng.random((P, P))
    return st / st.sum()


def _circ_conv(a, b):
    """Circular convolution of two N x N grids by shifted copies (np.roll), no FFT."""
    out = np.zeros_like(a)
    N = a.shape[0]
    for v in range(N):
        for u in range(N):
            if b[v, u] != 0.0:
                out += b[v, u] * np.roll(a, (v, u), axis=(0, 1))
    return out


def _flip(a):
    """a(-u, -v) on the periodic grid."""
    return np.roll(a[::-1, ::-1], (1, 1), axis=(0, 1))


def test_delta_inputs_give_delta_kernel():
    d = np.zeros((3, 3)); d[1, 1] = 1.0
    W = deco.decorrelation_kernel(2.0 * d, 0.5 * d, 3.0 * d, 4.0, 9.0, 16)
    ref = np.zeros((16, 16)); ref[0, 0] = 1.0
    assert np.max(np.abs(W - ref)) < 1e-15
    st = deco.decorrelation_stamp(2.0 * d, 0.5 * d, 3.0 * d, 4.0, 9.0, 16, 5)
    ref5 = np.zeros((5, 5)); ref5[2, 2] = 1.0
    assert np.max(np.abs(st - ref5)) < 1e-15


def test_kernel_whitens_the_real_space_noise_covariance():
    """D1 + D3: Cov(D) = var_S P_R * P_R~ + var_R (P_S*K) * (P_S*K)~ built by shifted copies; W * Cov * W~ must be
    F(0) x delta, with F(0) = var_S (sum P_R)^2 + var_R (sum P_S sum K)^2.  A dropped square, a swapped PSF, a
    missing K or a wrong normalisation all fail this."""
    N = 24
    K, PS, PR = _stamp(5, 1, 0.7) * 1.3, _stamp(7, 2, 0.8), _stamp(7, 3, 0.75)
    vS, vR = 25.0, 3.0
    gK, gS, gR = deco.embed(K, N), deco.embed(PS, N), deco.embed(PR, N)
    q = _circ_conv(gS, gK)
    cov = vS * _circ_conv(gR, _flip(gR)) + vR * _circ_conv(q, _flip(q))
    W = deco.decorrelation_kernel(K, PS, PR, vS, vR, N)
    white = _circ_conv(_circ_conv(cov, W), _flip(W))
    F0 = vS * PR.sum() ** 2 + vR * (PS.sum() * K.sum()) ** 2
    ref = np.zeros((N, N)); ref[0, 0] = F0
    # W^ reaches sqrt(F(0) / min F) ~ 30 here, so rounding is amplified by ~1e3 over the plain 1e-16
    assert np.max(np.abs(white - ref)) < 1e-11 * F0


def test_flux_scale_and_symmetry():
    N = 32
    K, PS, PR = _stamp(5, 4), _stamp(5, 5), _stamp(5, 6)
    W = deco.decorrelation_kernel(K, PS, PR, 2.0, 7.0, N)
    F = deco.noise_power(K, PS, PR, 2.0, 7.0, N)
    eps = 1e-15 * np.sqrt(F[0, 0] / F.min()) * N           # rounding scale: max W^ x a sum of N^2 terms
    assert abs(W.sum() - 1.0) < eps                        # W^(0) = 1
    assert np.max(np.abs(W - _flip(W))) < eps              # even kernel
    W2 = deco.decorrelation_kernel(K, PS, PR, 20.0, 70.0, N)
    assert np.max(np.abs(W - W2)) < eps                    # only the variance ratio matters
    W3 = deco.decorrelation_kernel(K[::-1, ::-1], PS, PR, 2.0, 7.0, N)
    assert np.max(np.abs(W - W3)) < eps                    # |K^|^2 is even


def test_against_bruteforce_dft_loops():
    """The library FFT step against the DFT definition written as plain loops over taps (N = 8)."""
    N = 8
    K, PS, PR = _stamp(3, 7, 0.8), _stamp(3, 8, 0.7), _stamp(5, 9, 0.9)
    vS, vR = 1.5, 0.5

    def dft(st, kx, ky):
        w = (st.shape[0] - 1) // 2
        z = 0.0 + 0.0j
        for v in range(-w, w + 1):
            for u in range(-w, w + 1):
                z += st[v + w, u + w] * np.exp(-2j * np.pi * (kx * u + ky * v) / N)
        return z

    F = np.empty((N, N))
    for ky in range(N):
        for kx in range(N):
            F[ky, kx] = vS * abs(dft(PR, kx, ky)) ** 2 + vR * abs(dft(PS, kx, ky)) ** 2 * abs(dft(K, kx, ky)) ** 2
    assert np.max(np.abs(F - deco.noise_power(K, PS, PR, vS, vR, N))) < 1e-14 * F.max()
    Ld, wd = 5, 2
    ref = np.empty((Ld, Ld))
    for v in range(-wd, wd + 1):
        for u in range(-wd, wd + 1):
            z = 0.0
            for ky in range(N):
                for kx in range(N):
                    z += np.sqrt(F[0, 0] / F[ky, kx]) * np.cos(2 * np.pi * (kx * u + ky * v) / N)
            ref[v + wd, u + wd] = z / (N * N)
    eps = 1e-15 * np.sqrt(F[0, 0] / F.min()) * N           # rounding scale: max W^ x a sum of N^2 terms
    assert np.max(np.abs(ref - deco.decorrelation_stamp(K, PS, PR, vS, vR, N, Ld))) < eps


def test_stamp_is_the_crop_of_the_kernel():
    N, Ld = 20, 7
    K, PS, PR = _stamp(5, 10), _stamp(5, 11), _stamp(3, 12)
    W = deco.decorrelation_kernel(K, PS, PR, 1.0, 1.0, N)
    st = deco.decorrelation_stamp(K, PS, PR, 1.0, 1.0, N, Ld)
    assert st[3, 3] == W[0, 0] and st[3, 4] == W[0, 1] and st[2, 3] == W[N - 1, 0] and st[6, 0] == W[3, N - 3]


def test_zero_of_the_power_spectrum_is_refused():
    d = np.zeros((3, 3)); d[1, 1] = 1.0
    box = np.zeros((3, 3)); box[1, 0] = box[1, 1] = 0.5    # P^ vanishes at kx = N/2
    with pytest.raises(ValueError):
        deco.decorrelation_kernel(d, box, box, 1.0, 1.0, 8)


@pytest.mark.parametrize("DK", [0, 1, 2])
def test_local_kernel_is_the_response_to_a_point_source(DK):
    """D2 against the pinned subtraction oracle (reading C2: the polynomial weight is taken at the SOURCE pixel): for
    R = delta at (x0, y0), S = 0 and zero background coefficients, -D(x0 + u, y0 + v) = K(u, v; x0, y0)."""
    nx, ny, L, DB = 20, 16, 5, 0
    rng = np.random.default_rng(DK)
    n = oracle.num_unknowns(L, DK, DB)
    c = rng.standard_normal(n); c[-1] = 0.0
    x0, y0 = 13, 4
    R = np.zeros((ny, nx)); R[y0, x0] = 1.0
    D = oracle.subtract(np.zeros((ny, nx)), R, L, DK, DB, c)
    K = deco.local_kernel(c, L, DK, x0, y0, nx, ny)
    w = 2
    for v in range(-w, w + 1):
        for u in range(-w, w + 1):
            assert abs(-D[(y0 + v) % ny, (x0 + u) % nx] - K[v + w, u + w]) < 1e-14
