"""Pins of the CPU oracle (pins P1-P11) -- CPU only.

Each test fixes a part of oracle/sfft_oracle.c against something other than itself:
values the task statement prints (golden/), closed forms, exact special cases,
numpy library routines (FFT cross-correlation, lstsq, eigvalsh) and brute force on
tiny inputs built with a different mechanism (np.roll).
"""
import numpy as np
import pytest

import oracle
from paper_2509_18544_b200 import starfield


def _rng_pair(nx, ny, seed, sky=30.0):
    rng = np.random.default_rng(seed)
    R = sky + 10.0 * rng.standard_normal((ny, nx))
    S = sky + 10.0 * rng.standard_normal((ny, nx))
    return S, R


def _idx(L, t, u, v):
    w = (L - 1) // 2
    return t * L * L + (v + w) * L + (u + w)


def _xt(n):
    return (2.0 * np.arange(n) + 1.0 - n) / n


def _poly_list(deg):
    return [(d - j, j) for d in range(deg + 1) for j in range(d + 1)]


# ---------------------------------------------------------------- golden / layout
def test_unknown_counts_golden(golden_dir):
    rows = [l.split() for l in (golden_dir / "unknown_counts.txt").read_text().splitlines()
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 4
    for L, DK, DB, n in rows:
        assert oracle.num_unknowns(int(L), int(DK), int(DB)) == int(n)


def test_poly_order_golden(golden_dir):
    rows = [l.split() for l in (golden_dir / "poly_order.txt").read_text().splitlines()
            if l.strip() and not l.startswith("#")]
    for t, i, j in rows:
        assert oracle.poly_index(int(t)) == (int(i), int(j))
    assert [oracle.poly_index(t) for t in range(10)] == _poly_list(3)


def test_coord_is_centred():
    # C3: xt = (2x+1-nx)/nx, antisymmetric about the frame centre, inside (-1,1)
    for n in (7, 32, 4088):
        xs = np.array([oracle.coord(x, n) for x in range(n)])
        np.testing.assert_allclose(xs, -xs[::-1], atol=0)
        assert abs(xs[0] + (n - 1) / n) < 1e-16 and xs.max() < 1.0
        np.testing.assert_allclose(np.diff(xs), 2.0 / n, rtol=1e-11)


def test_weighted_and_poly_images():
    S, R = _rng_pair(19, 13, 0)
    mask = (np.random.default_rng(1).random(R.shape) > 0.3).astype(np.uint8)
    X, Y = np.meshgrid(_xt(19), _xt(13))
    np.testing.assert_allclose(oracle.weighted_image(R, None, 2, 1), X**2 * Y * R, rtol=1e-14)
    np.testing.assert_allclose(oracle.weighted_image(R, mask, 1, 3), X * Y**3 * R * mask, rtol=1e-14)
    np.testing.assert_allclose(oracle.poly_image(19, 13, 1, 2), X * Y**2, rtol=1e-14)


# ---------------------------------------------------------------- lag sums
@pytest.mark.parametrize("nx,ny", [(40, 56), (64, 64), (37, 23)])
def test_lag_sum_matches_fft_cross_correlation(nx, ny):
    """X(a,b)[du,dv] = irfft2(conj(rfft2 a) rfft2 b)[dv mod ny, du mod nx] (library FFT)."""
    rng = np.random.default_rng(5)
    a = rng.standard_normal((ny, nx))
    b = rng.standard_normal((ny, nx))
    X = np.fft.irfft2(np.conj(np.fft.rfft2(a)) * np.fft.rfft2(b), s=(ny, nx))
    for du, dv in [(0, 0), (1, 0), (0, 1), (-3, 2), (5, -4), (-6, -6), (nx + 1, -ny - 2)]:
        got = oracle.lag_sum(a, b, du, dv)
        assert abs(got - X[dv % ny, du % nx]) < 1e-11 * nx * ny


def test_lag_sum_brute_force_and_sign():
    """Tiny brute force with python loops: b is read at (x+du, y+dv)."""
    rng = np.random.default_rng(6)
    nx, ny = 7, 5
    a = rng.standard_normal((ny, nx))
    b = rng.standard_normal((ny, nx))
    for du, dv in [(2, 0), (0, -1), (-3, 4)]:
        ref = sum(a[y, x] * b[(y + dv) % ny, (x + du) % nx] for y in range(ny) for x in range(nx))
        assert abs(oracle.lag_sum(a, b, du, dv) - ref) < 1e-13


def test_lag_symmetry_P11():
    rng = np.random.default_rng(7)
    a = rng.standard_normal((24, 32))
    b = rng.standard_normal((24, 32))
    for du, dv in [(1, 2), (-4, 3), (6, -6)]:
        assert abs(oracle.lag_sum(a, b, du, dv) - oracle.lag_sum(b, a, -du, -dv)) < 1e-12
        assert abs(oracle.lag_sum(a, a, du, dv) - oracle.lag_sum(a, a, -du, -dv)) < 1e-12


# ---------------------------------------------------------------- P4 brute force
def _dense_design(R, mask, L, DK, DB):
    """Design matrix built with np.roll: column (t,u,v) = T_t rolled by (+v rows, +u cols)."""
    ny, nx = R.shape
    w = (L - 1) // 2
    X, Y = np.meshgrid(_xt(nx), _xt(ny))
    Rf = R if mask is None else R * mask
    cols = []
    for (i, j) in _poly_list(DK):
        T = X**i * Y**j * Rf
        for v in range(-w, w + 1):
            for u in range(-w, w + 1):
                cols.append(np.roll(T, (v, u), axis=(0, 1)).ravel())
    for (p, q) in _poly_list(DB):
        cols.append((X**p * Y**q).ravel())
    return np.stack(cols, axis=1)


@pytest.mark.parametrize("nx,ny,L,DK,DB,masked", [
    (32, 32, 5, 1, 1, False), (32, 24, 5, 1, 1, False), (32, 24, 3, 2, 2, True), (24, 32, 7, 0, 0, False)])
def test_P4_brute_force_dense_least_squares(nx, ny, L, DK, DB, masked):
    S, R = _rng_pair(nx, ny, 11)
    mask = (np.random.default_rng(12).random(R.shape) > 0.1).astype(np.uint8) if masked else None
    A = _dense_design(R, mask, L, DK, DB)
    b = (S if mask is None else S * mask).ravel()
    # the oracle's own explicit A agrees with the np.roll construction
    np.testing.assert_allclose(oracle.design_matrix(R, mask, L, DK, DB), A, rtol=0, atol=1e-12)
    G, h = oracle.build_system(S, R, mask, L, DK, DB)
    Gd, hd = oracle.build_system_dense(S, R, mask, L, DK, DB)
    Gn, hn = A.T @ A, A.T @ b
    scale = np.sqrt(np.outer(np.diag(Gn), np.diag(Gn)))
    assert np.max(np.abs(G - Gn) / scale) < 1e-13       # lag shortcut == dense A^T A
    assert np.max(np.abs(Gd - Gn) / scale) < 1e-13
    assert np.max(np.abs(h - hn) / (np.sqrt(np.diag(Gn)) * np.linalg.norm(b))) < 1e-13
    assert np.max(np.abs(hd - hn) / (np.sqrt(np.diag(Gn)) * np.linalg.norm(b))) < 1e-13
    c = oracle.solve(G, h)
    c_ls = np.linalg.lstsq(A, b, rcond=None)[0]
    assert np.max(np.abs(c - c_ls)) < 1e-9 * np.max(np.abs(c_ls))
    # D from the real-space convolution equals b - A c when nothing is masked
    if mask is None:
        D = oracle.subtract(S, R, L, DK, DB, c)
        np.testing.assert_allclose(D.ravel(), b - A @ c, atol=1e-10 * np.abs(S).max())


# ---------------------------------------------------------------- P1 SPD
def test_P1_symmetric_positive_definite():
    p = starfield.make_pair(0, nx=64, ny=48, n_stars=40)
    Gd, _ = oracle.build_system_dense(p["S"], p["R"], None, 5, 1, 1)  # every entry summed on its own
    assert np.max(np.abs(Gd - Gd.T)) <= 1e-13 * np.abs(Gd).max()
    G, h = oracle.build_system(p["S"], p["R"], None, 5, 1, 1)
    d = 1.0 / np.sqrt(np.diag(G))
    ev = np.linalg.eigvalsh(G * np.outer(d, d))
    assert ev.min() > 0
    c, Lf = oracle.solve(G, h, return_factor=True)
    np.testing.assert_allclose(Lf @ Lf.T, G * np.outer(d, d), atol=1e-13)
    np.testing.assert_allclose(G @ c, h, rtol=0, atol=1e-9 * np.abs(h).max())


def test_solve_matches_library():
    rng = np.random.default_rng(3)
    B = rng.standard_normal((60, 40))
    G = B.T @ B + 0.1 * np.eye(40)
    h = rng.standard_normal(40)
    np.testing.assert_allclose(oracle.solve(G, h), np.linalg.solve(G, h), rtol=1e-10)


# ---------------------------------------------------------------- exact special cases
def test_P2_identity_when_S_equals_R():
    _, R = _rng_pair(32, 24, 21)
    L, DK, DB = 5, 1, 1
    G, h = oracle.build_system(R, R, None, L, DK, DB)
    c = oracle.solve(G, h)
    expect = np.zeros_like(c)
    expect[_idx(L, 0, 0, 0)] = 1.0
    assert np.max(np.abs(c - expect)) < 1e-9
    D = oracle.subtract(R, R, L, DK, DB, c)
    assert np.max(np.abs(D)) < 1e-8 * np.abs(R).max()


@pytest.mark.parametrize("u0,v0", [(2, 0), (0, -1), (-2, 1)])
def test_P5_pure_shift_pins_sign_convention(u0, v0):
    """S(x,y) = R(x-u0, y-v0)  =>  delta at (u0,v0) in the constant kernel term."""
    _, R = _rng_pair(40, 32, 22)
    S = np.roll(R, (v0, u0), axis=(0, 1))
    L, DK, DB = 5, 1, 0
    G, h = oracle.build_system(S, R, None, L, DK, DB)
    c = oracle.solve(G, h)
    expect = np.zeros_like(c)
    expect[_idx(L, 0, u0, v0)] = 1.0
    assert np.max(np.abs(c - expect)) < 1e-9
    assert np.max(np.abs(oracle.subtract(S, R, L, DK, DB, c))) < 1e-8 * np.abs(R).max()


def test_P6_affine():
    _, R = _rng_pair(32, 32, 23)
    S = 1.7 * R + 12.5
    L, DK, DB = 3, 1, 1
    c = oracle.solve(*oracle.build_system(S, R, None, L, DK, DB))
    expect = np.zeros_like(c)
    expect[_idx(L, 0, 0, 0)] = 1.7
    expect[L * L * 3] = 12.5
    assert np.max(np.abs(c - expect)) < 1e-8


def test_P3_planted_kernel_and_background_recovered():
    """Noiseless S = sum a_true shift(T) + B_true with a noisy R: recover to 1e-9."""
    rng = np.random.default_rng(24)
    nx, ny, L, DK, DB = 96, 80, 5, 1, 1
    p = starfield.make_pair(0, nx=nx, ny=ny, n_stars=60, seed=9)
    R = p["R"]  # contains white noise (required for conditioning)
    n = oracle.num_unknowns(L, DK, DB)
    c_true = np.zeros(n)
    w = (L - 1) // 2
    g = np.exp(-0.5 * (np.arange(-w, w + 1) / 1.0) ** 2)
    k0 = np.outer(g, g) / np.outer(g, g).sum()
    c_true[: L * L] = k0.ravel()
    c_true[L * L: 3 * L * L] = 0.05 * rng.standard_normal(2 * L * L)
    c_true[3 * L * L:] = [3.0, -1.5, 0.7]
    A = _dense_design(R, None, L, DK, DB)
    S = (A @ c_true).reshape(ny, nx)
    c = oracle.solve(*oracle.build_system(S, R, None, L, DK, DB))
    kb = slice(0, 3 * L * L)
    assert np.max(np.abs(c[kb] - c_true[kb])) < 1e-9 * np.max(np.abs(c_true[kb]))
    assert np.max(np.abs(c[3 * L * L:] - c_true[3 * L * L:])) < 1e-9 * 3.0
    D = oracle.subtract(S, R, L, DK, DB, c)
    assert np.max(np.abs(D)) < 1e-8 * np.abs(S).max()


def test_P7_phi_closed_form():
    nx, ny = 36, 28
    S, R = _rng_pair(nx, ny, 25)
    L, DK, DB = 3, 0, 2
    G, _ = oracle.build_system(S, R, None, L, DK, DB)
    polys = _poly_list(DB)

    def power_sum(n, k):  # closed forms for k <= 2, numpy for the rest
        if k % 2 == 1:
            return 0.0
        if k == 0:
            return float(n)
        if k == 2:
            return (n * n - 1.0) / (3.0 * n)
        return float(np.sum(_xt(n) ** k))

    base = L * L
    for a, (p, q) in enumerate(polys):
        for b, (pp, qq) in enumerate(polys):
            expect = power_sum(nx, p + pp) * power_sum(ny, q + qq)
            assert abs(G[base + a, base + b] - expect) < 1e-12 * nx * ny


def test_P8_normal_equation_residual_on_output():
    p = starfield.make_pair(0, nx=96, ny=64, n_stars=50)
    S, R = p["S"], p["R"]
    L, DK, DB = 5, 1, 1
    c = oracle.solve(*oracle.build_system(S, R, None, L, DK, DB))
    D = oracle.subtract(S, R, L, DK, DB, c)
    w = (L - 1) // 2
    for t, (i, j) in enumerate(_poly_list(DK)):
        T = oracle.weighted_image(R, None, i, j)
        for u, v in [(0, 0), (w, -w), (-1, 2)]:
            r = oracle.lag_sum(T, D, u, v)
            assert abs(r) < 1e-10 * np.linalg.norm(T) * np.linalg.norm(S)
    for (pp, qq) in _poly_list(DB):
        P = oracle.poly_image(96, 64, pp, qq)
        assert abs(np.sum(P * D)) < 1e-10 * np.linalg.norm(P) * np.linalg.norm(S)


def test_P9_not_spd_error_path():
    R = np.full((24, 24), 5.0)
    S = np.random.default_rng(1).standard_normal((24, 24))
    G, h = oracle.build_system(S, R, None, 3, 1, 0)
    with pytest.raises(oracle.OracleError) as e:
        oracle.solve(G, h)
    assert e.value.code == -5
    R = np.zeros((24, 24))
    R[10, 11] = 1.0  # a single delta with DK >= 1: x*R and y*R are multiples of R
    G, h = oracle.build_system(S, R, None, 3, 1, 0)
    with pytest.raises(oracle.OracleError):
        oracle.solve(G, h)


def test_P10_linearity_in_S():
    S1, R = _rng_pair(32, 32, 31)
    S2, _ = _rng_pair(32, 32, 32)
    L, DK, DB = 3, 1, 1
    c1 = oracle.solve(*oracle.build_system(S1, R, None, L, DK, DB))
    c2 = oracle.solve(*oracle.build_system(S2, R, None, L, DK, DB))
    c12 = oracle.solve(*oracle.build_system(S1 + S2, R, None, L, DK, DB))
    assert np.max(np.abs(c12 - c1 - c2)) < 1e-10 * np.max(np.abs(c12))


# ---------------------------------------------------------------- subtraction vs library FFT
@pytest.mark.parametrize("DK", [0, 2])
def test_subtract_matches_fft_convolution(DK):
    """M = sum_t (xt^i yt^j R) (*) K_t by the convolution theorem (numpy FFT), any coefficients."""
    nx, ny, L, DB = 48, 40, 5, 2
    S, R = _rng_pair(nx, ny, 41)
    rng = np.random.default_rng(42)
    n = oracle.num_unknowns(L, DK, DB)
    c = rng.standard_normal(n)
    w = (L - 1) // 2
    X, Y = np.meshgrid(_xt(nx), _xt(ny))
    M = np.zeros((ny, nx))
    for t, (i, j) in enumerate(_poly_list(DK)):
        K = np.zeros((ny, nx))
        for v in range(-w, w + 1):
            for u in range(-w, w + 1):
                K[v % ny, u % nx] = c[_idx(L, t, u, v)]
        M += np.fft.irfft2(np.fft.rfft2(X**i * Y**j * R) * np.fft.rfft2(K), s=(ny, nx))
    B = sum(c[L * L * len(_poly_list(DK)) + s] * X**p * Y**q for s, (p, q) in enumerate(_poly_list(DB)))
    D = oracle.subtract(S, R, L, DK, DB, c)
    np.testing.assert_allclose(D, S - M - B, atol=1e-10 * np.abs(M).max())
    xs = np.array([0, 1, nx - 1, 17, 5])
    ys = np.array([0, ny - 1, 3, 22, ny - 2])
    np.testing.assert_allclose(oracle.subtract_at(S, R, L, DK, DB, c, xs, ys), D[ys, xs], rtol=0, atol=1e-12)


def test_system_entry_matches_assembled():
    S, R = _rng_pair(32, 24, 51)
    mask = (np.random.default_rng(52).random(R.shape) > 0.05).astype(np.uint8)
    L, DK, DB = 3, 1, 1
    G, h = oracle.build_system(S, R, mask, L, DK, DB)
    n = G.shape[0]
    rng = np.random.default_rng(53)
    for _ in range(25):
        r, c = rng.integers(0, n, 2)
        assert abs(oracle.system_entry(S, R, mask, L, DK, DB, r, c) - G[r, c]) <= 1e-12 * abs(G).max()
    for r in (0, 5, n - 1, n - 3):
        assert abs(oracle.system_entry(S, R, mask, L, DK, DB, r, -1) - h[r]) <= 1e-12 * abs(h).max()


def test_mask_semantics_C7():
    """Masked pixels are zeroed in S and R for the fit; P_s is not masked."""
    S, R = _rng_pair(32, 24, 61)
    mask = (np.random.default_rng(62).random(R.shape) > 0.2).astype(np.uint8)
    G1, h1 = oracle.build_system(S, R, mask, 3, 1, 1)
    G2, h2 = oracle.build_system(S * mask, R * mask, None, 3, 1, 1)
    np.testing.assert_allclose(G1, G2, rtol=0, atol=1e-12 * np.abs(G2).max())
    np.testing.assert_allclose(h1, h2, rtol=0, atol=1e-12 * np.abs(h2).max())


def test_invalid_arguments():
    S, R = _rng_pair(16, 16, 1)
    with pytest.raises(oracle.OracleError):
        oracle.build_system(S, R, None, 4, 1, 1)       # even L
    with pytest.raises(oracle.OracleError):
        oracle.build_system(S, R, None, 11, 1, 1)      # nx < 2L-1


def test_config0_conditioning_and_fit_quality():
    """Config 0 of BASELINE.json: the fit leaves noise-level residuals (sanity of the recipe)."""
    p = starfield.make_pair(0)
    G, h = oracle.build_system(p["S"], p["R"], None, p["L"], p["DK"], p["DB"])
    assert G.shape == (148, 148)
    c = oracle.solve(G, h)
    D = oracle.subtract(p["S"], p["R"], p["L"], p["DK"], p["DB"], c)
    # residual RMS ~ sqrt(sigma_S^2 + |K|^2 sigma_R^2), well below the star signal
    assert 4.0 < D.std() < 12.0
    assert abs(c[: 49].sum() - 1.0) < 0.1  # flux scaling of the constant kernel term ~ 1


# ---------------------------------------------------------------- f2: cross-convolution with a PSF stamp
def _stamp(P, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((P, P))            # deliberately asymmetric: a flipped or transposed tap layout fails


def test_convolve_stamp_delta_and_shift():
    """A unit tap at offset (u0, v0) moves the image by (+u0, +v0) with wrap-around (reading C6)."""
    rng = np.random.default_rng(3)
    img = rng.standard_normal((23, 31))
    P, w = 7, 3
    yy, xx = np.mgrid[:23, :31]
    for u0, v0 in [(0, 0), (2, -3), (-1, 1), (3, 3)]:
        st = np.zeros((P, P)); st[v0 + w, u0 + w] = 1.0
        out = oracle.convolve_stamp(img, st)
        assert np.array_equal(out, img[(yy - v0) % 23, (xx - u0) % 31])


def test_convolve_stamp_against_scipy_and_fft():
    """Two independent routes: scipy.ndimage.convolve(mode='wrap') and the convolution theorem with numpy FFTs."""
    from scipy import ndimage
    rng = np.random.default_rng(4)
    ny, nx, P = 40, 52, 9
    w = (P - 1) // 2
    img = rng.standard_normal((ny, nx)) * 50 + 100
    st = _stamp(P, 5)
    out = oracle.convolve_stamp(img, st)
    ref = ndimage.convolve(img, st, mode="wrap")
    assert np.max(np.abs(out - ref)) <= 1e-11 * np.max(np.abs(ref))
    emb = np.zeros((ny, nx))
    for v in range(-w, w + 1):
        for u in range(-w, w + 1):
            emb[v % ny, u % nx] = st[v + w, u + w]
    ref2 = np.fft.ifft2(np.fft.fft2(img) * np.fft.fft2(emb)).real
    assert np.max(np.abs(out - ref2)) <= 1e-11 * np.max(np.abs(ref2))
    # flux: sum(out) = sum(img) * sum(stamp)
    assert abs(out.sum() - img.sum() * st.sum()) <= 1e-9 * abs(img).sum() * abs(st).sum()


def test_convolve_stamp_is_the_model_term_of_the_subtraction_oracle():
    """D = S - R (*) K - B of the C oracle with DK = DB = 0, S = 0, b = 0 gives -(R (*) K): the two oracles
    (numpy shifts here, C loops there) must agree on the tap layout and the boundary."""
    rng = np.random.default_rng(6)
    ny, nx, P = 33, 29, 5
    R = rng.standard_normal((ny, nx)) * 10 + 30
    st = _stamp(P, 7)
    c = np.concatenate([st.ravel(), [0.0]])
    D = oracle.subtract(np.zeros((ny, nx)), R, P, 0, 0, c)
    out = oracle.convolve_stamp(R, st)
    assert np.max(np.abs(out + D)) <= 1e-12 * np.max(np.abs(out))


def test_convolve_stamp_at_matches_full():
    rng = np.random.default_rng(8)
    img = rng.standard_normal((37, 41))
    st = _stamp(7, 9)
    full = oracle.convolve_stamp(img, st)
    xs = np.array([0, 1, 40, 20, 3, 39]); ys = np.array([0, 36, 2, 18, 35, 36])
    got = oracle.convolve_stamp_at(img, st, xs, ys)
    assert np.max(np.abs(got - full[ys, xs])) <= 1e-12 * np.max(np.abs(full))
