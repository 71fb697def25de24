"""GPU parity: libsfft (through the C ABI binding) against the CPU oracle, element by element on
the same seeded inputs.  Tolerances are BASELINE.json north_star's, in the norm-wise form of
DESIGN.md readings C12/C13:
   G:  |dG_ij| <= 1e-10 sqrt(G_ii G_jj);   h: |dh_i| <= 1e-10 sqrt(G_ii) ||m.S||_2
   c:  max|da| <= 1e-8 max|a| (kernel block), max|db| <= 1e-8 max|b| (background block)
   D:  max|dD| <= 1e-6 * noise RMS of the science image
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2509_18544_b200 import SfftError, SfftPlan, starfield

pytestmark = pytest.mark.gpu

TOL_G, TOL_H, TOL_C, TOL_D = 1e-10, 1e-10, 1e-8, 1e-6


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def run_gpu(S, R, mask, L, DK, DB):
    ny, nx = S.shape
    p = SfftPlan(nx, ny, L, DK, DB)
    dS, dR = dev(S), dev(R)
    dM = dev(mask) if mask is not None else None
    p.build_system(dS, dR, dM)
    G, h = p.get_system()
    p.solve()
    D, c = p.subtract()
    p.sync_status()
    return p, G.cpu().numpy(), h.cpu().numpy(), c.cpu().numpy(), D.cpu().numpy()


def assert_system(G, h, G0, h0, Sf):
    d = np.sqrt(np.diag(G0))
    assert np.all(np.abs(G - G0) <= TOL_G * np.outer(d, d)), np.max(np.abs(G - G0) / np.outer(d, d))
    assert np.all(np.abs(h - h0) <= TOL_H * d * np.linalg.norm(Sf)), np.max(np.abs(h - h0) / (d * np.linalg.norm(Sf)))
    assert np.array_equal(G, G.T)
    # the plain element-wise relative error, for every entry that is not a cancellation: floor 1e-6 of the scale
    big = np.abs(G0) >= 1e-6 * np.outer(d, d)
    assert np.max(np.abs(G - G0)[big] / np.abs(G0)[big]) <= 1e-8


def assert_coeffs(c, c0, nker):
    assert np.max(np.abs(c - c0)[:nker]) <= TOL_C * np.max(np.abs(c0[:nker]))
    assert np.max(np.abs(c - c0)[nker:]) <= TOL_C * np.max(np.abs(c0[nker:]))


def full_parity(S, R, mask, L, DK, DB, noise_rms):
    p, G, h, c, D = run_gpu(S, R, mask, L, DK, DB)
    G0, h0 = oracle.build_system(S, R, mask, L, DK, DB)
    Sf = S * mask if mask is not None else S
    assert_system(G, h, G0, h0, Sf)
    c0 = oracle.solve(G0, h0)
    nker = L * L * (DK + 1) * (DK + 2) // 2
    assert_coeffs(c, c0, nker)
    D0 = oracle.subtract(S, R, L, DK, DB, c0)
    assert np.max(np.abs(D - D0)) <= TOL_D * noise_rms
    # convolution alone (oracle coefficients through the GPU subtract), reading C13
    D1 = p.subtract_with(dev(c0)).cpu().numpy()
    assert np.max(np.abs(D1 - D0)) <= TOL_D * noise_rms
    p.destroy()
    return c, D


# sizes spanning several FFT tiles and ragged tails: powers of two (no padding), non powers of two
# (zero padding + native-grid wrap corrections), nx != ny, odd sizes, every polynomial degree.
@pytest.mark.parametrize("nx,ny,L,DK,DB,masked", [
    (128, 64, 5, 1, 1, False),
    (100, 72, 5, 1, 1, False),
    (100, 72, 5, 2, 2, True),
    (61, 67, 7, 0, 0, False),
    (90, 130, 3, 3, 3, False),
    (200, 120, 9, 1, 2, True),
    (64, 64, 1, 2, 1, False),
    (257, 129, 5, 2, 0, False),
])
def test_parity_small(nx, ny, L, DK, DB, masked):
    S, R = starfield.random_pair(nx, ny, seed=nx * 7 + ny)
    mask = None
    if masked:
        rng = np.random.default_rng(5)
        mask = (rng.random((ny, nx)) > 0.05).astype(np.uint8)
        yy, xx = np.mgrid[:ny, :nx]
        mask[(yy - ny // 3) ** 2 + (xx - nx // 2) ** 2 < 36] = 0  # a masked disc
    full_parity(S, R, mask, L, DK, DB, noise_rms=20.0)


# L >= 13 takes the wide-lag instances of the a2 kernels (lag bound 2w > 20 in the Omega pass: split lag halves /
# the widest row-reduction instance), which configs[0..3] never reach (L <= 11).  Element by element against the oracle.
@pytest.mark.parametrize("nx,ny,L,DK,DB,masked", [
    (96, 80, 13, 1, 1, False),
    (128, 100, 21, 0, 0, False),
    (100, 90, 15, 2, 1, True),      # non power of two, masked, 21 template pairs
    (75, 131, 17, 1, 2, False),     # odd sizes, nx != ny
    (64, 64, 21, 1, 0, False),      # power of two, the largest kernel the library takes
])
def test_parity_wide_kernels(nx, ny, L, DK, DB, masked):
    S, R = starfield.random_pair(nx, ny, seed=1000 + nx + ny + L)
    mask = None
    if masked:
        rng = np.random.default_rng(15)
        mask = (rng.random((ny, nx)) > 0.05).astype(np.uint8)
        mask[:2, 5:30] = 0
    full_parity(S, R, mask, L, DK, DB, noise_rms=20.0)


@pytest.mark.parametrize("nx,ny", [(72, 4096), (4096, 72)])
def test_longest_sides(nx, ny):
    """The longest side the library takes (include/sfft.h: SFFT_MAX_SIDE = 4096): no padding along it, 1024 / 512
    padded points along the short one, wrap corrections on the short side only."""
    S, R = starfield.random_pair(nx, ny, seed=nx + ny)
    full_parity(S, R, None, 5, 1, 1, noise_rms=20.0)


def test_sides_above_the_limit_are_rejected():
    for nx, ny in ((4097, 64), (64, 5000)):
        with pytest.raises(SfftError):
            SfftPlan(nx, ny, 3, 0, 0)


def test_masked_then_unmasked_pair_on_one_plan():
    """A plan used with a mask keeps a second set of (unmasked) template spectra for the subtraction (reading C7);
    the next pair WITHOUT a mask, and another template, must not convolve the stale set."""
    nx, ny, L, DK, DB = 100, 72, 5, 1, 1
    S1, R1 = starfield.random_pair(nx, ny, seed=201)
    S2, R2 = starfield.random_pair(nx, ny, seed=202)
    rng = np.random.default_rng(3)
    mask = (rng.random((ny, nx)) > 0.05).astype(np.uint8)
    p = SfftPlan(nx, ny, L, DK, DB)
    nker = L * L * 3
    for S, R, m in ((S1, R1, mask), (S2, R2, None), (S1, R1, mask), (S2, R1, None)):
        p.build_system(dev(S), dev(R), dev(m) if m is not None else None)
        p.solve()
        D, c = p.subtract()
        p.sync_status()
        G0, h0 = oracle.build_system(S, R, m, L, DK, DB)
        c0 = oracle.solve(G0, h0)
        assert_coeffs(c.cpu().numpy(), c0, nker)
        D0 = oracle.subtract(S, R, L, DK, DB, c0)
        assert np.max(np.abs(D.cpu().numpy() - D0)) <= TOL_D * 20.0
    # the batched calls after a masked single pair
    p.set_template(dev(R2))
    Ds, cs = p.subtract_batch([dev(S2), dev(S1)])
    p.sync_status()
    for S, D in ((S2, Ds[0]), (S1, Ds[1])):
        G0, h0 = oracle.build_system(S, R2, None, L, DK, DB)
        D0 = oracle.subtract(S, R2, L, DK, DB, oracle.solve(G0, h0))
        assert np.max(np.abs(D.cpu().numpy() - D0)) <= TOL_D * 20.0
    p.destroy()


def test_masked_pair_on_the_pipelined_column_path():
    """600 x 520 pads to 1024 x 1024: the persistent column kernels (My >= 512), tile-major spectra,
    a mask (separate unmasked template spectra for the subtraction, reading C7) and wrap corrections."""
    S, R = starfield.random_pair(600, 520, seed=41)
    rng = np.random.default_rng(6)
    mask = (rng.random((520, 600)) > 0.03).astype(np.uint8)
    yy, xx = np.mgrid[:520, :600]
    mask[(yy - 100) ** 2 + (xx - 450) ** 2 < 64] = 0
    mask[:3, :40] = 0                                     # masked pixels on the frame border (wrap path)
    full_parity(S, R, mask, 7, 2, 1, noise_rms=20.0)


def test_tall_frame_on_the_compile_time_4096_column_path():
    """72 x 4000 pads to 128 x 4096: the My = 4096 instances of the pipelined column kernels (the ones the
    4088 x 4088 bench runs) on a frame the oracle finishes in seconds: 96 zero rows, the packed column
    kx = 0, a mask and wrap corrections."""
    nx, ny = 72, 4000
    S, R = starfield.random_pair(nx, ny, seed=77)
    rng = np.random.default_rng(8)
    mask = (rng.random((ny, nx)) > 0.04).astype(np.uint8)
    mask[ny - 2:, :10] = 0
    full_parity(S, R, mask, 5, 2, 1, noise_rms=20.0)


def test_debug_read_spectrum_layout():
    """The test hook hands spectra out as [My][Hx+1] (kx = 0..Mx/2) whatever the device layout is: compare the
    template spectra (weights xt^i yt^j) with numpy's rfft2 of the zero-padded weighted frames -- this pins the row and
    column transforms, the untangle and the separation of the packed column kx = 0 / Mx/2 on their own."""
    S, R = starfield.random_pair(96, 80, seed=5)
    p = SfftPlan(96, 80, 3, 1, 0)
    p.build_system(dev(S), dev(R))
    Mx, My = p.debug_read(7)
    for t in range(3):
        i, j = oracle.poly_index(t)
        spec = p.debug_read(0, t)
        pad = np.zeros((My, Mx)); pad[:80, :96] = oracle.weighted_image(R, None, i, j)
        ref = np.fft.rfft2(pad)
        assert spec.shape == ref.shape
        assert np.max(np.abs(spec - ref)) <= 1e-9 * np.max(np.abs(ref)), t
    pad = np.zeros((My, Mx)); pad[:80, :96] = S
    assert np.max(np.abs(p.debug_read(1) - np.fft.rfft2(pad))) <= 1e-9 * np.max(np.abs(pad)) * 80 * 96
    p.destroy()


def test_minimum_frame_size():
    L = 5
    S, R = starfield.random_pair(2 * L - 1, 2 * L - 1, seed=3)
    full_parity(S, R, None, L, 0, 0, noise_rms=20.0)


def test_config0_tiny():
    c = starfield.make_pair(0)
    full_parity(c["S"], c["R"], None, c["L"], c["DK"], c["DB"], c["noise_rms"])


def test_config1_mid():
    c = starfield.make_pair(1)
    full_parity(c["S"], c["R"], None, c["L"], c["DK"], c["DB"], c["noise_rms"])


def test_config2_recipe_reduced_non_pow2():
    """configs[2]'s recipe (elliptical PSFs, deeper template, transients) at 511 x 389."""
    c = starfield.make_pair(2, nx=511, ny=389, n_stars=1000)
    full_parity(c["S"], c["R"], None, 11, 2, 2, c["noise_rms"])


def test_P2_identity_on_gpu():
    _, R = starfield.random_pair(96, 80, seed=11)
    p, G, h, c, D = run_gpu(R, R, None, 5, 1, 1)
    e = np.zeros_like(c); e[2 * 5 + 2] = 1.0
    assert np.max(np.abs(c - e)) < 1e-9
    assert np.max(np.abs(D)) < 1e-8


def test_P5_pure_shift_on_gpu():
    _, R = starfield.random_pair(100, 72, seed=12)
    S = np.roll(R, (2, -1), axis=(0, 1))  # S(x,y) = R(x+1, y-2): delta at (u,v) = (-1, 2)
    p, G, h, c, D = run_gpu(S, R, None, 5, 0, 0)
    k = c[:25].reshape(5, 5)
    assert abs(k[2 + 2, 2 - 1] - 1.0) < 1e-9 and np.abs(D).max() < 1e-8


def test_not_spd_is_reported():
    R = np.full((64, 64), 3.0)
    S, _ = starfield.random_pair(64, 64, seed=1)
    p = SfftPlan(64, 64, 3, 1, 0)
    p.build_system(dev(S), dev(R))
    p.solve()
    with pytest.raises(SfftError) as ei:
        p.sync_status()
    assert ei.value.code == -5
    with pytest.raises(oracle.OracleError):
        G0, h0 = oracle.build_system(S, R, None, 3, 1, 0)
        oracle.solve(G0, h0)


def test_state_and_argument_errors():
    with pytest.raises(SfftError):
        SfftPlan(64, 64, 4, 0, 0)       # even L
    with pytest.raises(SfftError):
        SfftPlan(8, 64, 5, 0, 0)        # nx < 2L-1
    with pytest.raises(SfftError):
        SfftPlan(64, 64, 3, 4, 0)       # DK out of range
    p = SfftPlan(64, 64, 3, 0, 0)
    with pytest.raises(SfftError) as ei:
        p.solve()
    assert ei.value.code == -4
    with pytest.raises(SfftError):
        p.subtract()
    with pytest.raises(SfftError):
        p.subtract_batch([torch.zeros(64, 64, dtype=torch.float64, device="cuda")])
    with pytest.raises(TypeError):
        p.build_system(torch.zeros(64, 64), torch.zeros(64, 64))


def test_batched_matches_single_and_oracle():
    """configs[3]'s structure at reduced size: one template, B science images; template-side work
    once.  Each image must match the single-pair path to rounding level and the oracle to tolerance."""
    t = starfield.make_pair(3, nx=300, ny=260, n_stars=600)
    B, L, DK, DB = 3, 11, 2, 2
    Ss = [t["S"]] + [starfield.make_batch_science(t, b) for b in range(1, B)]
    p = SfftPlan(300, 260, L, DK, DB)
    dR = dev(t["R"]); dSs = [dev(s) for s in Ss]
    p.set_template(dR)
    Ds, cs = p.subtract_batch(dSs)
    p.sync_status()
    cs = cs.cpu().numpy()
    for b in range(B):
        p1, G, h, c, D = run_gpu(Ss[b], t["R"], None, L, DK, DB)
        # same sums, different split order (several images per Theta pass): rounding level, an order inside C12 / C13
        assert np.max(np.abs(c - cs[b])) <= 0.1 * TOL_C * np.max(np.abs(c))
        assert np.max(np.abs(D - Ds[b].cpu().numpy())) <= 0.1 * TOL_D * t["noise_rms"]
        G0, h0 = oracle.build_system(Ss[b], t["R"], None, L, DK, DB)
        c0 = oracle.solve(G0, h0)
        assert_coeffs(cs[b], c0, L * L * 6)
        D0 = oracle.subtract(Ss[b], t["R"], L, DK, DB, c0)
        assert np.max(np.abs(Ds[b].cpu().numpy() - D0)) <= TOL_D * t["noise_rms"]
    # P10: linearity in S for a fixed template
    p.subtract_batch([dSs[0] + dSs[1]], coeffs=(c12 := torch.empty((1, p.n), dtype=torch.float64, device="cuda")))
    p.sync_status()
    assert np.max(np.abs(c12.cpu().numpy()[0] - cs[0] - cs[1])) <= 1e-9 * np.max(np.abs(cs[0]))


def test_difference_host_matches_device_path():
    c = starfield.make_pair(0)
    p, G, h, cd, D = run_gpu(c["S"], c["R"], None, c["L"], c["DK"], c["DB"])
    Dh, ch = p.difference_host(torch.from_numpy(c["S"]).pin_memory(), torch.from_numpy(c["R"]).pin_memory())
    assert np.array_equal(Dh.numpy(), D) and np.array_equal(ch.numpy(), cd)


def test_difference_host_batch_matches_device_batch():
    """The PCIe-pipelined host call (three staging slots, two copy streams): B = 7 images (two full turns of the slots and
    a ragged one) must reproduce the device-resident batched call bit for bit, with and without a mask."""
    nx, ny, L, DK, DB, B = 100, 72, 5, 1, 1, 7
    _, R = starfield.random_pair(nx, ny, seed=300)
    Ss = [starfield.random_pair(nx, ny, seed=301 + b)[0] for b in range(B)]
    rng = np.random.default_rng(4)
    for mask in (None, (rng.random((ny, nx)) > 0.05).astype(np.uint8)):
        p = SfftPlan(nx, ny, L, DK, DB)
        p.set_template(dev(R), dev(mask) if mask is not None else None)
        Ds, cs = p.subtract_batch([dev(s) for s in Ss])
        p.sync_status()
        hm = torch.from_numpy(mask).pin_memory() if mask is not None else None
        Dh, ch = p.difference_host_batch(torch.from_numpy(R).pin_memory(), [torch.from_numpy(s).pin_memory() for s in Ss], hm)
        for b in range(B):
            # (the device call runs the images in groups of four through one Theta pass, the host call one by one: the
            #  same sums in another split order -- rounding level, as in test_batched_groups_of_images_masked)
            assert np.max(np.abs(ch[b].numpy() - cs[b].cpu().numpy())) <= 1e-10 * np.max(np.abs(ch[b].numpy())), b
            assert np.max(np.abs(Dh[b].numpy() - Ds[b].cpu().numpy())) <= 1e-8 * 20.0, b
        Dh2, ch2 = p.difference_host_batch(torch.from_numpy(R).pin_memory(), [torch.from_numpy(s).pin_memory() for s in Ss], hm)
        for b in range(B):
            assert torch.equal(Dh[b], Dh2[b]) and torch.equal(ch[b], ch2[b])
        p.destroy()


# ---------------------------------------------------------------- f2: cross-convolution with a PSF stamp
# Bar: |out_gpu - out_oracle| <= 1e-11 * max|img| * sum|stamp| everywhere.  The FFT route's rounding error is
# ~ log2(Mx My) * 2^-53 * max|img| * sum|stamp| ~ 3e-15 of that product, so the bar has three
# orders of margin and still catches a wrong tap, a flipped stamp or a missed border correction (errors ~ 1e-2).
TOL_CONV = 1e-11


def _psf_stamp(P, seed, sigma=1.3):
    """A normalised, deliberately off-centre and asymmetric PSF-like stamp."""
    rng = np.random.default_rng(seed)
    w = (P - 1) // 2
    yy, xx = np.mgrid[-w:w + 1, -w:w + 1]
    st = np.exp(-0.5 * (((xx - 0.3) / sigma) ** 2 + ((yy + 0.2) / (1.4 * sigma)) ** 2)) + 0.01 * rng.random((P, P))
    return st / st.sum()


@pytest.mark.parametrize("nx,ny,P,DK,DB", [
    (128, 64, 5, 0, 0),      # powers of two: no padding, no border correction
    (100, 72, 7, 2, 1),      # zero padding + native-grid wrap correction; a plan whose DK, DB are not 0
    (61, 67, 3, 1, 0),       # odd sizes
    (90, 130, 1, 0, 0),      # a single tap
    (600, 520, 11, 0, 0),    # the pipelined column kernels (My = 1024)
    (72, 4000, 5, 0, 0),     # the My = 4096 instances
])
def test_convolve_stamp_parity(nx, ny, P, DK, DB):
    S, R = starfield.random_pair(nx, ny, seed=nx + 3 * ny)
    st = _psf_stamp(P, seed=P) if P > 1 else np.array([[0.7]])
    p = SfftPlan(nx, ny, P, DK, DB)
    out = p.convolve_stamp(dev(R), dev(st)).cpu().numpy()
    ref = oracle.convolve_stamp(R, st)
    assert np.max(np.abs(out - ref)) <= TOL_CONV * np.max(np.abs(R)) * np.abs(st).sum()
    p.destroy()


def test_cross_convolve_then_subtract_on_one_plan():
    """Pipeline order: cross-convolve both images, then run the SFFT subtraction on the
    cross-convolved pair with the SAME plan: the convolution must not disturb the plan's state."""
    nx, ny, L = 100, 72, 5
    S, R = starfield.random_pair(nx, ny, seed=11)
    psfS, psfR = _psf_stamp(L, 1, 1.1), _psf_stamp(L, 2, 0.9)
    p = SfftPlan(nx, ny, L, 1, 1)
    Sc, Rc = p.cross_convolve(dev(S), dev(R), dev(psfS), dev(psfR))
    Sc0, Rc0 = oracle.convolve_stamp(S, psfR), oracle.convolve_stamp(R, psfS)
    assert np.max(np.abs(Sc.cpu().numpy() - Sc0)) <= TOL_CONV * np.max(np.abs(S)) * np.abs(psfR).sum()
    assert np.max(np.abs(Rc.cpu().numpy() - Rc0)) <= TOL_CONV * np.max(np.abs(R)) * np.abs(psfS).sum()
    p.build_system(Sc, Rc)
    G, h = p.get_system()
    p.solve()
    D, c = p.subtract()
    p.sync_status()
    G0, h0 = oracle.build_system(Sc0, Rc0, None, L, 1, 1)
    assert_system(G.cpu().numpy(), h.cpu().numpy(), G0, h0, Sc0)
    c0 = oracle.solve(G0, h0)
    assert_coeffs(c.cpu().numpy(), c0, L * L * 3)
    D0 = oracle.subtract(Sc0, Rc0, L, 1, 1, c0)
    assert np.max(np.abs(D.cpu().numpy() - D0)) <= TOL_D * 20.0
    p.destroy()


def test_scratch_users_between_build_and_subtract():
    """sfft_convolve_stamp and sfft_decorrelation_stamp use the science-spectrum and intermediate buffers as scratch; both
    are dead between the plan's calls, so calling them between build_system, solve and subtract must change nothing."""
    nx, ny, L = 100, 72, 5
    S, R = starfield.random_pair(nx, ny, seed=21)
    p = SfftPlan(nx, ny, L, 1, 1)
    p.build_system(dev(S), dev(R)); p.solve(); D0, c0 = p.subtract(); p.sync_status()
    D0, c0 = D0.clone(), c0.clone()
    st = dev(_psf_stamp(L, 3, 1.0))
    p.build_system(dev(S), dev(R))
    junk = p.convolve_stamp(dev(R), st)
    p.solve()
    W = p.decorrelation_stamp(st, st, st, 4.0, 1.0, 32)
    junk2 = p.convolve_stamp(dev(S), W)
    D1, c1 = p.subtract()
    p.sync_status()
    assert torch.equal(c0, c1) and torch.equal(D0, D1)
    p.destroy()


def test_convolve_stamp_argument_errors():
    p = SfftPlan(64, 64, 3, 0, 0)
    img = torch.zeros((64, 64), dtype=torch.float64, device="cuda")
    st = torch.zeros((3, 3), dtype=torch.float64, device="cuda")
    with pytest.raises(SfftError):
        p.convolve_stamp(img, st, out=img)          # aliased
    with pytest.raises(ValueError):
        p.convolve_stamp(img, torch.zeros((5, 5), dtype=torch.float64, device="cuda"))
    p.destroy()


def test_stamp_mode_1000_cutout():
    """f4: the path on a 1000 x 1000 stamp ("minimum size of 1000 x 1000 px") with the configs[2]
    recipe, L = 11, DK = 2, DB = 2: 1000 pads to 1024 (wrap corrections on), n = 732, full element-wise parity."""
    c = starfield.make_pair(2, nx=1000, ny=1000, n_stars=3600)
    full_parity(c["S"], c["R"], None, 11, 2, 2, c["noise_rms"])


@pytest.mark.parametrize("B", [2, 4, 5, 9])
def test_batched_groups_of_images_masked(B):
    """The batched path takes the science images up to four at a time through one Theta pass (4 NK pairs over NK + 4
    spectra) and pipelines the groups; full and ragged groups, a mask and a zero-padded frame, every image against
    the single-pair path (same sums in another split order, so the bar is rounding level: 1e-10 relative on the
    coefficients, 1e-8 of the noise RMS on D)."""
    nx, ny, L, DK, DB = 100, 72, 5, 2, 1
    _, R = starfield.random_pair(nx, ny, seed=100)
    Ss = [starfield.random_pair(nx, ny, seed=101 + b)[0] for b in range(B)]
    rng = np.random.default_rng(9)
    mask = (rng.random((ny, nx)) > 0.04).astype(np.uint8)
    p = SfftPlan(nx, ny, L, DK, DB)
    p.set_template(dev(R), dev(mask))
    Ds, cs = p.subtract_batch([dev(s) for s in Ss])
    p.sync_status()
    cs = cs.cpu().numpy()
    for b in range(B):
        p1, G, h, c, D = run_gpu(Ss[b], R, mask, L, DK, DB)
        assert np.max(np.abs(c - cs[b])) <= 1e-10 * np.max(np.abs(c)), b
        assert np.max(np.abs(D - Ds[b].cpu().numpy())) <= 1e-8 * 20.0, b
        p1.destroy()
    p.destroy()
