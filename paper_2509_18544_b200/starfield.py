"""Seeded synthetic Roman-like star fields: the inputs of every test and of bench.py.

This module is the ONE piece of code shared by the CPU oracle's tests and the CUDA
path's tests/bench.  It holds no SFFT arithmetic (no weighted images, no normal
equations, no convolution with a fitted kernel): it only draws images.  numpy only.

The fields stand in for the OpenUniverse2024 simulated Roman images the paper runs on
(PAPER.md:43, 99, 105 -- 4088x4088 detector frames; not available here).  The recipe is
SURVEY.md section 8(d) / BASELINE.json `configs`:

* numpy ``default_rng(seed)`` (PCG64);
* star positions uniform in [0,nx) x [0,ny) at sub-pixel precision;
* fluxes from dN/dF ~ F^-2 on [1e2, 1e5] by inverse CDF;
* a star is a pixel-centre-sampled 2-D Gaussian of the *local* PSF (evaluated at the
  star's position), total flux F, rendered on a +-6 sigma stamp;
* the same star list in R (template) and S (science); the same sky constant in both,
  gradients only in S; transients are point sources in S only;
* noise is drawn independently for R and S after all signal has been added.

``xt, yt`` below are the centred pixel coordinates (2x+1-nx)/nx in (-1,1) and
``rho2 = (xt^2 + yt^2)/2``; they only parametrise how the PSF width and the sky vary
across the field.
"""
from __future__ import annotations

import numpy as np

__all__ = ["CONFIGS", "make_pair", "make_batch_science", "random_pair"]

# (name, nx, ny, n_stars, L, DK, DB, seed)
CONFIGS = {
    0: dict(name="tiny256", nx=256, ny=256, n_stars=200, L=7, DK=1, DB=0, seed=1),
    1: dict(name="mid1024", nx=1024, ny=1024, n_stars=2000, L=11, DK=2, DB=1, seed=2),
    2: dict(name="roman4088", nx=4088, ny=4088, n_stars=60000, L=11, DK=2, DB=2, seed=3),
    3: dict(name="batch4088", nx=4088, ny=4088, n_stars=60000, L=11, DK=2, DB=2, seed=3),
    4: dict(name="large_kernel4088", nx=4088, ny=4088, n_stars=60000, L=21, DK=3, DB=2, seed=5),
}

_FWHM = 2.3548200450309493


def _powerlaw_flux(rng, n, lo=1e2, hi=1e5):
    u = rng.random(n)
    return 1.0 / (1.0 / lo - u * (1.0 / lo - 1.0 / hi))


def _coords(x, n):
    return (2.0 * x + 1.0 - n) / n


def _render(img, xs, ys, flux, sig_a, sig_b, theta):
    """Add elliptical Gaussians (pixel-centre sampled) to img in place.

    sig_a, sig_b: per-star major/minor sigma; theta: position angle (radians).
    """
    ny, nx = img.shape
    ct, st = np.cos(theta), np.sin(theta)
    for k in range(xs.shape[0]):
        sa, sb = float(sig_a[k]), float(sig_b[k])
        h = int(np.ceil(6.0 * max(sa, sb)))
        x0, y0 = float(xs[k]), float(ys[k])
        ix, iy = int(np.floor(x0)), int(np.floor(y0))
        xa, xb = max(ix - h, 0), min(ix + h + 1, nx)
        ya, yb = max(iy - h, 0), min(iy + h + 1, ny)
        if xa >= xb or ya >= yb:
            continue
        dx = np.arange(xa, xb, dtype=np.float64) - x0
        dy = np.arange(ya, yb, dtype=np.float64) - y0
        DX, DY = np.meshgrid(dx, dy)
        a = ct[k] * DX + st[k] * DY
        b = -st[k] * DX + ct[k] * DY
        g = np.exp(-0.5 * ((a / sa) ** 2 + (b / sb) ** 2))
        img[ya:yb, xa:xb] += (float(flux[k]) / (2.0 * np.pi * sa * sb)) * g


def _local(xs, ys, nx, ny):
    xt = _coords(xs, nx)
    yt = _coords(ys, ny)
    return xt, yt, 0.5 * (xt * xt + yt * yt)


def _grid(nx, ny):
    xt = _coords(np.arange(nx, dtype=np.float64), nx)[None, :]
    yt = _coords(np.arange(ny, dtype=np.float64), ny)[:, None]
    return xt, yt


def _star_list(rng, nx, ny, n_stars):
    xs = rng.random(n_stars) * nx
    ys = rng.random(n_stars) * ny
    fl = _powerlaw_flux(rng, n_stars)
    return xs, ys, fl


def _transients(rng, nx, ny, n, lo=1e3, hi=1e4):
    xs = rng.random(n) * nx
    ys = rng.random(n) * ny
    fl = np.exp(rng.uniform(np.log(lo), np.log(hi), n))
    return xs, ys, fl


def _noise_poisson(rng, expected, read_sigma, scale=1.0):
    """Poisson on expected counts + Gaussian read noise, both scaled by `scale`
    about the expectation (scale=1/3 models the deeper template stack)."""
    lam = np.clip(expected, 0.0, None)
    pois = rng.poisson(lam).astype(np.float64) - lam
    read = rng.normal(0.0, read_sigma, expected.shape)
    return expected + scale * (pois + read)


def make_pair(config: int, *, nx=None, ny=None, n_stars=None, seed=None):
    """Return dict(S, R, L, DK, DB, noise_rms, name, stars) for BASELINE.json configs[config].

    nx/ny/n_stars/seed override the config's values (used by tests that want the
    same recipe at a size the oracle finishes quickly).  For config 3 this returns the
    template and science image b=0; see make_batch_science for the others.
    """
    c = dict(CONFIGS[config])
    nx = c["nx"] if nx is None else int(nx)
    ny = c["ny"] if ny is None else int(ny)
    n_stars = c["n_stars"] if n_stars is None else int(n_stars)
    seed = c["seed"] if seed is None else int(seed)
    rng = np.random.default_rng(seed)
    xs, ys, fl = _star_list(rng, nx, ny, n_stars)
    xt, yt, rho2 = _local(xs, ys, nx, ny)
    gx, gy = _grid(nx, ny)
    R = np.zeros((ny, nx))
    S = np.zeros((ny, nx))
    theta = np.zeros(n_stars)

    if config == 0:
        sig_r = np.full(n_stars, 1.5)
        sig_s = 2.0 + 0.002 * xs
        _render(R, xs, ys, fl, sig_r, sig_r, theta)
        _render(S, xs, ys, fl, sig_s, sig_s, theta)
        # one transient, position/flux fixed by the recipe (scaled with the frame)
        tx, ty, tf = np.array([131.3 * nx / 256.0]), np.array([124.6 * ny / 256.0]), np.array([5e3])
        ts = 2.0 + 0.002 * tx
        _render(S, tx, ty, tf, ts, ts, np.zeros(1))
        R += 100.0
        S += 100.0 + 0.01 * np.arange(nx, dtype=np.float64)[None, :]
        R += rng.normal(0.0, 5.0, R.shape)
        S += rng.normal(0.0, 5.0, S.shape)
        noise_rms = 5.0
    elif config == 1:
        sig_r = 1.4 * (1.0 + 0.15 * (2.0 * rho2 - 1.0))
        sig_s = 1.8 * (1.0 + 0.15 * (2.0 * rho2 - 1.0))
        _render(R, xs, ys, fl, sig_r, sig_r, theta)
        _render(S, xs, ys, fl, sig_s, sig_s, theta)
        R += 200.0
        S += 200.0 * (1.0 + 0.05 * gx)
        R = _noise_poisson(rng, R, 8.0)
        S = _noise_poisson(rng, S, 8.0)
        noise_rms = float(np.sqrt(200.0 + 64.0))
    elif config in (2, 3, 4):
        if config == 4:
            s_r = 2.0 * (1.0 + 0.15 * (2.0 * rho2 - 1.0))
            s_s = 3.0 + 1.0 * rho2
        else:
            s_r = (1.9 + 0.1 * rho2) / _FWHM
            s_s = (2.1 + 0.2 * rho2) / _FWHM
        theta[:] = np.deg2rad(30.0)
        _render(R, xs, ys, fl, s_r * 1.05, s_r * 0.95, theta)
        if config == 3:
            # template = config 2's R bit for bit (same seed, same draw order: the
            # transient draws are made and dropped); science images come from
            # make_batch_science
            _transients(rng, nx, ny, 20)
            R += 200.0
            R = _noise_poisson(rng, R, 8.0, scale=1.0 / 3.0)
            out = dict(c)
            out.update(nx=nx, ny=ny, n_stars=n_stars, R=R, S=None,
                       noise_rms=float(np.sqrt(200.0 + 64.0)), stars=(xs, ys, fl))
            out["S"] = make_batch_science(out, 0)
            return out
        _render(S, xs, ys, fl, s_s * 1.05, s_s * 0.95, theta)
        txs, tys, tfl = _transients(rng, nx, ny, 20)
        _, _, trho2 = _local(txs, tys, nx, ny)
        t_s = (3.0 + 1.0 * trho2) if config == 4 else (2.1 + 0.2 * trho2) / _FWHM
        _render(S, txs, tys, tfl, t_s * 1.05, t_s * 0.95, np.full(20, np.deg2rad(30.0)))
        R += 200.0
        S += 200.0 * (1.0 + 0.05 * gx + 0.02 * gy * gy)
        R = _noise_poisson(rng, R, 8.0, scale=1.0 / 3.0)
        S = _noise_poisson(rng, S, 8.0)
        noise_rms = float(np.sqrt(200.0 + 64.0))
    else:
        raise ValueError(f"unknown config {config}")

    out = dict(c)
    out.update(nx=nx, ny=ny, n_stars=n_stars, R=R, S=S, noise_rms=noise_rms, stars=(xs, ys, fl))
    return out


def make_batch_science(template: dict, b: int):
    """Science image b of BASELINE.json configs[3]: same stars as the template,
    own PSF perturbation, own noise and own 20 transients; seed 4000+b."""
    nx, ny = template["nx"], template["ny"]
    xs, ys, fl = template["stars"]
    rng = np.random.default_rng(4000 + int(b))
    delta = rng.uniform(-0.05, 0.15)
    eps = rng.uniform(-0.1, 0.1)
    _, _, rho2 = _local(xs, ys, nx, ny)
    gx, gy = _grid(nx, ny)
    s_s = ((2.1 + delta) + (0.2 + eps) * rho2) / _FWHM
    S = np.zeros((ny, nx))
    theta = np.full(xs.shape[0], np.deg2rad(30.0))
    _render(S, xs, ys, fl, s_s * 1.05, s_s * 0.95, theta)
    txs, tys, tfl = _transients(rng, nx, ny, 20)
    _, _, trho2 = _local(txs, tys, nx, ny)
    t_s = ((2.1 + delta) + (0.2 + eps) * trho2) / _FWHM
    _render(S, txs, tys, tfl, t_s * 1.05, t_s * 0.95, np.full(20, np.deg2rad(30.0)))
    S += 200.0 * (1.0 + 0.05 * gx + 0.02 * gy * gy)
    return _noise_poisson(rng, S, 8.0)


def random_pair(nx, ny, seed, *, sky=50.0, amp=20.0):
    """A structureless pair for edge-case tests: white noise + sky in R,
    an independent draw in S.  (Used where only shapes matter.)"""
    rng = np.random.default_rng(seed)
    R = sky + amp * rng.standard_normal((ny, nx))
    S = sky + amp * rng.standard_normal((ny, nx))
    return S, R
