"""Seeded synthetic workloads C0..C4 (BASELINE.json `configs`).

These are STAND-INS for the paper's datasets (HST images, AO / LOST PSFs: PAPER.md:320-324,
:444-446), which are not available; they have the shapes, value ranges and structure of the
paper's experiments.  This module serves both the CPU oracle and the CUDA library and holds
NONE of the method's arithmetic (no SGP/RL step, no objective, no operator of the library):
only the image-formation model g = Poisson(K * f + b) with numpy's FFT, plus random draws.
It imports neither `oracle` nor the CUDA binding.

Every workload is a dict:
  g      list of p detected images (sy x sx), float64, Poisson counts
  psf    list of p PSFs on the object grid (ny x nx), centred at (ny/2, nx/2), sum = 1
  b      list of p background constants
  truth  the object f~ on the object grid (ny x nx)
  S      (oy, ox, sy, sx): the image domain inside the object grid; None for periodic problems
  opts   option overrides (names of the sgp_options fields) for that config
  name, seed
"""
from __future__ import annotations

import numpy as np

BASE_SEED = 12102258


def _rng(idx: int, extra: int = 0) -> np.random.Generator:
    return np.random.default_rng(BASE_SEED + idx + 1000 * extra)


def _coords(ny, nx):
    y = np.arange(ny, dtype=np.float64)[:, None] - ny // 2
    x = np.arange(nx, dtype=np.float64)[None, :] - nx // 2
    return y, x


def _circ_conv(psf_centered, f):
    """circular convolution with the PSF centre moved to (0,0) (image formation, periodic case)"""
    K = np.fft.ifftshift(psf_centered)
    return np.fft.irfft2(np.fft.rfft2(K) * np.fft.rfft2(f), s=f.shape)


def _lin_conv_crop(psf_centered, f, S):
    """non-periodic convolution on a 2x zero-padded grid, cropped to S (boundary problems)"""
    ny, nx = f.shape
    PY, PX = 2 * ny, 2 * nx
    fp = np.zeros((PY, PX)); fp[:ny, :nx] = f
    kp = np.zeros((PY, PX)); kp[:ny, :nx] = psf_centered
    kp = np.roll(kp, (-(ny // 2), -(nx // 2)), axis=(0, 1))
    full = np.fft.irfft2(np.fft.rfft2(kp) * np.fft.rfft2(fp), s=(PY, PX))[:ny, :nx]
    oy, ox, sy, sx = S
    return full[oy:oy + sy, ox:ox + sx]


def _poisson(rng, mean):
    return rng.poisson(np.maximum(mean, 0.0)).astype(np.float64)


# ----------------------------------------------------------------------------- PSFs

def psf_gaussian(ny, nx, sigma):
    y, x = _coords(ny, nx)
    k = np.exp(-(y * y + x * x) / (2.0 * sigma * sigma))
    return k / k.sum()


def psf_airy(n, pupil_diameter_px=None):
    """|FFT2(circular pupil)|^2; pupil diameter n/2 px = Nyquist sampling (C1, C4)"""
    d = pupil_diameter_px if pupil_diameter_px is not None else n / 2.0
    y, x = _coords(n, n)
    pupil = ((y * y + x * x) <= (d / 2.0) ** 2).astype(np.float64)
    k = np.abs(np.fft.fftshift(np.fft.fft2(np.fft.ifftshift(pupil)))) ** 2
    return k / k.sum()


def psf_lbt(n, angle_deg):
    """two 8.4 m discs, centres 14.4 m apart (22.8 m edge to edge = n/2 px), baseline rotated (C2, C4b)"""
    px_per_m = (n / 2.0) / 22.8
    r = 0.5 * 8.4 * px_per_m
    half = 0.5 * 14.4 * px_per_m
    a = np.deg2rad(angle_deg)
    cy, cx = half * np.sin(a), half * np.cos(a)
    y, x = _coords(n, n)
    pupil = (((y - cy) ** 2 + (x - cx) ** 2) <= r * r) | (((y + cy) ** 2 + (x + cx) ** 2) <= r * r)
    k = np.abs(np.fft.fftshift(np.fft.fft2(np.fft.ifftshift(pupil.astype(np.float64))))) ** 2
    return k / k.sum()


def psf_gauss_moffat(ny, nx, sigma=2.0, fwhm=64.0, beta=2.5, core=0.8):
    """0.8 Gaussian core + 0.2 Moffat wing (C3); gamma from the FWHM"""
    y, x = _coords(ny, nx)
    r2 = y * y + x * x
    g = np.exp(-r2 / (2.0 * sigma * sigma)); g /= g.sum()
    gamma = fwhm / (2.0 * np.sqrt(2.0 ** (1.0 / beta) - 1.0))
    m = (1.0 + r2 / (gamma * gamma)) ** (-beta); m /= m.sum()
    k = core * g + (1.0 - core) * m
    return k / k.sum()


# ----------------------------------------------------------------------------- objects

def _add_stars(f, rng, count, flux_lo=1e3, flux_hi=1e5, ys=None, xs=None):
    ny, nx = f.shape
    if ys is None:
        ys = rng.integers(0, ny, count)
        xs = rng.integers(0, nx, count)
    flux = 10.0 ** rng.uniform(np.log10(flux_lo), np.log10(flux_hi), count)
    np.add.at(f, (ys, xs), flux)
    return f


def object_galaxies(n, rng, n_gal=5, n_stars=50):
    """exponential-disc and de Vaucouleurs galaxies plus point stars (C1, C4a, C4c)"""
    y, x = _coords(n, n)
    f = np.zeros((n, n))
    for i in range(n_gal):
        cy, cx = rng.uniform(-n / 4, n / 4, 2)
        q = rng.uniform(0.3, 1.0)
        th = rng.uniform(0.0, np.pi)
        scale = rng.uniform(n / 64.0, n / 16.0)
        flux = 10.0 ** rng.uniform(6.0, 8.0)
        yr = (y - cy) * np.cos(th) - (x - cx) * np.sin(th)
        xr = (y - cy) * np.sin(th) + (x - cx) * np.cos(th)
        r = np.sqrt(xr * xr + (yr / q) ** 2)
        prof = np.exp(-r / scale) if i % 2 == 0 else np.exp(-7.669 * ((r / scale) ** 0.25 - 1.0))
        f += flux * prof / prof.sum()
    return _add_stars(f, rng, n_stars)


def object_cluster(n, rng, n_stars=200):
    """open cluster with Plummer-profile radii plus a faint Gaussian nebula (C2, C4b)"""
    a = n / 16.0
    ys, xs = [], []
    while len(ys) < n_stars:
        u = rng.uniform(0.0, 1.0)
        r = a * np.sqrt(u / (1.0 - u))
        ph = rng.uniform(0.0, 2.0 * np.pi)
        yy, xx = int(round(n // 2 + r * np.sin(ph))), int(round(n // 2 + r * np.cos(ph)))
        if 0 <= yy < n and 0 <= xx < n:
            ys.append(yy); xs.append(xx)
    f = np.zeros((n, n))
    _add_stars(f, rng, n_stars, ys=np.array(ys), xs=np.array(xs))
    y, x = _coords(n, n)
    neb = np.exp(-(y * y + x * x) / (2.0 * (n / 8.0) ** 2))
    return f + 1e6 * neb / neb.sum()


# ----------------------------------------------------------------------------- configs

def c0_stars_gaussian(n=256, seed_idx=0):
    """C0: 20 point stars, Gaussian PSF sigma = 2 px, b = 10, periodic"""
    rng = _rng(seed_idx, n)
    truth = _add_stars(np.zeros((n, n)), rng, 20)
    psf = psf_gaussian(n, n, 2.0)
    b = 10.0
    g = _poisson(rng, _circ_conv(psf, truth) + b)
    opts = dict(L1=1e-10, L2=1e10, adaptive_L=0, m_alpha=3, armijo_memory=10, beta=1e-4, theta=0.4,
                max_iter=100, stop_rule=0)
    return dict(name=f"C0_{n}", seed=BASE_SEED + seed_idx, g=[g], psf=[psf], b=[b], truth=truth, S=None, opts=opts)


def c0_rect(ny=128, nx=320, seed_idx=7, n_stars=20):
    """the C0 recipe on a rectangular ny x nx grid (ragged shapes for the parity tests: ny != nx, radix-5 lengths)"""
    rng = _rng(seed_idx, ny * 4096 + nx)
    truth = _add_stars(np.zeros((ny, nx)), rng, n_stars)
    psf = psf_gaussian(ny, nx, 2.0)
    b = 10.0
    g = _poisson(rng, _circ_conv(psf, truth) + b)
    opts = dict(L1=1e-10, L2=1e10, adaptive_L=0, m_alpha=3, armijo_memory=10, beta=1e-4, theta=0.4,
                max_iter=100, stop_rule=0)
    return dict(name=f"C0_{ny}x{nx}", seed=BASE_SEED + seed_idx, g=[g], psf=[psf], b=[b], truth=truth, S=None, opts=opts)


def c1_galaxies_airy(n=512, seed_idx=1, max_iter=1000, stop_rule=2):
    """C1 (and C4a at n=4096, C4c at n=2048): galaxies + stars, Airy PSF, b = 20"""
    rng = _rng(seed_idx, n)
    truth = object_galaxies(n, rng)
    psf = psf_airy(n)
    b = 20.0
    g = _poisson(rng, _circ_conv(psf, truth) + b)
    opts = dict(max_iter=max_iter, stop_rule=stop_rule, disc_threshold=1.0)
    return dict(name=f"C1_{n}", seed=BASE_SEED + seed_idx, g=[g], psf=[psf], b=[b], truth=truth, S=None, opts=opts)


def c2_lbt_multi(n=512, seed_idx=2, max_iter=500, p=3):
    """C2 (and C4b at n=2048): p Fizeau images, baseline rotated by 180/p degrees, b_j = 15"""
    rng = _rng(seed_idx, n)
    truth = object_cluster(n, rng)
    psfs = [psf_lbt(n, 180.0 * j / p) for j in range(p)]
    b = [15.0] * p
    g = [_poisson(rng, _circ_conv(k, truth) + bj) for k, bj in zip(psfs, b)]
    opts = dict(max_iter=max_iter, stop_rule=0)
    return dict(name=f"C2_{n}x{p}", seed=BASE_SEED + seed_idx, g=g, psf=psfs, b=b, truth=truth, S=None, opts=opts)


def c3_boundary(s=1024, sbar=1280, seed_idx=3, n_stars=2000, max_iter=300, fwhm=64.0):
    """C3: image S (s x s) centred in the object grid S-bar (sbar x sbar); stars also outside S"""
    rng = _rng(seed_idx, sbar)
    off = (sbar - s) // 2
    S = (off, off, s, s)
    truth = _add_stars(np.zeros((sbar, sbar)), rng, n_stars)
    psf = psf_gauss_moffat(sbar, sbar, 2.0, fwhm * sbar / 1280.0 if sbar < 1280 else fwhm)
    b = 5.0
    g = _poisson(rng, _lin_conv_crop(psf, truth, S) + b)
    opts = dict(max_iter=max_iter, stop_rule=0, sigma_R=1e-2)
    return dict(name=f"C3_{s}in{sbar}", seed=BASE_SEED + seed_idx, g=[g], psf=[psf], b=[b], truth=truth, S=S, opts=opts)


def c4a(n=4096):
    w = c1_galaxies_airy(n, seed_idx=4, max_iter=200, stop_rule=0); w["name"] = f"C4a_{n}"; return w


def c4b(n=2048):
    w = c2_lbt_multi(n, seed_idx=5, max_iter=200); w["name"] = f"C4b_{n}x3"; return w


def c4c(n=2048):
    w = c1_galaxies_airy(n, seed_idx=6, max_iter=200, stop_rule=0); w["name"] = f"C4c_{n}"; return w


CONFIGS = {"C0": c0_stars_gaussian, "C0r": c0_rect, "C1": c1_galaxies_airy, "C2": c2_lbt_multi, "C3": c3_boundary,
           "C4a": c4a, "C4b": c4b, "C4c": c4c}


def make(name: str, **kw):
    return CONFIGS[name](**kw)
