"""Seeded phantom generators (no transform arithmetic lives here).

Geometry convention shared by every consumer: pixel ``img[iy, ix]`` has centred
coordinates X = ix - c, Y = iy - c with c = N // 2.  Disc rasterisation is
binary: a pixel takes the value iff (ix-cx)^2 + (iy-cy)^2 <= r^2.  Every disc
satisfies |centre - c| + r <= N/2 - 2 (inside the inscribed circle).
"""
import math

import numpy as np


def _disc_params(rng, N, n_disks, rmin, rmax, vmin, vmax):
    c = N // 2
    out = []
    for _ in range(n_disks):
        r = rng.uniform(rmin, rmax)
        rho_max = max(N / 2.0 - 2.0 - r, 0.0)
        rho = rho_max * math.sqrt(rng.uniform())
        phi = rng.uniform(0.0, 2.0 * math.pi)
        cx = c + rho * math.cos(phi)
        cy = c + rho * math.sin(phi)
        v = rng.uniform(vmin, vmax)
        out.append((cx, cy, r, v))
    return out


def _disc_mask(N, cx, cy, r):
    """Boolean mask and the bounding box it lives in (keeps 2048^2 cheap)."""
    x_lo = max(int(math.floor(cx - r)), 0)
    x_hi = min(int(math.ceil(cx + r)) + 1, N)
    y_lo = max(int(math.floor(cy - r)), 0)
    y_hi = min(int(math.ceil(cy + r)) + 1, N)
    ix = np.arange(x_lo, x_hi)[None, :]
    iy = np.arange(y_lo, y_hi)[:, None]
    m = (ix - cx) ** 2 + (iy - cy) ** 2 <= r * r
    return (slice(y_lo, y_hi), slice(x_lo, x_hi)), m


def additive_disks(N, seed, n_disks, rmin, rmax, vmin, vmax, noise_sigma=0.0):
    """Sum of uniform discs (+ optional white Gaussian noise on every pixel)."""
    rng = np.random.default_rng(seed)
    img = np.zeros((N, N), dtype=np.float64)
    for cx, cy, r, v in _disc_params(rng, N, n_disks, rmin, rmax, vmin, vmax):
        sl, m = _disc_mask(N, cx, cy, r)
        img[sl][m] += v
    if noise_sigma > 0.0:
        img += rng.normal(0.0, noise_sigma, size=(N, N))
    return img.astype(np.float32)


def painted_disks(N, seed, n_disks, rmin, rmax, levels=(1.0 / 3.0, 2.0 / 3.0, 1.0)):
    """Piecewise-constant phantom: discs painted in order (overwrite)."""
    rng = np.random.default_rng(seed)
    img = np.zeros((N, N), dtype=np.float64)
    for i, (cx, cy, r, _) in enumerate(_disc_params(rng, N, n_disks, rmin, rmax, 0.0, 1.0)):
        sl, m = _disc_mask(N, cx, cy, r)
        img[sl][m] = levels[i % len(levels)]
    return img.astype(np.float32)


def two_sphere_slice(N, w=1.5, kappa=1.0):
    """Deterministic two-sphere slice with an edge-enhanced (Laplacian) rim.

    Two discs of radius r0 = 0.15 N centred at (c +- 0.15 N, c).  Radial
    profile f(r) = S(u) + kappa * w^2 * lap S(u), u = (r0 - r)/w,
    S(u) = (1 + erf u)/2 and lap g = g'' + g'/r (2-D radial Laplacian), i.e.
    w^2 lap S = S''(u) - (w/r) S'(u).  Stand-in for the phase-contrast slice of
    two glass spheres.
    """
    from scipy.special import erf  # phantom profile only

    c = N // 2
    r0 = 0.15 * N
    iy, ix = np.mgrid[0:N, 0:N].astype(np.float64)
    img = np.zeros((N, N), dtype=np.float64)
    for sx in (-1.0, 1.0):
        cx = c + sx * 0.15 * N
        cy = float(c)
        r = np.hypot(ix - cx, iy - cy)
        u = (r0 - r) / w
        e = np.exp(-u * u) / math.sqrt(math.pi)      # S'(u)
        S = 0.5 * (1.0 + erf(u))
        Spp = -2.0 * u * e                           # S''(u)
        rr = np.maximum(r, 0.5)                      # S'(u) vanishes there anyway
        img += S + kappa * (Spp - (w / rr) * e)
    return img.astype(np.float32)


def make_image(cfg_id: int):
    """The seeded phantom of BASELINE.json config ``cfg_id`` (1-4)."""
    from .configs import CONFIGS

    cfg = CONFIGS[cfg_id]
    if cfg_id == 1:
        return additive_disks(cfg.N, cfg.seed, 3, 4.0, 16.0, 0.5, 1.0)
    if cfg_id == 2:
        return additive_disks(cfg.N, cfg.seed, 20, 8.0, 64.0, 0.0, 1.0, noise_sigma=0.01)
    if cfg_id == 3:
        return painted_disks(cfg.N, cfg.seed, 50, 8.0, 128.0)
    if cfg_id == 4:
        return two_sphere_slice(cfg.N)
    raise ValueError("make_image covers configs 1-4; use make_batch_slice for 5")


def make_batch_slice(i: int, N: int = 2048):
    """Slice ``i`` of config 5: 20 additive discs, r~U[32,256], v~U[0,1]."""
    scale = N / 2048.0
    return additive_disks(N, 5000 + i, 20, 32.0 * scale, 256.0 * scale, 0.0, 1.0)


# ---- small analytic test images (used by the oracle pins) -------------------

def gaussian_blob(N, x0, y0, s):
    """exp(-((X-x0)^2 + (Y-y0)^2) / (2 s^2)) in centred coordinates, float64."""
    c = N // 2
    iy, ix = np.mgrid[0:N, 0:N].astype(np.float64)
    return np.exp(-(((ix - c) - x0) ** 2 + ((iy - c) - y0) ** 2) / (2.0 * s * s))


def single_disk(N, x0, y0, r, value=1.0, supersample=1):
    """Uniform disc, centre (x0,y0) in centred coordinates; optional s x s
    supersampled coverage (supersample=1 -> binary raster)."""
    c = N // 2
    if supersample == 1:
        iy, ix = np.mgrid[0:N, 0:N].astype(np.float64)
        return value * (((ix - c) - x0) ** 2 + ((iy - c) - y0) ** 2 <= r * r).astype(np.float64)
    s = supersample
    off = (np.arange(s) + 0.5) / s - 0.5
    iy, ix = np.mgrid[0:N, 0:N].astype(np.float64)
    acc = np.zeros((N, N))
    for oy in off:
        for ox in off:
            acc += (((ix - c + ox) - x0) ** 2 + ((iy - c + oy) - y0) ** 2 <= r * r)
    return value * acc / (s * s)


def white_noise(N, seed):
    return np.random.default_rng(seed).standard_normal((N, N)).astype(np.float32)


def delta_image(N, iy0, ix0, value=1.0):
    img = np.zeros((N, N), dtype=np.float32)
    img[iy0, ix0] = value
    return img


def random_complex(shape, seed):
    rng = np.random.default_rng(seed)
    return (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)).astype(np.complex64)
