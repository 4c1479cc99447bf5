"""Seeded volume generators (numpy + scipy.ndimage only; float64 internally, cast to fp32 last).

Recipe (restated in DESIGN.md):
  field   : standard_normal(dims) -> gaussian_filter(sigma, mode='reflect') -> + blobs -> min-max to [0,1000]
  blobs   : soft-edged ellipsoids, centre uniform in the central 60 %, semi-axes U(0.06,0.15)*nx,
            amplitude +-U(1.5,3) field standard deviations, edge 1/(1+exp(8(rho-1)))
  mask    : sphere of the given radius about the volume centre ((n-1)/2 per axis), uint8
  shift   : moving(p) = fixed(clamp(p - s)) + noise          => fixed(p) <-> moving(p+s)
  rbf     : u = sum_8 v_k exp(-|x-c_k|^2 / 2 sigma_k^2), rescaled to max|u| = amplitude;
            moving(x) = trilinear(fixed, x - u(x)), edge-clamped + noise   => d ~ round(u(centre))
  noise   : Gaussian N(0,s) added, or Rician sqrt((I+n1)^2 + n2^2) with n1,n2 ~ N(0,s)
  seeds   : field = seed, noise = seed+1, warp = seed+2, blobs = seed+3

Arrays are indexed [z][y][x]; triples in the API are (x, y, z).
"""
from __future__ import annotations

from typing import Optional, Tuple

import numpy as np
from scipy import ndimage

from .configs import Config


def spherical_mask(dims, radius: float) -> np.ndarray:
    nx, ny, nz = dims
    z = np.arange(nz, dtype=np.float64)[:, None, None] - (nz - 1) / 2.0
    y = np.arange(ny, dtype=np.float64)[None, :, None] - (ny - 1) / 2.0
    x = np.arange(nx, dtype=np.float64)[None, None, :] - (nx - 1) / 2.0
    return ((x * x + y * y + z * z) <= radius * radius).astype(np.uint8)


def make_mask(cfg: Config) -> Optional[np.ndarray]:
    if cfg.mask_radius is None:
        return None
    return spherical_mask(cfg.dims, cfg.mask_radius)


def _blobs(dims, n_blobs: int, field_sd: float, seed: int) -> np.ndarray:
    nx, ny, nz = dims
    rng = np.random.default_rng(seed)
    out = np.zeros((nz, ny, nx), dtype=np.float64)
    z = np.arange(nz, dtype=np.float64)[:, None, None]
    y = np.arange(ny, dtype=np.float64)[None, :, None]
    x = np.arange(nx, dtype=np.float64)[None, None, :]
    for _ in range(n_blobs):
        c = np.array([rng.uniform(0.2, 0.8) * (n - 1) for n in (nx, ny, nz)])
        ax = rng.uniform(0.06, 0.15, size=3) * nx
        ax[2] = min(ax[2], 0.45 * nz)
        amp = rng.uniform(1.5, 3.0) * field_sd * (1.0 if rng.uniform() < 0.5 else -1.0)
        rho = np.sqrt(((x - c[0]) / ax[0]) ** 2 + ((y - c[1]) / ax[1]) ** 2 + ((z - c[2]) / ax[2]) ** 2)
        out += amp / (1.0 + np.exp(np.clip(8.0 * (rho - 1.0), -60.0, 60.0)))
    return out


def make_fixed(cfg: Config) -> np.ndarray:
    """The pre-operative ("fixed") volume as float64 in [0, 1000], shape [nz][ny][nx]."""
    nx, ny, nz = cfg.dims
    rng = np.random.default_rng(cfg.seed)
    f = rng.standard_normal((nz, ny, nx))
    f = ndimage.gaussian_filter(f, cfg.sigma, mode="reflect")
    if cfg.n_blobs:
        f = f + _blobs(cfg.dims, cfg.n_blobs, float(f.std()), cfg.seed + 3)
    lo, hi = float(f.min()), float(f.max())
    return (f - lo) * (1000.0 / (hi - lo))


def _rbf_field(dims, amplitude: float, seed: int):
    """Displacement u(x) as three float64 arrays (ux, uy, uz), each [nz][ny][nx]."""
    nx, ny, nz = dims
    rng = np.random.default_rng(seed)
    z = np.arange(nz, dtype=np.float64)[:, None, None]
    y = np.arange(ny, dtype=np.float64)[None, :, None]
    x = np.arange(nx, dtype=np.float64)[None, None, :]
    ux = np.zeros((nz, ny, nx)); uy = np.zeros((nz, ny, nx)); uz = np.zeros((nz, ny, nx))
    for _ in range(8):
        v = rng.standard_normal(3)
        v /= np.linalg.norm(v)
        s = rng.uniform(0.08, 0.2) * nx
        c = np.array([rng.uniform(0.15, 0.85) * (n - 1) for n in (nx, ny, nz)])
        g = np.exp(-(((x - c[0]) ** 2 + (y - c[1]) ** 2 + (z - c[2]) ** 2) / (2.0 * s * s)))
        ux += v[0] * g; uy += v[1] * g; uz += v[2] * g
    m = float(np.sqrt(ux * ux + uy * uy + uz * uz).max())
    k = amplitude / m
    return ux * k, uy * k, uz * k


def _add_noise(vol: np.ndarray, kind: str, sigma: float, seed: int) -> np.ndarray:
    if kind == "none" or sigma == 0.0:
        return vol
    rng = np.random.default_rng(seed)
    if kind == "gauss":
        return vol + rng.normal(0.0, sigma, size=vol.shape)
    if kind == "rician":
        n1 = rng.normal(0.0, sigma, size=vol.shape)
        n2 = rng.normal(0.0, sigma, size=vol.shape)
        return np.sqrt((vol + n1) ** 2 + n2 ** 2)
    raise ValueError(kind)


def make_pair(cfg: Config, return_field: bool = False):
    """Returns (fixed fp32, moving fp32, mask uint8 | None) [+ (ux,uy,uz) float64 if asked]."""
    fixed = make_fixed(cfg)
    nx, ny, nz = cfg.dims
    field = None
    if cfg.moving == "shift":
        sx, sy, sz = cfg.shift
        iz = np.clip(np.arange(nz) - sz, 0, nz - 1)
        iy = np.clip(np.arange(ny) - sy, 0, ny - 1)
        ix = np.clip(np.arange(nx) - sx, 0, nx - 1)
        moving = fixed[np.ix_(iz, iy, ix)]
        if return_field:
            field = tuple(np.full(fixed.shape, float(s)) for s in (sx, sy, sz))
    elif cfg.moving == "rbf":
        ux, uy, uz = _rbf_field(cfg.dims, cfg.rbf_amplitude, cfg.seed + 2)
        moving = np.empty_like(fixed)
        zz = np.arange(nz, dtype=np.float64)
        yy = np.arange(ny, dtype=np.float64)[:, None]
        xx = np.arange(nx, dtype=np.float64)[None, :]
        for k in range(nz):  # slab by slab to bound memory at 512x512x176
            coords = np.stack([zz[k] - uz[k], np.broadcast_to(yy, (ny, nx)) - uy[k],
                               np.broadcast_to(xx, (ny, nx)) - ux[k]])
            moving[k] = ndimage.map_coordinates(fixed, coords, order=1, mode="nearest")
        if return_field:
            field = (ux, uy, uz)
    else:
        raise ValueError(cfg.moving)
    moving = _add_noise(moving, cfg.noise, cfg.noise_sigma, cfg.seed + 1)
    out = (np.ascontiguousarray(fixed, dtype=np.float32),
           np.ascontiguousarray(moving, dtype=np.float32),
           make_mask(cfg))
    if return_field:
        return out + (field,)
    return out
