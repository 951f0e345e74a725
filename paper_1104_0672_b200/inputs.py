"""Seeded synthetic inputs: maps and radial-profile tables.  No arithmetic of the method lives here.

This is the one module both the oracle-side tests and the CUDA-side tests/bench draw inputs from
(it imports neither).  The maps stand in for the paper's Planck-HFI simulations and CMB realisations
(PAPER.md:195, 209-219), which are not available; the recipe is SURVEY.md section 8d / DESIGN.md:

    seed = 11040672 + 100 * cfg + map_index,   numpy.random.default_rng(seed).standard_normal  (fp64),
    cast to the config's dtype; config 4 adds 1000 point sources of amplitude 100 at pixel indices
    drawn uniformly with default_rng(11040672 + 499).

Profile tables are K(theta_t), theta_t = t * theta_max / (n - 1), t = 0 .. n-1 (endpoints included),
n = 65536 in BASELINE.json's configs.
"""
from __future__ import annotations

import math

import numpy as np

BASE_SEED = 11040672
ARCMIN = math.pi / (180.0 * 60.0)
DEG = math.pi / 180.0
FWHM_TO_SIGMA = 1.0 / 2.3548          # BASELINE.json configs[0]: sigma = FWHM / 2.3548
NTABLE = 65536


def white_noise(npix: int, cfg: int, map_index: int = 0, dtype=np.float32) -> np.ndarray:
    rng = np.random.default_rng(BASE_SEED + 100 * cfg + map_index)
    return rng.standard_normal(npix).astype(dtype)


def white_noise_maps(npix: int, cfg: int, nmaps: int, dtype=np.float32) -> np.ndarray:
    return np.stack([white_noise(npix, cfg, k, dtype) for k in range(nmaps)])


def add_point_sources(m: np.ndarray, nsrc: int = 1000, amplitude: float = 100.0,
                      seed: int = BASE_SEED + 499) -> np.ndarray:
    """Config 4: sources at uniformly drawn pixel indices (equal-area pixels); collisions add."""
    rng = np.random.default_rng(seed)
    idx = rng.integers(0, m.shape[-1], size=nsrc)
    out = m.copy()
    np.add.at(out, (..., idx), np.asarray(amplitude, dtype=m.dtype))
    return out


def table_thetas(theta_max: float, n: int = NTABLE) -> np.ndarray:
    return np.arange(n, dtype=np.float64) * (theta_max / (n - 1))


def gaussian_table(fwhm: float, theta_max: float, n: int = NTABLE) -> np.ndarray:
    """K(theta) = exp(-theta^2 / (2 sigma^2)), peak 1."""
    sigma = fwhm * FWHM_TO_SIGMA
    t = table_thetas(theta_max, n)
    return np.exp(-0.5 * (t / sigma) ** 2)


def tophat_table(theta_max: float, n: int = NTABLE) -> np.ndarray:
    """K = 1 on the whole table; the disc edge is the support test gamma < theta_max."""
    return np.ones(n)


def mexican_hat_table(s: float, theta_max: float, n: int = NTABLE) -> np.ndarray:
    """K(theta) = (2 - theta^2/s^2) exp(-theta^2 / (2 s^2)), no prefactor."""
    t = table_thetas(theta_max, n)
    return (2.0 - (t / s) ** 2) * np.exp(-0.5 * (t / s) ** 2)


def config(cfg: int) -> dict:
    """The five workloads of BASELINE.json, as plain parameters (no geometry, no arithmetic)."""
    if cfg == 1:
        fwhm = 5.0 * DEG
        return dict(cfg=1, pix=("ecp", 64, 128), fwhm=fwhm, theta_max=3.0 * fwhm * FWHM_TO_SIGMA,
                    kernel="gaussian", nmaps=1)
    if cfg == 2:
        fwhm = 30.0 * ARCMIN
        return dict(cfg=2, pix=("ecp", 1024, 2048), fwhm=fwhm, theta_max=2.5 * fwhm, kernel="gaussian", nmaps=1)
    if cfg == 3:
        fwhm = 10.0 * ARCMIN
        return dict(cfg=3, pix=("healpix", 512), fwhm=fwhm, theta_max=3.0 * fwhm, kernel="gaussian", nmaps=1)
    if cfg == 4:
        fwhm = 5.0 * ARCMIN
        return dict(cfg=4, pix=("healpix", 2048), fwhm=fwhm, theta_max=3.0 * fwhm, kernel="gaussian", nmaps=1,
                    point_sources=1000)
    if cfg == 5:
        return dict(cfg=5, pix=("healpix", 2048), nmaps=16,
                    kernels=[dict(kernel="tophat", theta_max=10.0 * ARCMIN),
                             dict(kernel="mexican_hat", s=4.0 * ARCMIN, theta_max=20.0 * ARCMIN)])
    raise ValueError("cfg must be 1..5")


def kernel_table(spec: dict, n: int = NTABLE) -> np.ndarray:
    k = spec["kernel"]
    if k == "gaussian":
        return gaussian_table(spec["fwhm"], spec["theta_max"], n)
    if k == "tophat":
        return tophat_table(spec["theta_max"], n)
    if k == "mexican_hat":
        return mexican_hat_table(spec["s"], spec["theta_max"], n)
    raise ValueError(k)
