"""Synthetic PSF images for the BASELINE.json configs (inputs only).

The paper's PSFs are 41x41 SDSS images; these are the analytic stand-ins
BASELINE.json names: a circular Gaussian (C0) and a circular Moffat (C1-C4),
sampled at pixel centres on a KxK grid centred on pixel (K-1)/2 and normalised to
unit sum.  Built in float64, cast to float32 once by the caller.
"""
from __future__ import annotations

import numpy as np


def _r2(K: int) -> np.ndarray:
    assert K % 2 == 1
    h = (K - 1) // 2
    a = np.arange(K, dtype=np.float64) - h
    return a[:, None] ** 2 + a[None, :] ** 2


def gaussian_psf(K: int, fwhm: float) -> np.ndarray:
    sigma = fwhm / (2.0 * np.sqrt(2.0 * np.log(2.0)))
    p = np.exp(-_r2(K) / (2.0 * sigma * sigma))
    return p / p.sum()


def moffat_psf(K: int, fwhm: float, beta: float) -> np.ndarray:
    rd = fwhm / (2.0 * np.sqrt(2.0 ** (1.0 / beta) - 1.0))
    p = (1.0 + _r2(K) / (rd * rd)) ** (-beta)
    return p / p.sum()


def asymmetric_psf(K: int, seed: int = 7) -> np.ndarray:
    """Positive, normalised, deliberately non-symmetric PSF (a lopsided Moffat
    plus seeded speckle) so that a flipped or transposed kernel fails parity."""
    rng = np.random.default_rng(seed)
    h = (K - 1) // 2
    a = np.arange(K, dtype=np.float64) - h
    yy, xx = np.meshgrid(a, a, indexing="ij")
    p = (1.0 + ((xx - 0.7) ** 2 + 1.8 * (yy + 0.4) ** 2 + 0.6 * xx * yy) / 6.0) ** (-2.5)
    p *= 1.0 + 0.3 * rng.random((K, K))
    return p / p.sum()
