"""Oracle for the truncation-error estimate: Legendre transform of a radial profile (Eq. 2) and Eq. 7.

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).  fp64, slow, written to be read against the paper.

Eq. 2:    K_l = 2 pi int_{-1}^{1} K(z) P_l(z) dz,            z = cos(theta)
Eq. 7:   sigma^2 = sum_{l=0}^{lmax} (2l+1)/(4 pi) dK_l^2 C_l

"where dK_l is the Legendre expansion of the difference of the exact and the truncated kernel":
the exact kernel is the tabulated profile on its whole support [0, theta_max), the truncated one is the same
profile cut at alpha_cut, so the difference is the profile on [alpha_cut, theta_max) and zero
elsewhere (reading R19).  The profile between table nodes is the linear interpolant in theta that the
convolution itself uses (oracle/direct.py kernel_lerp).

The integral is written as the plain definition in theta,  K_l = 2 pi int K(theta) P_l(cos theta) sin(theta) dtheta,
evaluated by a composite Gauss-Legendre rule (numpy leggauss nodes, scipy eval_legendre values) on panels short
against the oscillation length pi / l of P_l that end at the table nodes; no recurrences, no blocking.
"""
from __future__ import annotations

import numpy as np
from scipy.special import eval_legendre

from .direct import kernel_lerp

_GL_ORDER = 8


def _panels(theta_lo: float, theta_hi: float, lmax: int, ntab: int, theta_max: float) -> np.ndarray:
    """Panel edges on [theta_lo, theta_hi]: at most a quarter of P_lmax's oscillation length each, and every table node
    in between is an edge (the interpolant's slope jumps there; a Gauss rule across a kink converges slowly)."""
    width = min(0.25 * np.pi / (lmax + 1), (theta_hi - theta_lo))
    npan = max(1, int(np.ceil((theta_hi - theta_lo) / width)))
    nodes = np.arange(ntab) * (theta_max / (ntab - 1))
    nodes = nodes[(nodes > theta_lo) & (nodes < theta_hi)]
    return np.unique(np.concatenate([np.linspace(theta_lo, theta_hi, npan + 1), nodes]))


def kernel_legendre(table: np.ndarray, theta_max: float, lmax: int, theta_lo: float = 0.0,
                    theta_hi: float | None = None) -> np.ndarray:
    """K_l, l = 0 .. lmax, of the profile restricted to theta_lo <= theta < theta_hi (Eq. 2)."""
    theta_hi = theta_max if theta_hi is None else theta_hi
    out = np.zeros(lmax + 1)
    if not theta_hi > theta_lo:
        return out
    x, w = np.polynomial.legendre.leggauss(_GL_ORDER)
    edges = _panels(theta_lo, theta_hi, lmax, table.shape[0], theta_max)
    a, b = edges[:-1, None], edges[1:, None]
    theta = (0.5 * (a + b) + 0.5 * (b - a) * x[None, :]).ravel()
    weight = (0.5 * (b - a) * w[None, :]).ravel()
    K = kernel_lerp(table, theta_max, theta)
    f = K * np.sin(theta) * weight
    z = np.cos(theta)
    for ell in range(lmax + 1):
        out[ell] = 2.0 * np.pi * np.sum(f * eval_legendre(ell, z))
    return out


def truncation_error(table: np.ndarray, theta_max: float, theta_cut: float, c_ell: np.ndarray) -> tuple[float, float]:
    """(sigma^2, signal^2): Eq. 7 for the cut at theta_cut, and the same sum with the whole kernel's K_l
    (the variance of the exactly convolved map), both up to lmax = len(c_ell) - 1."""
    c_ell = np.asarray(c_ell, dtype=np.float64)
    lmax = c_ell.shape[0] - 1
    ell = np.arange(lmax + 1)
    dK = kernel_legendre(table, theta_max, lmax, theta_lo=min(theta_cut, theta_max), theta_hi=theta_max)
    Kl = kernel_legendre(table, theta_max, lmax)
    w = (2 * ell + 1) / (4.0 * np.pi) * c_ell
    return float(np.sum(w * dK ** 2)), float(np.sum(w * Kl ** 2))
