"""Pins for oracle/legendre.py (Eq. 2; Eq. 7) against things that are not the oracle:
textbook closed forms, completeness of the Legendre polynomials, and the brute-force sum on white noise."""
import numpy as np
import pytest
from scipy import special

from oracle import geometry, direct, legendre
from paper_1104_0672_b200 import inputs

DEG = inputs.DEG


def disc_legendre_closed_form(lmax, theta_lo, theta_hi):
    """2 pi int_{cos hi}^{cos lo} P_l dz = 2 pi [P_{l+1} - P_{l-1}](z) / (2l+1) between the limits; l = 0: 2 pi (z_lo - z_hi)."""
    zl, zh = np.cos(theta_lo), np.cos(theta_hi)
    out = np.empty(lmax + 1)
    out[0] = 2 * np.pi * (zl - zh)
    for l in range(1, lmax + 1):
        F = lambda z: (special.eval_legendre(l + 1, z) - special.eval_legendre(l - 1, z)) / (2 * l + 1)  # noqa: E731
        out[l] = 2 * np.pi * (F(zl) - F(zh))
    return out


@pytest.mark.parametrize("lo_hi", [(0.0, 12 * DEG), (5 * DEG, 12 * DEG)], ids=["disc", "annulus"])
def test_disc_closed_form(lo_hi):
    """All l at once: catches a dropped sin(theta), a wrong 2 pi, wrong limits of the restricted profile, too coarse panels."""
    lo, hi = lo_hi
    tab = inputs.tophat_table(12 * DEG, 4097)
    got = legendre.kernel_legendre(tab, 12 * DEG, 200, theta_lo=lo, theta_hi=hi)
    ref = disc_legendre_closed_form(200, lo, hi)
    assert np.abs(got - ref).max() <= 1e-12


def test_gaussian_flat_sky_limit():
    """Narrow Gaussian: K_l -> 2 pi sigma^2 exp(-l(l+1) sigma^2 / 2) (the beam window function); relative deviation
    O(sigma^2).  Catches a profile evaluated in the wrong variable (z instead of theta) or a wrong table spacing."""
    fwhm = 2.0 * DEG
    sigma = fwhm * inputs.FWHM_TO_SIGMA
    tmax = 6 * sigma
    tab = inputs.gaussian_table(fwhm, tmax, 2049)
    lmax = 150
    got = legendre.kernel_legendre(tab, tmax, lmax)
    ell = np.arange(lmax + 1)
    ref = 2 * np.pi * sigma ** 2 * np.exp(-0.5 * ell * (ell + 1) * sigma ** 2)
    sel = ref > 1e-3 * ref[0]
    assert np.abs(got[sel] / ref[sel] - 1).max() < 5e-3
    assert np.abs(got[0] / ref[0] - 1) < 5 * sigma ** 2


def test_completeness_parseval():
    """sum_l (2l+1)/(4 pi) K_l^2 -> 2 pi int K(z)^2 dz for lmax beyond the profile's band (smooth profile)."""
    s = 4 * DEG
    tmax = 6 * s
    tab = inputs.mexican_hat_table(s, tmax, 2049) * (1 - (inputs.table_thetas(tmax, 2049) / tmax) ** 2) ** 2    # smooth at the cut
    lmax = 160
    Kl = legendre.kernel_legendre(tab, tmax, lmax)
    ell = np.arange(lmax + 1)
    lhs = np.sum((2 * ell + 1) / (4 * np.pi) * Kl ** 2)
    th = np.linspace(0, tmax, 200001)
    f = direct.kernel_lerp(tab, tmax, th) ** 2 * np.sin(th)
    rhs = 2 * np.pi * np.sum(0.5 * (f[1:] + f[:-1]) * np.diff(th))
    assert abs(lhs / rhs - 1) < 1e-6


def test_eq7_white_noise_against_brute_force():
    """Eq. 7 read against an experiment: unit white noise per pixel has C_l = Omega_pix; the difference between the map
    smoothed with the whole profile and with the profile cut at theta_cut (both by the brute-force sum, oracle #1) must
    have the mean square Eq. 7 predicts.  Catches a wrong reading of 'difference of the exact and the truncated kernel',
    a missing (2l+1)/4pi, K_l off by a factor."""
    nside = 16
    geom = geometry.healpix_ring(nside)
    fwhm = 12 * DEG
    tmax = 3.0 * fwhm * inputs.FWHM_TO_SIGMA
    n = 4097
    ncut = 2561                        # the cut falls on a table node: both tables interpolate the same values
    tcut = (ncut - 1) * tmax / (n - 1)
    tab = inputs.gaussian_table(fwhm, tmax, n)
    x = np.random.default_rng(7).standard_normal((8, geom.npix))
    full = direct.direct_sum(geom, tab, tmax, x)
    # the cut profile as a table of its own on [0, tcut) (support test gamma < tcut)
    cut = direct.direct_sum(geom, tab[:ncut], tcut, x)
    measured = float(np.mean((full - cut) ** 2))
    omega = 4 * np.pi / geom.npix
    lmax = 16 * nside                  # pixel white noise is not band-limited: the sum runs until dK_l has died out
    sigma2, signal2 = legendre.truncation_error(tab, tmax, tcut, np.full(lmax + 1, omega))
    assert abs(sigma2 / measured - 1) < 0.08, (sigma2, measured)
    assert abs(signal2 / float(np.mean(full ** 2)) - 1) < 0.08


def test_truncation_error_limits():
    """theta_cut = theta_max: nothing is cut, sigma^2 = 0; theta_cut = 0: everything is, sigma^2 = signal^2."""
    tmax = 10 * DEG
    tab = inputs.gaussian_table(5 * DEG, tmax, 2049)
    cl = 1.0 / (1.0 + np.arange(65)) ** 2
    s2, sig2 = legendre.truncation_error(tab, tmax, tmax, cl)
    assert s2 == 0.0 and sig2 > 0
    s2, sig2 = legendre.truncation_error(tab, tmax, 0.0, cl)
    assert abs(s2 / sig2 - 1) < 1e-12
