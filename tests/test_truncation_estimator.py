"""Truncation-error estimate of the library (Eq. 2 / Eq. 7; include/arkcos.h) against
oracle/legendre.py.  Host-side functions: no GPU needed except for the last test."""
import numpy as np
import pytest

from oracle import legendre
from paper_1104_0672_b200 import arkcos, inputs

DEG = inputs.DEG
TOL = 1e-7          # relative to max |K_l|: the two sides integrate the same piecewise-linear profile with different rules


def profiles():
    tmax = 12 * DEG
    return {"gaussian": (inputs.gaussian_table(6 * DEG, tmax, 1025), tmax),
            "mexican_hat": (inputs.mexican_hat_table(3 * DEG, tmax, 1025), tmax),
            "disc": (inputs.tophat_table(tmax, 257), tmax),
            "coarse": (inputs.gaussian_table(6 * DEG, tmax, 5), tmax)}


@pytest.mark.parametrize("name", ["gaussian", "mexican_hat", "disc", "coarse"])
def test_legendre_transform_equals_oracle(name):
    tab, tmax = profiles()[name]
    lmax = 256
    for lo, hi in [(0.0, tmax), (5 * DEG, 9 * DEG), (0.31 * tmax, tmax)]:
        got = arkcos.arkcos_kernel_legendre(tab, tmax, lmax, lo, hi)
        ref = legendre.kernel_legendre(tab, tmax, lmax, lo, hi)
        assert np.abs(got - ref).max() <= TOL * np.abs(ref).max()


def test_truncation_error_equals_oracle():
    tab, tmax = profiles()["mexican_hat"]
    cl = 1.0 / (1.0 + np.arange(301.0)) ** 2
    for cut in [0.0, 4.4 * DEG, 7.3 * DEG, tmax, 2 * tmax]:
        s2, sig = arkcos.arkcos_kernel_truncation_error(tab, tmax, cut, cl)
        r2, rsig = legendre.truncation_error(tab, tmax, cut, cl)
        assert abs(sig - rsig) <= TOL * rsig
        assert abs(s2 - r2) <= TOL * rsig
    assert arkcos.arkcos_kernel_truncation_error(tab, tmax, tmax, cl)[0] == 0.0


def test_choose_cut_is_the_smallest_passing_candidate():
    tab, tmax = profiles()["gaussian"]
    cl = np.ones(200)
    ngrid = 64
    for tol in [1e-1, 1e-2, 1e-3]:
        cut, s2, sig = arkcos.arkcos_kernel_choose_cut(tab, tmax, cl, tol, ngrid)
        g = round(cut / tmax * ngrid)
        assert abs(cut - g * tmax / ngrid) < 1e-15 and 0 < g < ngrid
        r2, rsig = legendre.truncation_error(tab, tmax, cut, cl)
        assert abs(s2 - r2) <= TOL * rsig and r2 <= tol ** 2 * rsig
        r2_in, _ = legendre.truncation_error(tab, tmax, (g - 1) * tmax / ngrid, cl)
        assert r2_in > tol ** 2 * rsig
    # a looser tolerance never asks for a larger support
    cuts = [arkcos.arkcos_kernel_choose_cut(tab, tmax, cl, t, ngrid)[0] for t in (1e-3, 1e-2, 1e-1)]
    assert cuts[0] >= cuts[1] >= cuts[2]
    # nothing can be dropped at tolerance zero
    assert arkcos.arkcos_kernel_choose_cut(tab, tmax, cl, 0.0, ngrid)[0] == tmax


def test_choose_ell_nyquist_tail_property():
    tab, tmax = profiles()["gaussian"]
    lmax = 400
    cl = np.ones(lmax + 1)
    Kl = legendre.kernel_legendre(tab, tmax, lmax)
    ell = np.arange(lmax + 1)
    p = (2 * ell + 1) / (4 * np.pi) * Kl ** 2 * cl
    for tol in [1e-2, 1e-3]:
        L = int(arkcos.arkcos_kernel_choose_ell_nyquist(tab, tmax, cl, tol))
        assert 0 < L < lmax
        assert p[L + 1:].sum() <= tol ** 2 * p.sum() < p[L:].sum()


def test_estimator_argument_checks():
    tab, tmax = profiles()["disc"]
    cl = np.ones(10)
    with pytest.raises(arkcos.ArkcosError):
        arkcos.arkcos_kernel_legendre(tab, tmax, -1)
    with pytest.raises(arkcos.ArkcosError):
        arkcos.arkcos_kernel_legendre(tab, tmax, 8, 0.5 * tmax, 0.25 * tmax)
    with pytest.raises(arkcos.ArkcosError):
        arkcos.arkcos_kernel_legendre(tab[:1], tmax, 8)
    with pytest.raises(arkcos.ArkcosError):
        arkcos.arkcos_kernel_choose_cut(tab, tmax, cl, 1e-3, 0)
    with pytest.raises(arkcos.ArkcosError):
        arkcos.arkcos_kernel_truncation_error(tab, tmax, -1.0, cl)


@pytest.mark.gpu
def test_chosen_cut_carries_the_predicted_error_on_the_gpu():
    """Eq. 7 end to end: cut the profile where arkcos_kernel_choose_cut says, convolve white noise (C_l = Omega_pix) with the
    whole and with the cut profile on the GPU; the fractional RMS difference is sqrt(sigma2 / signal2) within sampling noise."""
    import torch
    nside = 256
    npix = 12 * nside * nside
    fwhm = 80 * inputs.ARCMIN          # sigma = 2.5 pixels: the annulus that is cut away is sampled by many pixels
    tmax = 3.5 * fwhm * inputs.FWHM_TO_SIGMA
    n, ngrid = 4097, 64
    tab = inputs.gaussian_table(fwhm, tmax, n)
    lmax = 64 * nside                  # pixel white noise is not band-limited, and the annulus that is cut away has sharp edges:
    cl = np.full(lmax + 1, 4 * np.pi / npix)     # dK_l^2 (2l+1) falls off as 1/l^2 only, the sum needs l far beyond the pixel scale
    cut, s2, sig = arkcos.arkcos_kernel_choose_cut(tab, tmax, cl, 3e-3, ngrid)
    g = round(cut / tmax * ngrid)
    assert 0 < g < ngrid
    ncut = g * (n - 1) // ngrid + 1
    x = torch.from_numpy(inputs.white_noise(npix, 9)).cuda()
    full = arkcos.convolve_torch(arkcos.Plan(("healpix", nside), tab, tmax, arkcos.F32), x).double()
    part = arkcos.convolve_torch(arkcos.Plan(("healpix", nside), tab[:ncut], cut, arkcos.F32), x).double()
    measured = float(((full - part) ** 2).sum() / (full ** 2).sum())
    print('measured', measured, 'predicted', s2 / sig)
    assert measured <= (3e-3) ** 2 * 1.3
    assert abs(measured / (s2 / sig) - 1) < 0.12, (measured, s2 / sig)
