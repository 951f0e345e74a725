"""CPU tests of the library's host logic (no compute calls): the C ABI loads and exports every symbol the header
declares, argument checking, and the plan's geometry / band / M' tables against the oracle's independent restatement."""
import os
import re

import numpy as np
import pytest

from oracle import geometry, hybrid
from paper_1104_0672_b200 import arkcos, inputs
from plan_checks import plan_mprime

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_header_symbols_exported():
    hdr = open(os.path.join(ROOT, "include", "arkcos.h")).read()
    declared = set(re.findall(r"\b(arkcos_[a-z0-9_]+)\s*\(", hdr))
    assert declared, "no declarations found"
    lib = arkcos._lib()
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in arkcos.h but not exported"
    assert declared == set(arkcos.SYMBOLS), declared ^ set(arkcos.SYMBOLS)


def test_launches_per_convolve():
    """Kernel-row generator + ring FFT launches per size class and direction + band kernels of the classes present."""
    tab = inputs.gaussian_table(5 * inputs.ARCMIN, 15 * inputs.ARCMIN)
    p = arkcos.Plan(("healpix", 2048), tab, 15 * inputs.ARCMIN, tables_only=True)
    n = p.launches_per_convolve
    assert n == 26        # rows + 2 x (4 Bluestein size classes + 4 power-of-two classes + shortest rings) + 7 band launches (the pole kernel is two)
    assert arkcos.Plan(("healpix", 2048), tab, 15 * inputs.ARCMIN, cache_kernel_rows=1,
                       tables_only=True).launches_per_convolve == n - 1
    assert arkcos.Plan(("ecp", 64, 128), inputs.gaussian_table(0.1, 0.2, 64), 0.2, arkcos.F64,
                       tables_only=True).launches_per_convolve == 5      # rows, forward FFT, band (pole kernel: two launches), inverse FFT (fp64: shared-memory FFT)


def test_strerror_and_bad_args():
    assert arkcos.arkcos_strerror(0) == "success"
    assert "invalid" in arkcos.arkcos_strerror(arkcos.INVALID_ARG)
    tab = inputs.gaussian_table(0.1, 0.2, 64)
    for bad in [("ecp", 8, 24), ("ecp", 0, 16), ("healpix", 3), ("healpix", 8192)]:
        with pytest.raises(arkcos.ArkcosError) as e:
            arkcos.Plan(bad, tab, 0.2, tables_only=True)
        assert e.value.status == arkcos.INVALID_ARG
    with pytest.raises(arkcos.ArkcosError) as e:
        arkcos.Plan(("healpix", 4), tab, 0.2, variant=2, tables_only=True)
    assert e.value.status == arkcos.INVALID_ARG
    assert arkcos.Plan(("healpix", 4), tab, 0.2, variant=1, tables_only=True).nrings == 15     # the basic scheme
    with pytest.raises(arkcos.ArkcosError):
        arkcos.Plan(("healpix", 4), tab, -1.0, tables_only=True)
    p = arkcos.Plan(("healpix", 4), tab, 0.2, tables_only=True)
    with pytest.raises(arkcos.ArkcosError) as e:          # a tables-only plan cannot compute
        p.convolve(16, 4096, 1)
    assert e.value.status == arkcos.INVALID_ARG
    lib = arkcos._lib()
    assert lib.arkcos_plan_destroy(None) == 0
    assert lib.arkcos_plan_npix(None) == -1


@pytest.mark.parametrize("pix", [("ecp", 64, 128), ("healpix", 16), ("healpix", 64)])
def test_plan_geometry_matches_oracle(pix):
    geom = geometry.ecp(pix[1], pix[2]) if pix[0] == "ecp" else geometry.healpix_ring(pix[1])
    tmax = 0.11
    tab = inputs.gaussian_table(0.05, tmax, 1024)
    ell = 77.5
    p = arkcos.Plan(pix, tab, tmax, ell_nyquist=ell, tables_only=True)
    assert p.npix == geom.npix and p.nrings == geom.nrings
    assert p.ell_nyquist == (ell if pix[0] == "healpix" else 0.0)
    mp = plan_mprime(p, geom, tmax, ell) if pix[0] == "healpix" else None
    for i in range(geom.nrings):
        r = p.ring_info(i)
        assert abs(r["theta"] - geom.theta[i]) < 1e-15
        assert r["n"] == geom.n[i] and r["offset"] == geom.offset[i]
        assert abs(r["phi0"] - geom.phi0[i]) < 1e-16
        b = geometry.band(geom, i, tmax)
        assert (r["band_lo"], r["band_hi"]) == (b[0], b[-1]) and b.size == b[-1] - b[0] + 1
        if pix[0] == "healpix" and mp[i] >= 512:
            assert mp[i] % 128 == 0          # runs of cap rings share one grid length (reading R10)
    st = p.stats()
    assert st["ring_pairs"] == sum(geometry.band(geom, i, tmax).size for i in range(geom.nrings))
    assert st["row_samples"] > 0 and st["mac_flops"] > 0 and st["fft_flops"] > 0


def test_polar_oversample_and_auto_ell():
    nside = 64
    geom = geometry.healpix_ring(nside)
    pixsz = np.sqrt(4 * np.pi / geom.npix)
    fwhm = 2.91 * pixsz
    tmax = 3 * fwhm
    tab = inputs.gaussian_table(fwhm, tmax)
    p = arkcos.Plan(("healpix", nside), tab, tmax, polar_oversample=2, tables_only=True)
    assert all(p.ring_info(i)["mprime"] == 2 * 4 * nside for i in (0, 50, 200))
    # automatic choice: between 4.5/sigma and 6.5/sigma for a Gaussian (1e-7 spectral tail)
    q = arkcos.Plan(("healpix", nside), tab, tmax, tables_only=True)
    sigma = fwhm * inputs.FWHM_TO_SIGMA
    assert 4.5 / sigma < q.ell_nyquist < 6.5 / sigma
    # a disc never converges: the cap 8 nside is returned
    t = arkcos.Plan(("healpix", nside), inputs.tophat_table(tmax), tmax, tables_only=True)
    assert t.ell_nyquist == pytest.approx(8 * nside, rel=2e-3)
