"""Pins for oracle/geometry.py: what the paper and the mathematics fix."""
import numpy as np
import pytest

from oracle import geometry


@pytest.mark.parametrize("nside", [1, 2, 4, 16, 64])
def test_healpix_counts(nside):
    g = geometry.healpix_ring(nside)
    assert g.nrings == 4 * nside - 1                          # PAPER.md:125 "4 nside - 1 sets"
    assert g.npix == 12 * nside * nside
    # caps: nside-1 rings, ring n has 4 n pixels; equatorial: 2 nside + 1 rings of 4 nside
    assert list(g.n[: nside - 1]) == [4 * n for n in range(1, nside)]
    assert np.all(g.n[nside - 1: 3 * nside] == 4 * nside) and (3 * nside - (nside - 1)) == 2 * nside + 1
    assert list(g.n[3 * nside:]) == [4 * n for n in range(nside - 1, 0, -1)]
    assert g.offset[0] == 0 and np.all(np.diff(g.offset) == g.n)


@pytest.mark.parametrize("nside", [2, 8, 32])
def test_healpix_latitudes(nside):
    g = geometry.healpix_ring(nside)
    z = np.cos(g.theta)
    assert np.all(np.diff(g.theta) > 0)
    assert abs(z[nside - 1] - 2.0 / 3.0) < 1e-14              # cap formula and belt formula meet at z = 2/3
    assert abs(1 - nside ** 2 / (3.0 * nside ** 2) - 2.0 / 3.0) < 1e-15
    assert abs(z[2 * nside - 1]) < 1e-15                      # equator ring
    np.testing.assert_allclose(z, -z[::-1], atol=1e-15)       # north/south mirror
    np.testing.assert_array_equal(g.n, g.n[::-1])
    np.testing.assert_allclose(g.phi0, g.phi0[::-1], atol=0)
    # equal-area: sum_p Omega = 4 pi exactly; the quadrature of z^2 is 4 pi / 3 up to O(1/nside^2)
    assert abs((g.omega * g.n).sum() - 4 * np.pi) < 1e-12
    assert abs((g.omega * g.n * z ** 2).sum() / (4 * np.pi / 3) - 1) < 1.0 / nside ** 2


def test_healpix_phi0():
    nside = 4
    g = geometry.healpix_ring(nside)
    for idx in range(g.nrings):
        i = idx + 1
        if i < nside or i > 3 * nside:                        # every cap ring shifted by pi / (4 n)
            assert g.phi0[idx] == pytest.approx(np.pi / g.n[idx])
        else:                                                  # every other equatorial ring
            assert g.phi0[idx] == (pytest.approx(np.pi / (4 * nside)) if (i - nside) % 2 == 0 else 0.0)
    # half a pixel in every shifted ring
    shifted = g.phi0 > 0
    np.testing.assert_allclose(g.phi0[shifted], 0.5 * 2 * np.pi / g.n[shifted])


def test_healpix_nside1_pixel_centres():
    # nside = 1: the 12 base-pixel centres are z = 2/3, 0, -2/3 with phi = pi/4 + k pi/2 (rings 1, 3) and
    # k pi/2 (ring 2) -- the textbook picture of the HEALPix base tessellation.
    g = geometry.healpix_ring(1)
    np.testing.assert_allclose(np.cos(g.theta), [2 / 3, 0, -2 / 3], atol=1e-15)
    np.testing.assert_allclose(g.phi(0), np.pi / 4 + np.arange(4) * np.pi / 2)
    np.testing.assert_allclose(g.phi(1), np.arange(4) * np.pi / 2)


def test_ecp():
    g = geometry.ecp(64, 128)
    assert g.npix == 8192 and g.nrings == 64
    np.testing.assert_allclose(g.theta, (np.arange(64) + 0.5) * np.pi / 64)
    assert np.all(g.phi0 == 0) and np.all(g.n == 128)
    np.testing.assert_allclose(g.omega, np.sin(g.theta) * (np.pi / 64) * (2 * np.pi / 128))
    # midpoint rule for the area of the sphere: 4 pi (1 + O(1/Ntheta^2))
    assert abs((g.omega * g.n).sum() / (4 * np.pi) - 1) < 2e-4


def test_band_is_sufficient():
    # no pixel outside the band can be inside the cap: gamma >= |theta_i - theta_j|
    g = geometry.healpix_ring(4)
    from oracle.direct import unit_vectors
    v = unit_vectors(g)
    gamma = np.arccos(np.clip(v @ v.T, -1, 1))
    ring_of = np.repeat(np.arange(g.nrings), g.n)
    tmax = 0.4
    for i in range(g.nrings):
        b = set(geometry.band(g, i, tmax).tolist())
        rows = gamma[g.ring_slice(i)]
        reached = set(ring_of[np.nonzero((rows < tmax).any(axis=0))[0]].tolist())
        assert reached <= b


def test_golden_paper_counts():
    """The paper's own statements about the ring structure (tests/golden/healpix_counts_paper.txt)."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "healpix_counts_paper.txt")
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        nside, ncaps, nequ, nrings, ncoef, npix = map(int, line.split())
        g = geometry.healpix_ring(nside)
        assert ncaps == nside - 1 and nequ == 2 * nside + 1
        assert g.nrings == nrings == 2 * ncaps + nequ and g.npix == npix
        assert int((g.n == 4 * nside).sum()) == nequ and int(g.n.max()) // 2 + 1 == ncoef
        assert list(g.n[:ncaps]) == [4 * n for n in range(1, nside)]


def test_golden_point_source_regression():
    """Oracle #1 against the stored response written by tests/golden/make_golden.py (oracle-only script)."""
    import os
    from oracle import direct
    sys_path = os.path.join(os.path.dirname(__file__), "golden")
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(sys_path, "make_golden.py"))
    mg = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mg)
    g = geometry.healpix_ring(mg.NSIDE)
    x = np.zeros(g.npix)
    x[mg.Q0] = 1.0
    out = direct.direct_sum(g, mg.table(), mg.TMAX, x)
    data = np.loadtxt(os.path.join(sys_path, "point_source_hp8.txt"))
    ref = np.zeros(g.npix)
    ref[data[:, 0].astype(int)] = data[:, 1]
    np.testing.assert_allclose(out, ref, rtol=1e-13, atol=0)
