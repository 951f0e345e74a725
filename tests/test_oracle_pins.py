"""Pins for the two oracles (oracle/direct.py, oracle/hybrid.py) against things that are not the oracle:
closed forms, exact identities, an independent restatement, brute force on tiny grids.
SURVEY.md section 8c "What pins each part" lists them; each test names the plausible mistake it catches.
"""
import numpy as np
import pytest
from scipy import special

from oracle import geometry, direct, hybrid
from paper_1104_0672_b200 import inputs

DEG = inputs.DEG


def frms(a, b):
    return float(np.sqrt(((a - b) ** 2).sum() / (b ** 2).sum()))


def gauss(fwhm, theta_max, n=65536):
    return inputs.gaussian_table(fwhm, theta_max, n)


# ---------------------------------------------------------------- oracle #1 ----------------------------------

@pytest.mark.parametrize("geom", [geometry.ecp(12, 24), geometry.healpix_ring(4), geometry.healpix_ring(7)],
                         ids=["ecp", "hp4", "hp7"])
def test_direct_c_equals_arccos_restatement(geom):
    """C routine (haversine form of Eq. 9) vs numpy arccos(n_p . n_q): catches a wrong A/B term, a wrong
    window, a dropped Omega, an off-by-one in the table lerp."""
    tmax = 35 * DEG
    tab = inputs.mexican_hat_table(10 * DEG, tmax)         # non-monotonic profile with a sign change
    x = np.random.default_rng(3).standard_normal((2, geom.npix))
    a = direct.direct_sum(geom, tab, tmax, x)
    b = direct.direct_sum_numpy(geom, tab, tmax, x)
    assert np.abs(a - b).max() <= 1e-11 * np.abs(b).max()


@pytest.mark.parametrize("kind", ["ecp", "healpix"])
def test_point_source_response(kind):
    """in = delta_q0  =>  out(p) = K(gamma_p,q0) Omega_q0 [gamma < theta_max]  (definition, normalisation,
    Omega on the *input* pixel, strict support)."""
    geom = geometry.ecp(16, 32) if kind == "ecp" else geometry.healpix_ring(8)
    fwhm, tmax = 15 * DEG, 30 * DEG
    sigma = fwhm * inputs.FWHM_TO_SIGMA
    tab = gauss(fwhm, tmax)
    v = direct.unit_vectors(geom)
    ring_of = np.repeat(np.arange(geom.nrings), geom.n)
    for q0 in (0, geom.npix // 3, geom.npix - 5):
        x = np.zeros(geom.npix)
        x[q0] = 1.0
        out = direct.direct_sum(geom, tab, tmax, x)
        gam = np.arccos(np.clip(v @ v[q0], -1, 1))
        expect = np.where(gam < tmax, np.exp(-0.5 * (gam / sigma) ** 2), 0.0) * geom.omega[ring_of[q0]]
        # 65536-point lerp of a Gaussian: relative table error <= (dtheta/sigma)^2/8 ~ 1e-9
        assert np.abs(out - expect).max() <= 3e-9 * expect.max()
        assert np.array_equal(out != 0, gam < tmax) or np.abs(gam[(out != 0) != (gam < tmax)] - tmax).max() < 1e-12


def test_direct_ring_subset_and_threads():
    geom = geometry.healpix_ring(4)
    tmax = 30 * DEG
    tab = gauss(20 * DEG, tmax)
    x = np.random.default_rng(5).standard_normal(geom.npix)
    full = direct.direct_sum(geom, tab, tmax, x)
    rings = np.array([14, 0, 7])
    sub, nthr = direct.direct_sum(geom, tab, tmax, x, out_rings=rings, nthreads=1, return_threads=True)
    assert nthr == 1
    np.testing.assert_array_equal(sub, np.concatenate([full[geom.ring_slice(r)] for r in rings]))


def test_constant_map():
    """Constant in -> ring-wise constant out = sum_q K Omega_q (exact); ~ integral of K over the sphere to
    quadrature accuracy on a fine grid with a wide kernel (SURVEY.md 8c reading 19)."""
    geom = geometry.ecp(96, 192)
    fwhm = 20 * DEG
    tmax = 3.5 * fwhm * inputs.FWHM_TO_SIGMA
    sigma = fwhm * inputs.FWHM_TO_SIGMA
    tab = gauss(fwhm, tmax)
    out = direct.direct_sum(geom, tab, tmax, np.full(geom.npix, 2.5), out_rings=np.array([3, 40, 48, 90]))
    rows = np.split(out, np.cumsum([192] * 3))
    for r in rows:
        assert np.ptp(r) <= 1e-12 * abs(r.mean())
    # integral of the truncated Gaussian over the sphere: 2 pi int_0^tmax K(t) sin t dt (numerically, 1e-10)
    t = np.linspace(0, tmax, 200001)
    f = np.exp(-0.5 * (t / sigma) ** 2) * np.sin(t)
    integral = 2 * np.pi * (f.sum() - 0.5 * (f[0] + f[-1])) * (t[1] - t[0])
    assert abs(rows[1].mean() / (2.5 * integral) - 1) < 2e-3       # mid-latitude ring
    assert abs(rows[2].mean() / (2.5 * integral) - 1) < 2e-3


def test_self_adjoint_and_mirror():
    """sum_p Omega_p g_p (K f)_p = sum_q Omega_q f_q (K g)_q (symmetric kernel); mirror symmetry of the sphere."""
    geom = geometry.healpix_ring(6)
    tmax = 25 * DEG
    tab = inputs.mexican_hat_table(7 * DEG, tmax)
    rng = np.random.default_rng(11)
    f, g = rng.standard_normal((2, geom.npix))
    Kf = direct.direct_sum(geom, tab, tmax, f)
    Kg = direct.direct_sum(geom, tab, tmax, g)
    om = np.repeat(geom.omega, geom.n)
    assert abs((om * g * Kf).sum() - (om * f * Kg).sum()) < 1e-13 * np.abs(om * g * Kf).sum()

    def mirror(m):      # theta -> pi - theta keeps phi: reverse the ring order, keep the order inside a ring
        return np.concatenate([m[geom.ring_slice(i)] for i in range(geom.nrings - 1, -1, -1)])
    np.testing.assert_allclose(direct.direct_sum(geom, tab, tmax, mirror(f)), mirror(Kf), rtol=0, atol=1e-13)


# ---------------------------------------------------------------- oracle #2 ----------------------------------

def test_dft_definition():
    """The DFT step: delta, constant, Parseval, and the library FFT used above DIRECT_DFT_MAX."""
    rng = np.random.default_rng(0)
    for N in (4, 12, 20, 97, 128):
        x = rng.standard_normal(N) + 1j * rng.standard_normal(N)
        X = hybrid.dft(x)
        np.testing.assert_allclose(X, np.fft.fft(x), atol=1e-11)
        np.testing.assert_allclose(hybrid.dft(X, +1) / N, x, atol=1e-12)
        assert abs((np.abs(X) ** 2).sum() - N * (np.abs(x) ** 2).sum()) < 1e-9
        e = np.zeros(N)
        e[1] = 1
        np.testing.assert_allclose(hybrid.dft(e), np.exp(-2j * np.pi * np.arange(N) / N), atol=1e-14)
    old = hybrid.DIRECT_DFT_MAX
    try:
        hybrid.DIRECT_DFT_MAX = 8
        np.testing.assert_allclose(hybrid.dft(x), X, atol=1e-11)
    finally:
        hybrid.DIRECT_DFT_MAX = old


def test_eq9_identity():
    """Eq. 9's right-hand side is 2 - 2 cos(gamma) exactly (spherical law of cosines)."""
    rng = np.random.default_rng(2)
    ti, tj = rng.uniform(0, np.pi, 2)
    psi = rng.uniform(-np.pi, np.pi, 50)
    cosg = np.cos(ti) * np.cos(tj) + np.sin(ti) * np.sin(tj) * np.cos(psi)
    np.testing.assert_allclose(hybrid.squared_chord(ti, tj, psi), 2 - 2 * cosg, atol=1e-14)
    # and literally as printed
    s2p, s2m = np.sin(0.5 * (ti + tj)) ** 2, np.sin(0.5 * (ti - tj)) ** 2
    np.testing.assert_allclose(2 * (s2p + s2m) - 2 * (s2p - s2m) * np.cos(psi), 2 - 2 * cosg, atol=1e-14)


def test_kernel_row_closed_form_bessel():
    """Jacobi-Anger: for K = exp(-x / (2 s^2)), x the squared chord, the row's Fourier coefficients are
    exp(-a/(2 s^2)) I_m(b/(2 s^2)), a = 2(1 - cos ti cos tj), b = 2 sin ti sin tj.  Pins the row generator and
    its transform (sign/normalisation of the DFT, the A/B split of Eq. 9, transposed theta_i/theta_j)."""
    ti, tj, s, M = 50 * DEG, 58 * DEG, 15 * DEG, 128
    # a table of exp(-x/(2 s^2)) as a function of theta: x = 4 sin^2(theta/2); support = whole sphere
    tmax = np.pi
    th = inputs.table_thetas(tmax, 1 << 20)
    tab = np.exp(-4 * np.sin(0.5 * th) ** 2 / (2 * s * s))
    row = hybrid.kernel_row(ti, tj, 2 * np.pi * np.arange(M) / M, tab, tmax * (1 + 1e-12))
    kt = hybrid.dft(row.astype(complex)) / M
    a, b = 2 * (1 - np.cos(ti) * np.cos(tj)), 2 * np.sin(ti) * np.sin(tj)
    m = np.arange(0, 20)
    z = b / (2 * s * s)
    expect = np.exp(-a / (2 * s * s) + z) * special.ive(m, z)
    assert np.abs(kt[m].real - expect).max() < 1e-10 * expect.max()
    assert np.abs(kt.imag).max() < 1e-15


@pytest.mark.parametrize("cfg1", [True, False])
def test_ecp_hybrid_equals_direct(cfg1):
    """On ECP the ring formulation is an exact circulant identity: #2 == #1 to 1e-13."""
    if cfg1:
        c = inputs.config(1)
        geom, tmax, tab = geometry.ecp(64, 128), c["theta_max"], inputs.kernel_table(c)
        rings = np.array([0, 1, 17, 31, 32, 63])
    else:
        geom, tmax = geometry.ecp(24, 40), 20 * DEG           # non power-of-two ring length, hard-edged kernel
        tab = inputs.tophat_table(tmax)
        rings = np.arange(24)
    x = inputs.white_noise(geom.npix, 1, dtype=np.float64)
    a = direct.direct_sum(geom, tab, tmax, x, out_rings=rings)
    b = hybrid.hybrid_convolve(geom, tab, tmax, x, out_rings=rings)
    assert np.abs(a - b).max() <= 1e-13 * np.abs(a).max()


def test_healpix_equatorial_band_exact():
    """Output rings whose whole band lies in the equatorial region: offset-aware sampling is exact."""
    nside = 8
    geom = geometry.healpix_ring(nside)
    tmax = 14 * DEG
    tab = inputs.tophat_table(tmax)                           # worst case for any interpolation: a disc
    x = np.random.default_rng(8).standard_normal(geom.npix)
    rings = np.array([i for i in range(geom.nrings)
                      if np.all(geom.n[geometry.band(geom, i, tmax)] == 4 * nside)])
    assert rings.size >= 5 and any(geom.phi0[r] > 0 for r in rings) and any(geom.phi0[r] == 0 for r in rings)
    a = direct.direct_sum(geom, tab, tmax, x, out_rings=rings)
    b = hybrid.hybrid_convolve(geom, tab, tmax, x, out_rings=rings)
    assert np.abs(a - b).max() <= 1e-13 * np.abs(a).max()


def test_healpix_point_source_sign_of_eq8():
    """A point source near the cap boundary: with the wrong sign in Eq. 8 (or delta_ij transposed) the response
    lands half a pixel off and the error is O(1); with the right one it is the interpolation error only."""
    nside = 16
    geom = geometry.healpix_ring(nside)
    pix = np.sqrt(4 * np.pi / geom.npix)
    fwhm = 3.0 * pix
    tmax = 3 * fwhm
    sigma = fwhm * inputs.FWHM_TO_SIGMA
    tab = gauss(fwhm, tmax)
    mp = hybrid.mprime_resolving(geom, tmax, 5.5 / sigma)
    x = np.zeros(geom.npix)
    q0 = int(geom.offset[nside - 3]) + 5                      # in the north cap, two rings above the belt
    x[q0] = 1.0
    rings = np.arange(nside - 8, nside + 4)
    a = direct.direct_sum(geom, tab, tmax, x, out_rings=rings)
    b = hybrid.hybrid_convolve(geom, tab, tmax, x, mprime=mp, out_rings=rings)
    assert np.abs(a - b).max() <= 1e-8 * np.abs(a).max()


def test_cap_method_error_orders():
    """Method error of the Fourier scheme in the caps vs the brute force (SURVEY.md 8c probe table):
    paper's M = 4 nside: ~1e-4 (variant B) and ~1e-3 (variant A) for a 2.9-pixel Gaussian; resolved rows: <1e-8."""
    nside = 16
    geom = geometry.healpix_ring(nside)
    pix = np.sqrt(4 * np.pi / geom.npix)
    fwhm = 2.91 * pix
    tmax, sigma = 3 * fwhm, fwhm * inputs.FWHM_TO_SIGMA
    tab = gauss(fwhm, tmax)
    x = np.random.default_rng(1).standard_normal(geom.npix)
    a = direct.direct_sum(geom, tab, tmax, x)
    eB = frms(hybrid.hybrid_convolve(geom, tab, tmax, x), a)
    eA = frms(hybrid.hybrid_convolve(geom, tab, tmax, x, variant="A"), a)
    eR = frms(hybrid.hybrid_convolve(geom, tab, tmax, x, mprime=hybrid.mprime_resolving(geom, tmax, 5.0 / sigma)), a)
    assert 3e-5 < eB < 1e-3 and 5e-4 < eA < 2e-2 and eB < eA and eR < 1e-8


def test_hybrid_linear_shift_mirror():
    """Operator structure of #2 on HEALPix incl. caps: linearity; N/S mirror; a rotation by pi/2 about the pole
    axis (a shift of N_i/4 pixels on every ring) commutes with the operator."""
    nside = 4
    geom = geometry.healpix_ring(nside)
    tmax = 30 * DEG
    tab = gauss(20 * DEG, tmax)
    rng = np.random.default_rng(21)
    f, g = rng.standard_normal((2, geom.npix))
    H = lambda m: hybrid.hybrid_convolve(geom, tab, tmax, m, mprime=64)   # noqa: E731
    Hf, Hg = H(f), H(g)
    np.testing.assert_allclose(H(2 * f - 3 * g), 2 * Hf - 3 * Hg, atol=1e-13)

    def rot(m):
        return np.concatenate([np.roll(m[geom.ring_slice(i)], int(geom.n[i]) // 4) for i in range(geom.nrings)])

    def mirror(m):
        return np.concatenate([m[geom.ring_slice(i)] for i in range(geom.nrings - 1, -1, -1)])
    np.testing.assert_allclose(H(rot(f)), rot(Hf), atol=1e-13)
    np.testing.assert_allclose(H(mirror(f)), mirror(Hf), atol=1e-13)


def test_ecp_phi_shift_one_pixel():
    geom = geometry.ecp(10, 16)
    tmax = 40 * DEG
    tab = gauss(25 * DEG, tmax)
    f = np.random.default_rng(4).standard_normal(geom.npix)
    sh = lambda m: np.roll(m.reshape(10, 16), 1, axis=1).ravel()          # noqa: E731
    for op in (lambda m: hybrid.hybrid_convolve(geom, tab, tmax, m), lambda m: direct.direct_sum(geom, tab, tmax, m)):
        np.testing.assert_allclose(op(sh(f)), sh(op(f)), atol=1e-13)


def test_funk_hecke_l0_l1():
    """Spectral action (Eq. 2-5): in = Y_lm sampled => out ~ K_l Y_lm, K_l = 2 pi int K P_l dz.
    Only to quadrature accuracy; l = 0, 1 on a fine ECP grid with a wide kernel."""
    geom = geometry.ecp(120, 240)
    fwhm = 16 * DEG
    sigma = fwhm * inputs.FWHM_TO_SIGMA
    tmax = 3.5 * sigma
    tab = gauss(fwhm, tmax)
    t = np.linspace(0, tmax, 400001)
    K = np.exp(-0.5 * (t / sigma) ** 2)
    w = np.full_like(t, t[1] - t[0])
    w[[0, -1]] *= 0.5
    K0 = 2 * np.pi * (K * np.sin(t) * w).sum()
    K1 = 2 * np.pi * (K * np.cos(t) * np.sin(t) * w).sum()
    ct = np.repeat(np.cos(geom.theta), geom.n)
    st = np.repeat(np.sin(geom.theta), geom.n)
    ph = np.concatenate([geom.phi(i) for i in range(geom.nrings)])
    rings = np.array([30, 59, 60, 95])
    sel = np.concatenate([np.arange(geom.offset[r], geom.offset[r + 1]) for r in rings])
    for lm, (Y, Kl) in {"00": (np.ones(geom.npix), K0), "10": (ct, K1), "11": (st * np.cos(ph), K1)}.items():
        for op in (direct.direct_sum, hybrid.hybrid_convolve):
            out = op(geom, tab, tmax, Y, out_rings=rings)
            assert np.abs(out - Kl * Y[sel]).max() < 2e-3 * abs(Kl), lm


# ---------------------------------------------------------------- oracle #2, variant A ------------------------
# The basic scheme (PAPER.md:125 zero-padding, PAPER.md:142 truncation at the ring's Nyquist frequency) treats the samples
# of input ring j as their band-limited trigonometric interpolant.  A single azimuthal harmonic on one input ring is
# therefore mapped to the same harmonic on every output ring of the band, scaled by the cosine transform of the
# kernel row:   in(j, l) = trig(m0 phi_jl)   =>   out(i, k) = Omega_j (N_j / M) kt_ij[m0] trig(m0 phi_ik)
# for m0 <= N_j / 2 and m0 <= N_i / 2, and 0 for m0 > N_i / 2; kt_ij[m0] = sum_d kappa_ij(psi_d) cos(m0 psi_d) over the
# M sample positions psi_d of the row (offset by phi0_i - phi0_j for two full-length rings).
# The expectation is evaluated here from that closed statement (hybrid.kernel_row is pinned by the Jacobi-Anger test).

def _variant_a_expectation(geom, i, j, m0, trig, tab, tmax, M):
    class_e = geom.n[i] == geom.n.max() and geom.n[j] == geom.n.max()
    delta = geom.phi0[i] - geom.phi0[j] if class_e else 0.0
    psi = delta + 2.0 * np.pi * np.arange(M) / M
    kt = float((hybrid.kernel_row(geom.theta[i], geom.theta[j], psi, tab, tmax) * np.cos(m0 * psi)).sum())
    if 2 * m0 > geom.n[i] or 2 * m0 > geom.n[j]:
        return np.zeros(int(geom.n[i]))
    return geom.omega[j] * (geom.n[j] / M) * kt * trig(m0 * geom.phi(i))


@pytest.mark.parametrize("case", ["interior", "nyquist_of_j", "edge_of_i"])
def test_variant_a_single_harmonic(case):
    """Pins the zero-pad weights (half/half split of ring j's own Nyquist bin, nothing above it), the truncation edge
    of the output ring (|m| = N_i/2 kept, N_i/2 + 1 dropped), the sign of Eq. 8 and the normalisation of variant A."""
    nside = 8
    geom = geometry.healpix_ring(nside)
    tmax = 40 * DEG
    tab = gauss(25 * DEG, tmax)
    M = 64
    if case == "interior":          # harmonic well below both Nyquist frequencies; cap, cap-boundary and equatorial pairs
        todo = [(5, 6, 3, np.cos), (6, 5, 3, np.sin), (7, 8, 7, np.cos), (9, 6, 4, np.sin), (12, 13, 9, np.cos), (13, 12, 9, np.sin)]
    elif case == "nyquist_of_j":    # m0 = N_j / 2 exactly: on a shifted ring cos(m0 phi_jl) = 0, sin(m0 phi_jl) = (-1)^l
        todo = [(6, 4, 10, np.sin), (5, 5, 12, np.sin), (7, 3, 8, np.sin), (3, 4, 10, np.sin)]      # last: N_i < N_j, truncated
    else:                           # output ring shorter than the input ring: m0 = N_i/2 - 1, N_i/2, N_i/2 + 1
        todo = [(3, 6, 7, np.cos), (3, 6, 8, np.sin), (3, 6, 9, np.cos), (3, 6, 9, np.sin), (4, 9, 11, np.cos)]
    for i, j, m0, trig in todo:
        x = np.zeros(geom.npix)
        x[geom.ring_slice(j)] = trig(m0 * geom.phi(j))
        assert np.abs(x).max() > 0.5
        out = hybrid.hybrid_convolve(geom, tab, tmax, x, variant="A", mprime=M, out_rings=np.array([i]))
        expect = _variant_a_expectation(geom, i, j, m0, trig, tab, tmax, int(geom.n[i]) if geom.n[i] == geom.n[j] == 4 * nside else M)
        scale = geom.omega[j] * geom.n[j]
        assert np.abs(out - expect).max() <= 1e-13 * scale, (case, i, j, m0)
        if case != "interior" and 2 * m0 <= geom.n[i] and 2 * m0 <= geom.n[j]:
            assert np.abs(expect).max() > 1e-4 * scale          # the kept edge modes really carry signal


def test_variant_a_ecp_equals_direct():
    """On ECP every pair is class E and N_i = N_j = M: zero-padding and truncation do nothing, so variant A is the
    same exact circulant identity as variant B ("vanish exactly")."""
    geom = geometry.ecp(12, 24)
    tmax = 35 * DEG
    tab = inputs.tophat_table(tmax)
    x = np.random.default_rng(17).standard_normal(geom.npix)
    a = direct.direct_sum(geom, tab, tmax, x)
    b = hybrid.hybrid_convolve(geom, tab, tmax, x, variant="A")
    assert np.abs(a - b).max() <= 1e-13 * np.abs(a).max()


def test_direct_dft_beyond_library_switch():
    """hybrid.dft switches to the library FFT above 1024 points: one direct-definition spot check at a longer length."""
    N = 1500
    x = np.random.default_rng(2).standard_normal(N) + 1j * np.random.default_rng(3).standard_normal(N)
    X = hybrid.dft(x)
    for m in (0, 1, 749, 750, 1499):
        assert abs(X[m] - (x * np.exp(-2j * np.pi * ((m * np.arange(N)) % N) / N)).sum()) <= 1e-10 * np.abs(x).sum()
