"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on seeded inputs.

Tolerances (BASELINE.json north_star):
  fp64 path          max |gpu - oracle| <= 1e-12 max |oracle|
  fp32 path, ECP     fractional RMS <= 1e-6 vs the fp64 brute-force sum
  fp32 path, HEALPix fractional RMS <= 1e-5 vs the brute-force sum; <= 1e-6 vs the fp64 hybrid oracle with the same M'
"""
import numpy as np
import pytest

from oracle import geometry, direct, hybrid
from paper_1104_0672_b200 import arkcos, inputs
from plan_checks import plan_mprime

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

DEG, ARCMIN = inputs.DEG, inputs.ARCMIN


def frms(a, b):
    a, b = np.asarray(a, float), np.asarray(b, float)
    return float(np.sqrt(((a - b) ** 2).sum() / (b ** 2).sum()))


def maxrel(a, b):
    return float(np.abs(np.asarray(a, float) - b).max() / np.abs(b).max())


def geom_of(pix):
    return geometry.ecp(pix[1], pix[2]) if pix[0] == "ecp" else geometry.healpix_ring(pix[1])


def gpu_convolve(pix, table, tmax, x, dtype=arkcos.F32, plan=None, **opts):
    """x: numpy [npix] or [nmaps, npix]; returns numpy of the same shape (and the plan)."""
    tdt = torch.float32 if dtype == arkcos.F32 else torch.float64
    nmaps = 1 if x.ndim == 1 else x.shape[0]
    if plan is None:
        plan = arkcos.Plan(pix, table, tmax, dtype, max_nmaps=nmaps, **opts)
    d_in = torch.from_numpy(np.ascontiguousarray(x)).to(device="cuda", dtype=tdt)
    d_out = torch.full_like(d_in, float("nan"))
    plan.convolve(d_in.data_ptr(), d_out.data_ptr(), nmaps, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return d_out.cpu().numpy(), plan


def take_rings(geom, full, rings):
    return np.concatenate([full[..., geom.ring_slice(int(r))] for r in rings], axis=-1)


def sample_rings(geom, extra=(), nrand=8, seed=0):
    R = geom.nrings
    base = {0, 1, 2, R // 4, R // 2 - 1, R // 2, R // 2 + 1, (3 * R) // 4, R - 3, R - 2, R - 1}
    rng = np.random.default_rng(seed)
    base |= set(int(v) for v in rng.integers(0, R, nrand)) | set(int(e) for e in extra)
    return np.array(sorted(r for r in base if 0 <= r < R))


# ------------------------------------------------------------------ config 1: ECP 64 x 128 -------------------------

def test_cfg1_fp64_and_fp32():
    c = inputs.config(1)
    geom, tab, tmax = geom_of(c["pix"]), inputs.kernel_table(c), c["theta_max"]
    x = inputs.white_noise(geom.npix, 1, dtype=np.float64)
    ref = direct.direct_sum(geom, tab, tmax, x)
    out64, _ = gpu_convolve(c["pix"], tab, tmax, x, arkcos.F64)
    assert maxrel(out64, ref) <= 1e-12
    x32 = x.astype(np.float32)
    ref32 = direct.direct_sum(geom, tab, tmax, x32.astype(np.float64))
    out32, _ = gpu_convolve(c["pix"], tab, tmax, x32, arkcos.F32)
    assert frms(out32, ref32) <= 1e-6
    # and against the scheme oracle
    assert maxrel(out64, hybrid.hybrid_convolve(geom, tab, tmax, x)) <= 1e-12


# ------------------------------------------------------------------ config 2: ECP 1024 x 2048 ----------------------

def test_cfg2_fp32_sampled_rings():
    c = inputs.config(2)
    geom, tab, tmax = geom_of(c["pix"]), inputs.kernel_table(c), c["theta_max"]
    x = inputs.white_noise(geom.npix, 2)
    out, _ = gpu_convolve(c["pix"], tab, tmax, x)
    assert np.isfinite(out).all()
    rings = sample_rings(geom, nrand=6, seed=2)
    ref = direct.direct_sum(geom, tab, tmax, x.astype(np.float64), out_rings=rings)
    assert frms(take_rings(geom, out, rings), ref) <= 1e-6


# ------------------------------------------------------------------ small HEALPix, whole map -----------------------

@pytest.mark.parametrize("nside,dtype", [(1, arkcos.F64), (2, arkcos.F64), (16, arkcos.F64), (16, arkcos.F32),
                                         (32, arkcos.F32)])
def test_healpix_small_full_map(nside, dtype):
    geom = geometry.healpix_ring(nside)
    pixsz = np.sqrt(4 * np.pi / geom.npix)
    fwhm = 2.5 * pixsz
    sigma, tmax = fwhm * inputs.FWHM_TO_SIGMA, min(3 * fwhm, np.pi)
    tab = inputs.gaussian_table(fwhm, tmax)
    ell = 5.5 / sigma
    x = inputs.white_noise(geom.npix, 9, dtype=np.float64 if dtype == arkcos.F64 else np.float32)
    out, plan = gpu_convolve(("healpix", nside), tab, tmax, x, dtype, ell_nyquist=ell)
    mp = plan_mprime(plan, geom, tmax, ell)
    ref2 = hybrid.hybrid_convolve(geom, tab, tmax, x.astype(np.float64), mprime=mp)
    ref1 = direct.direct_sum(geom, tab, tmax, x.astype(np.float64))
    if dtype == arkcos.F64:
        assert maxrel(out, ref2) <= 1e-12
    else:
        assert frms(out, ref2) <= 1e-6
    if nside >= 16:
        assert frms(out, ref1) <= 1e-5


@pytest.mark.parametrize("nside,fwhm_px,nmaps", [(128, 2.0, 2), (256, 3.0, 3), (256, 1.5, 1)])
def test_healpix_mid_size_all_kernel_classes(nside, fwhm_px, nmaps):
    """Sizes at which the cap-run kernel, the register-resident FFTs (Q = 512, 1024) and the pole / general / uniform
    kernels all serve some rings: every sampled ring equals oracle #2 at the plan's M' and oracle #1 to 1e-5."""
    geom = geometry.healpix_ring(nside)
    fwhm = fwhm_px * np.sqrt(4 * np.pi / geom.npix)
    tmax = 3 * fwhm
    tab = inputs.gaussian_table(fwhm, tmax)
    x = inputs.white_noise_maps(geom.npix, 11, nmaps)
    out, plan = gpu_convolve(("healpix", nside), tab, tmax, x)
    assert np.isfinite(out).all()
    mp = plan_mprime(plan, geom, tmax)
    R = geom.nrings
    rings = np.unique(np.concatenate([np.arange(0, 12), np.arange(nside // 8 - 2, nside // 8 + 3), [nside // 2, nside // 2 + 1],
                                      np.arange(nside - 16, nside + 16, 3), [2 * nside - 1, 3 * nside], R - 1 - np.arange(0, 40, 7)]))
    ref2 = hybrid.hybrid_convolve(geom, tab, tmax, x.astype(np.float64), mprime=mp, out_rings=rings)
    assert frms(take_rings(geom, out, rings), ref2) <= 1e-6
    ref1 = direct.direct_sum(geom, tab, tmax, x.astype(np.float64), out_rings=rings)
    assert frms(take_rings(geom, out, rings), ref1) <= 1e-5


@pytest.mark.parametrize("cache,nmaps", [(0, 3), (1, 3), (1, 5)], ids=["computed", "cached_spectra", "cached_spectra_5maps"])
@pytest.mark.parametrize("kernel", ["gauss", "tophat", "mexhat"])
def test_healpix_256_cap_runs_and_cached_spectra(kernel, cache, nmaps):
    """nside 256, 3 or 5 maps: single-period cap runs (Gaussian), multi-period ones (hard-edged kernels: M' up to 3 N_i) and
    the cached-spectra kernels (options.cache_kernel_spectra: two maps per read of G, four from four maps on) against
    oracle #2 at the plan's M'."""
    nside = 256
    geom = geometry.healpix_ring(nside)
    px = np.sqrt(4 * np.pi / geom.npix)
    tab, tmax = {"gauss": (inputs.gaussian_table(2.5 * px, 7.5 * px), 7.5 * px),
                 "tophat": (inputs.tophat_table(5.8 * px), 5.8 * px),
                 "mexhat": (inputs.mexican_hat_table(2.33 * px, 5 * 2.33 * px), 5 * 2.33 * px)}[kernel]
    x = inputs.white_noise_maps(geom.npix, 12, nmaps)
    out, plan = gpu_convolve(("healpix", nside), tab, tmax, x, cache_kernel_spectra=cache)
    assert np.isfinite(out).all()
    mp = np.array([plan.ring_info(i)["mprime"] for i in range(geom.nrings)])
    R = geom.nrings
    rings = np.unique(np.concatenate([[0, 5, 40, 127, 128, 129, 160, 200, 255, 256, 257, 300, 511, 700], R - 1 - np.array([0, 50, 130, 250])]))
    ref2 = hybrid.hybrid_convolve(geom, tab, tmax, x.astype(np.float64), mprime=mp, out_rings=rings)
    assert frms(take_rings(geom, out, rings), ref2) <= 1e-6
    # a second call on the same plan (accumulating fold: the output spectrum must be cleared every time)
    out2, _ = gpu_convolve(("healpix", nside), tab, tmax, x, plan=plan)
    assert frms(take_rings(geom, out2, rings), ref2) <= 1e-6


def test_healpix_paper_grid_polar_oversample():
    """polar_oversample = 1 is the paper's M = 4 nside: parity with oracle #2 at the same M."""
    nside = 16
    geom = geometry.healpix_ring(nside)
    fwhm = 3 * np.sqrt(4 * np.pi / geom.npix)
    tmax = 3 * fwhm
    tab = inputs.gaussian_table(fwhm, tmax)
    x = inputs.white_noise(geom.npix, 9, dtype=np.float64)
    out, _ = gpu_convolve(("healpix", nside), tab, tmax, x, arkcos.F64, polar_oversample=1)
    assert maxrel(out, hybrid.hybrid_convolve(geom, tab, tmax, x, mprime=4 * nside)) <= 1e-12


@pytest.mark.parametrize("dtype,oversample", [(arkcos.F64, 1), (arkcos.F64, 0), (arkcos.F32, 1)])
def test_variant_a_zero_pad_truncate(dtype, oversample):
    """variant = 1 is the paper's basic scheme: parity with oracle #2 run as variant "A"."""
    nside = 16
    geom = geometry.healpix_ring(nside)
    fwhm = 3 * np.sqrt(4 * np.pi / geom.npix)
    tmax = 3 * fwhm
    tab = inputs.gaussian_table(fwhm, tmax)
    x = inputs.white_noise(geom.npix, 9, dtype=np.float64 if dtype == arkcos.F64 else np.float32)
    out, plan = gpu_convolve(("healpix", nside), tab, tmax, x, dtype, variant=1, polar_oversample=oversample)
    mp = np.array([plan.ring_info(i)["mprime"] for i in range(geom.nrings)])
    ref = hybrid.hybrid_convolve(geom, tab, tmax, x.astype(np.float64), variant="A", mprime=mp)
    refB = hybrid.hybrid_convolve(geom, tab, tmax, x.astype(np.float64), variant="B", mprime=mp)
    assert maxrel(refB, ref) > 1e-4                      # the two variants really differ on white noise
    if dtype == arkcos.F64:
        assert maxrel(out, ref) <= 1e-12
    else:
        assert frms(out, ref) <= 1e-6
    # ECP: both variants coincide (every pair is class E, nothing above the common Nyquist frequency)
    ge = geometry.ecp(16, 32)
    te = inputs.gaussian_table(0.5, 1.0, 4096)
    xe = inputs.white_noise(ge.npix, 8, dtype=np.float64)
    oa, _ = gpu_convolve(("ecp", 16, 32), te, 1.0, xe, arkcos.F64, variant=1)
    assert maxrel(oa, direct.direct_sum(ge, te, 1.0, xe)) <= 1e-12


def test_hard_edged_kernels_vs_scheme_oracle():
    """Top-hat and Mexican hat (config 5's kernels) at nside 32, 3 maps: GPU == oracle #2; equatorial rings == oracle #1."""
    nside = 32
    geom = geometry.healpix_ring(nside)
    pixsz = np.sqrt(4 * np.pi / geom.npix)
    x = inputs.white_noise_maps(geom.npix, 5, 3)
    for tab, tmax in [(inputs.tophat_table(5.8 * pixsz), 5.8 * pixsz),
                      (inputs.mexican_hat_table(2.33 * pixsz, 5 * 2.33 * pixsz), 5 * 2.33 * pixsz)]:
        ell = 6.0 * nside
        out, plan = gpu_convolve(("healpix", nside), tab, tmax, x, arkcos.F32, ell_nyquist=ell)
        mp = plan_mprime(plan, geom, tmax, ell)
        ref2 = hybrid.hybrid_convolve(geom, tab, tmax, x.astype(np.float64), mprime=mp)
        assert frms(out, ref2) <= 1e-6
        eq = np.array([i for i in range(geom.nrings) if np.all(geom.n[geometry.band(geom, i, tmax)] == 4 * nside)])
        ref1 = direct.direct_sum(geom, tab, tmax, x.astype(np.float64), out_rings=eq)
        assert frms(take_rings(geom, out, eq), ref1) <= 1e-6


@pytest.mark.parametrize("pix", [("healpix", 32), ("ecp", 48, 128)], ids=["healpix32", "ecp48x128"])
def test_input_in_the_nyquist_bin_of_full_length_rings(pix):
    """Every ring carries (-1)^k times a ring amplitude: on rings of the full length that is the m = N/2 mode alone, so the
    equatorial (class-E) output rings are made by the Nyquist bin of the band step and nothing else (half weight for the two
    folded families, sine part on HEALPix's shifted rings).  Hard-edged kernel: G_ij[N/2] is far from zero."""
    geom = geom_of(pix)
    pixsz = np.sqrt(4 * np.pi / geom.npix)
    tmax = 5.8 * pixsz
    tab = inputs.tophat_table(tmax)
    amp = np.random.default_rng(17).standard_normal((2, geom.nrings))
    x = np.zeros((2, geom.npix), np.float32)
    for i in range(geom.nrings):
        x[:, geom.ring_slice(i)] = amp[:, i, None] * (1.0 - 2.0 * (np.arange(geom.n[i]) & 1))[None, :]
    out, _ = gpu_convolve(pix, tab, tmax, x, arkcos.F32)
    nfull = geom.n.max()
    eq = np.array([i for i in range(geom.nrings) if np.all(geom.n[geometry.band(geom, i, tmax)] == nfull)])
    assert eq.size >= geom.nrings // 4
    ref1 = direct.direct_sum(geom, tab, tmax, x.astype(np.float64), out_rings=eq)
    assert np.abs(ref1).max() > 1e-3 * np.abs(amp).max() * tab.max() * pixsz ** 2          # the test is not vacuous
    assert frms(take_rings(geom, out, eq), ref1) <= 1e-6


@pytest.mark.parametrize("dtype,nmaps", [(arkcos.F32, 3), (arkcos.F32, 1), (arkcos.F64, 9)])
def test_exact_caps_hard_edged_kernels(dtype, nmaps):
    """exact_caps = 1: cap-zone rings by the direct-space sum: the WHOLE map equals the
    brute-force oracle for the disc and the cut Mexican hat, which the Fourier scheme alone cannot do (reading R18)."""
    nside = 32
    geom = geometry.healpix_ring(nside)
    pixsz = np.sqrt(4 * np.pi / geom.npix)
    x = inputs.white_noise_maps(geom.npix, 5, nmaps)
    if dtype == arkcos.F64:
        x = x.astype(np.float64)
    for tab, tmax in [(inputs.tophat_table(5.8 * pixsz), 5.8 * pixsz),
                      (inputs.mexican_hat_table(2.33 * pixsz, 5 * 2.33 * pixsz), 5 * 2.33 * pixsz)]:
        out, _ = gpu_convolve(("healpix", nside), tab, tmax, x, dtype, exact_caps=1)
        ref1 = direct.direct_sum(geom, tab, tmax, x.astype(np.float64))
        if dtype == arkcos.F64:
            assert maxrel(out, ref1) <= 1e-12
        else:
            assert frms(out, ref1) <= 1e-6
        plain, _ = gpu_convolve(("healpix", nside), tab, tmax, x, dtype)
        assert frms(plain, ref1) > 1e-5            # without the option the caps carry the scheme's artifact level


@pytest.mark.parametrize("nside", [1, 2, 4, 8])
def test_exact_caps_tiny_grids_and_map_counts(nside):
    """exact_caps on the smallest grids (rings of 4 .. 32 pixels: quadrants of one pixel, whole-ring windows, most threads of
    a block idle) and with 1, 5, 17 maps (one, eight and a partial chunk of maps per thread; 3 fp64 maps) against the
    brute-force sum (Eq. 6)."""
    geom = geometry.healpix_ring(nside)
    pixsz = np.sqrt(4 * np.pi / geom.npix)
    for tmax in (1.5 * pixsz, min(4.0 * pixsz, 3.0)):
        tab = inputs.gaussian_table(tmax / 2, tmax)
        for dtype, nmaps in ((arkcos.F32, 1), (arkcos.F32, 5), (arkcos.F64, 3), (arkcos.F32, 17)):
            x = inputs.white_noise_maps(geom.npix, 3, nmaps)
            if dtype == arkcos.F64:
                x = x.astype(np.float64)
            out, _ = gpu_convolve(("healpix", nside), tab, tmax, x, dtype, exact_caps=1)
            ref = direct.direct_sum(geom, tab, tmax, x.astype(np.float64))
            assert maxrel(out, ref) <= (1e-12 if dtype == arkcos.F64 else 2e-6)


@pytest.mark.parametrize("dtype,nmaps", [(arkcos.F64, 3), (arkcos.F32, 5), (arkcos.F32, 2)])
def test_exact_caps_wide_kernel_long_windows(dtype, nmaps):
    """exact_caps with a kernel 100 pixels wide (Eq. 6): the input windows of a thread block are longer than the
    direct-space kernel stages in shared memory (its global-memory path), a ring has more ring pairs than one staging pass of
    the pair constants holds, whole-ring windows of up to 400 pixels next to the poles (the rotation along the ring runs
    that long), and the two-map form.  Sampled rings against the brute-force sum."""
    nside = 256
    geom = geometry.healpix_ring(nside)
    tmax = 0.32
    tab = inputs.gaussian_table(0.25, tmax)
    x = inputs.white_noise_maps(geom.npix, 7, nmaps)
    if dtype == arkcos.F64:
        x = x.astype(np.float64)
    out, plan = gpu_convolve(("healpix", nside), tab, tmax, x, dtype, exact_caps=1)
    assert np.isfinite(out).all()
    R = geom.nrings
    rings = np.array([0, 1, 5, 50, 99, 120, 200, 255, 256, 300, R - 1 - 301, R - 1 - 120, R - 1 - 50, R - 1])
    ref1 = direct.direct_sum(geom, tab, tmax, x.astype(np.float64), out_rings=rings)
    got = take_rings(geom, out, rings)
    if dtype == arkcos.F64:
        assert maxrel(got, ref1) <= 1e-12
    else:
        # 2e4 input pixels per output pixel summed in fp32: the bound of north_star for HEALPix, not the 1e-6 of compact kernels
        err = frms(got, ref1)
        print(f"\nwide kernel, fp32, {nmaps} maps: fractional RMS vs brute force = {err:.2e}")
        assert err <= 1e-5


# ------------------------------------------------------------------ config 3: HEALPix nside 512 --------------------

def test_cfg3_fp32_sampled_rings():
    c = inputs.config(3)
    nside = c["pix"][1]
    geom, tab, tmax = geom_of(c["pix"]), inputs.kernel_table(c), c["theta_max"]
    x = inputs.white_noise(geom.npix, 3)
    out, plan = gpu_convolve(c["pix"], tab, tmax, x)
    assert np.isfinite(out).all()
    rings = sample_rings(geom, extra=(nside - 2, nside - 1, nside, nside + 5, 2 * nside - 1, 330, 126), seed=3)
    ref = direct.direct_sum(geom, tab, tmax, x.astype(np.float64), out_rings=rings)
    assert frms(take_rings(geom, out, rings), ref) <= 1e-5
    # same M' in the scheme oracle on a few rings
    mp = plan_mprime(plan, geom, tmax)
    few = np.array([0, 5, 126, nside - 1, nside + 3, 2 * nside - 1])
    ref2 = hybrid.hybrid_convolve(geom, tab, tmax, x.astype(np.float64), mprime=mp, out_rings=few)
    assert frms(take_rings(geom, out, few), ref2) <= 1e-6


# ------------------------------------------------------------------ config 4: HEALPix nside 2048 -------------------

def test_cfg4_full_size_sampled_rings():
    c = inputs.config(4)
    nside = c["pix"][1]
    geom, tab, tmax = geom_of(c["pix"]), inputs.kernel_table(c), c["theta_max"]
    x = inputs.add_point_sources(inputs.white_noise(geom.npix, 4))
    out, plan = gpu_convolve(c["pix"], tab, tmax, x)
    assert np.isfinite(out).all()
    # rings: poles, prime-length / power-of-two-length cap rings (N = 4 * 509, 4 * 512), cap boundary +- band, equator,
    # random, and the rings of a few point sources
    src_rings = np.searchsorted(geom.offset, np.random.default_rng(inputs.BASE_SEED + 499).integers(0, geom.npix, 1000)[:6],
                                side="right") - 1
    rings = sample_rings(geom, extra=(508, 511, 1020, nside - 14, nside - 2, nside - 1, nside, nside + 12, 2 * nside - 1,
                                      3 * nside - 1, 3 * nside + 10, *src_rings), nrand=10, seed=4)
    ref = direct.direct_sum(geom, tab, tmax, x.astype(np.float64), out_rings=rings)
    got = take_rings(geom, out, rings)
    assert frms(got, ref) <= 1e-5
    # per-ring: no single ring is off (amplitude-100 sources included)
    o = 0
    for r in rings:
        n = int(geom.n[r])
        assert np.abs(got[o:o + n] - ref[o:o + n]).max() <= 3e-5 * np.abs(ref).max(), int(r)
        o += n


def test_nside4096_maximum_size_sampled_rings():
    """The largest HEALPix grid an fp32 plan accepts: the belt rings of 16384 pixels as two size-4096 transforms
    per ring, the cap rings of 8196 .. 16380 pixels by a Bluestein convolution of 16384 points built from the same transforms
    (rings 2048, 2049, 3000, 4094 and a mirror ring), the shorter ones as at the smaller sizes."""
    nside = 4096
    geom = geometry.healpix_ring(nside)
    fwhm, tmax = 2.5 * ARCMIN, 7.5 * ARCMIN
    tab = inputs.gaussian_table(fwhm, tmax)
    x = inputs.white_noise_maps(geom.npix, 6, 2)
    out, _ = gpu_convolve(("healpix", nside), tab, tmax, x)
    assert np.isfinite(out).all()
    rings = np.array([0, 3, 700, 2047, 2048, 2049, 3000, nside - 2, nside - 1, nside, nside + 5, 2 * nside - 1, 3 * nside + 2,
                      geom.nrings - 1 - 3000, geom.nrings - 1])
    ref = direct.direct_sum(geom, tab, tmax, x.astype(np.float64), out_rings=rings)
    assert frms(take_rings(geom, out, rings), ref) <= 1e-5


def test_ecp_rings_of_16384_pixels():
    """ECP rings of 16384 pixels (8192 complex points: two register-resident size-4096 transforms and a radix-2 step per ring,
    PAPER.md:125 / 142 for the ring transforms): every pair is exact on ECP, so the fp32 bound of 1e-6 applies."""
    pix = ("ecp", 24, 16384)
    geom = geom_of(pix)
    tmax = 0.15                         # neighbouring rings are 0.13 apart: bands of three rings, rows of up to 800 samples
    tab = inputs.gaussian_table(0.1, tmax)
    x = inputs.white_noise_maps(geom.npix, 8, 2)
    out, plan = gpu_convolve(pix, tab, tmax, x)
    assert np.isfinite(out).all()
    rings = np.array([0, 1, 7, 11, 12, 16, 23])
    ref = direct.direct_sum(geom, tab, tmax, x.astype(np.float64), out_rings=rings)
    assert frms(take_rings(geom, out, rings), ref) <= 1e-6


# ------------------------------------------------------------------ API behaviour -----------------------------------

def test_multi_map_equals_single_and_host_path():
    nside = 16
    geom = geometry.healpix_ring(nside)
    fwhm = 3 * np.sqrt(4 * np.pi / geom.npix)
    tmax = 3 * fwhm
    tab = inputs.gaussian_table(fwhm, tmax)
    x = inputs.white_noise_maps(geom.npix, 7, 4)
    out, plan = gpu_convolve(("healpix", nside), tab, tmax, x)
    for k in range(4):
        single, _ = gpu_convolve(("healpix", nside), tab, tmax, x[k], plan=plan)
        np.testing.assert_array_equal(single, out[k])
    h_in = torch.from_numpy(x).pin_memory()
    h_out = torch.empty_like(h_in).pin_memory()
    plan.convolve_host(h_in.data_ptr(), h_out.data_ptr(), 4, torch.cuda.current_stream().cuda_stream)
    np.testing.assert_array_equal(h_out.numpy(), out)
    # cached rows give the same bits
    out_c, _ = gpu_convolve(("healpix", nside), tab, tmax, x, cache_kernel_rows=1)
    np.testing.assert_array_equal(out_c, out)


def test_streaming_host_path_equals_device_path():
    """arkcos_convolve_host_async: five maps streamed through the two staging sets give the bits of arkcos_convolve."""
    nside = 32
    geom = geometry.healpix_ring(nside)
    fwhm = 3 * np.sqrt(4 * np.pi / geom.npix)
    tmax = 3 * fwhm
    tab = inputs.gaussian_table(fwhm, tmax)
    x = inputs.white_noise_maps(geom.npix, 7, 5)
    plan = arkcos.Plan(("healpix", nside), tab, tmax, arkcos.F32)
    ref = np.stack([gpu_convolve(("healpix", nside), tab, tmax, x[k], plan=plan)[0] for k in range(5)])
    h_in = torch.from_numpy(x).pin_memory()
    h_out = torch.full_like(h_in, float("nan")).pin_memory()
    for rep in range(2):
        for k in range(5):
            plan.convolve_host_async(h_in[k].data_ptr(), h_out[k].data_ptr(), 1)
        plan.synchronize()
        np.testing.assert_array_equal(h_out.numpy(), ref)
        h_out.fill_(float("nan"))


def test_argument_errors():
    tab = inputs.gaussian_table(0.2, 0.4, 256)
    plan = arkcos.Plan(("ecp", 8, 16), tab, 0.4, arkcos.F32, max_nmaps=2)
    a = torch.zeros(3, 128, device="cuda")
    b = torch.zeros(3, 128, device="cuda")
    s = torch.cuda.current_stream().cuda_stream
    for args in [(a.data_ptr(), a.data_ptr(), 1), (a.data_ptr(), b.data_ptr(), 3), (a.data_ptr(), b.data_ptr(), 0),
                 (0, b.data_ptr(), 1), (a.data_ptr(), a.data_ptr() + 256, 1)]:
        with pytest.raises(arkcos.ArkcosError) as e:
            plan.convolve(args[0], args[1], args[2], s)
        assert e.value.status == arkcos.INVALID_ARG
    plan.convolve(a.data_ptr(), b.data_ptr(), 2, s)
    torch.cuda.synchronize()
    assert torch.all(b[:2] == 0)


def test_degenerate_kernels():
    """Support narrower than the ring spacing (only the ring itself contributes) and support = the whole sphere."""
    geom = geometry.ecp(8, 16)
    x = inputs.white_noise(geom.npix, 8, dtype=np.float64)
    for tmax in (0.05, np.pi):
        tab = inputs.gaussian_table(0.8, tmax, 4096)
        out, _ = gpu_convolve(("ecp", 8, 16), tab, tmax, x, arkcos.F64)
        assert maxrel(out, direct.direct_sum(geom, tab, tmax, x)) <= 1e-12
    # HEALPix, support narrower than a pixel: in the equatorial region every pixel only sees itself (exact); in the
    # caps the Fourier scheme interpolates a sub-pixel kernel, so there the reference is the scheme oracle at the same M'
    geom = geometry.healpix_ring(4)
    xh = inputs.white_noise(geom.npix, 8, dtype=np.float64)
    tab = inputs.gaussian_table(0.01, 0.02, 4096)
    out, plan = gpu_convolve(("healpix", 4), tab, 0.02, xh, arkcos.F64, ell_nyquist=40.0)
    mp = plan_mprime(plan, geom, 0.02, 40.0)
    assert maxrel(out, hybrid.hybrid_convolve(geom, tab, 0.02, xh, mprime=mp)) <= 1e-12
    eq = slice(int(geom.offset[3]), int(geom.offset[12]))
    np.testing.assert_allclose(out[eq], xh[eq] * geom.omega[0], rtol=1e-12)


# ------------------------------------------------------------------ config 5: 16 maps, hard-edged kernels, full size -

@pytest.mark.parametrize("which", [0, 1], ids=["tophat", "mexican_hat"])
def test_cfg5_full_size(which):
    """DESIGN.md reading R18: GPU == oracle #2 at the plan's M' (<= 1e-6), equatorial-band rings == oracle #1 (<= 1e-6);
    the cap-ring difference to the brute-force sum is the artifact level of the Fourier scheme and is only reported."""
    c = inputs.config(5)
    spec = c["kernels"][which]
    nside, nmaps = c["pix"][1], c["nmaps"]
    geom, tab, tmax = geom_of(c["pix"]), inputs.kernel_table(spec), spec["theta_max"]
    x = inputs.white_noise_maps(geom.npix, 5, nmaps)
    out, plan = gpu_convolve(c["pix"], tab, tmax, x)
    assert np.isfinite(out).all()
    mp = plan_mprime(plan, geom, tmax)
    few = np.array([3, 700, nside - 1, nside + 2, 2 * nside - 1, 3 * nside + 1, geom.nrings - 40])
    ref2 = hybrid.hybrid_convolve(geom, tab, tmax, x.astype(np.float64), mprime=mp, out_rings=few)
    assert frms(take_rings(geom, out, few), ref2) <= 1e-6
    eq = np.array([nside + 40, 2 * nside - 1, 2 * nside, 3 * nside - 45])
    assert all(np.all(geom.n[geometry.band(geom, int(i), tmax)] == 4 * nside) for i in eq)
    ref1 = direct.direct_sum(geom, tab, tmax, x.astype(np.float64), out_rings=eq)
    assert frms(take_rings(geom, out, eq), ref1) <= 1e-6
    cap = np.array([100, 1000, nside - 5, nside + 3, geom.nrings - 700])
    refc = direct.direct_sum(geom, tab, tmax, x.astype(np.float64), out_rings=cap)
    print(f"\ncfg5 {spec['kernel']}: cap-ring fractional RMS vs brute force = {frms(take_rings(geom, out, cap), refc):.2e}"
          f" (ell_nyquist {plan.ell_nyquist:.0f})")
    # with exact_caps the cap zone is the direct-space sum: the 1e-5 of north_star holds on every ring
    del plan
    out_x, _ = gpu_convolve(c["pix"], tab, tmax, x, exact_caps=1)
    assert frms(take_rings(geom, out_x, cap), refc) <= 1e-6
    assert frms(take_rings(geom, out_x, eq), ref1) <= 1e-6
    np.testing.assert_array_equal(take_rings(geom, out_x, eq), take_rings(geom, out, eq))


# ------------------------------------------------------------------ regressions found by review ---------------------

def test_ecp_odd_ntheta_run_ending_on_middle_ring():
    """ECP with an odd number of rings and rows of 13..20 samples at the equator: the cap-run kernel serves a run that
    ends on the self-mirror middle ring; the mirror images of the other rings of that run must be cleared on every
    call (round-1 review: they were not, the result drifted from call to call)."""
    pix = ("ecp", 511, 1024)
    geom = geom_of(pix)
    tmax = 0.1
    tab = inputs.gaussian_table(0.06, tmax)
    x = inputs.white_noise(geom.npix, 21)
    out, plan = gpu_convolve(pix, tab, tmax, x)
    rings = np.array([0, 3, 100, 250, 254, 255, 256, 257, 260, 262, 400, 510])
    ref1 = direct.direct_sum(geom, tab, tmax, x.astype(np.float64), out_rings=rings)
    assert frms(take_rings(geom, out, rings), ref1) <= 1e-6
    out2, _ = gpu_convolve(pix, tab, tmax, x, plan=plan)
    assert frms(take_rings(geom, out2, rings), ref1) <= 1e-6
    np.testing.assert_array_equal(out, out2)


def test_cached_spectra_long_equatorial_rows():
    """cache_kernel_spectra with equatorial rows longer than 12 samples (disc of 14 pixels at nside 256): every bin,
    the Nyquist bin m = M/2 included, must come from the whole row (round-1 review: that bin used a row cut at 12)."""
    nside, nmaps = 256, 2
    geom = geometry.healpix_ring(nside)
    px = np.sqrt(4 * np.pi / geom.npix)
    tmax = 14 * px
    tab = inputs.tophat_table(tmax)
    x = inputs.white_noise_maps(geom.npix, 13, nmaps)
    # an input that lives at the Nyquist frequency of the equatorial rings makes that bin visible
    x[:, geom.offset[400]:geom.offset[401]] += 50.0 * (-1.0) ** np.arange(4 * nside, dtype=np.float32)
    x[:, geom.offset[511]:geom.offset[512]] += 50.0 * (-1.0) ** np.arange(4 * nside, dtype=np.float32)
    out, plan = gpu_convolve(("healpix", nside), tab, tmax, x, cache_kernel_spectra=1)
    eq = np.array([i for i in range(geom.nrings) if np.all(geom.n[geometry.band(geom, i, tmax)] == 4 * nside)])
    rings = eq[[0, 1, len(eq) // 3, len(eq) // 2, len(eq) - 1]]
    rings = np.unique(np.concatenate([rings, [398, 400, 403, 509, 511, 514]]))
    ref1 = direct.direct_sum(geom, tab, tmax, x.astype(np.float64), out_rings=rings)
    assert frms(take_rings(geom, out, rings), ref1) <= 1e-6


# ------------------------------------------------------------------ several kernels, one forward transform --------

def test_multi_kernel_batching_shares_forward_ffts():
    """arkcos_convolve_multi (PAPER.md:19-21 wavelet banks, :233 asymmetric beams as O(10) radial terms): K = 4 kernels on one
    map pair; every kernel's result equals its own arkcos_convolve (same kernels on the same spectra) and the brute-force sum."""
    nside = 256
    geom = geometry.healpix_ring(nside)
    px = np.sqrt(4 * np.pi / geom.npix)
    kernels = [("gauss", inputs.gaussian_table(3.0 * px, 9.0 * px), 9.0 * px),
               ("mexhat_a", inputs.mexican_hat_table(1.6 * px, 8.0 * px), 8.0 * px),
               ("mexhat_b", inputs.mexican_hat_table(2.4 * px, 12.0 * px), 12.0 * px),
               ("disc", inputs.tophat_table(6.0 * px), 6.0 * px)]
    nmaps = 2
    x = inputs.white_noise_maps(geom.npix, 7, nmaps)
    plans = [arkcos.Plan(("healpix", nside), tab, tmax, arkcos.F32, max_nmaps=nmaps) for _, tab, tmax in kernels]
    d_in = torch.from_numpy(x).cuda()
    d_out = torch.full((len(plans), nmaps, geom.npix), float("nan"), device="cuda", dtype=torch.float32)
    st = torch.cuda.current_stream().cuda_stream
    arkcos.arkcos_convolve_multi(plans, d_in.data_ptr(), d_out.data_ptr(), nmaps, st)
    torch.cuda.synchronize()
    multi = d_out.cpu().numpy()
    assert np.isfinite(multi).all()
    rings = sample_rings(geom, extra=(nside - 2, nside - 1, nside, nside + 1, 3 * nside - 1), nrand=6, seed=5)
    eq_rings = np.array([r for r in rings if nside + 16 <= r <= 3 * nside - 18])
    for k, (name, tab, tmax) in enumerate(kernels):
        single, _ = gpu_convolve(("healpix", nside), tab, tmax, x, plan=plans[k])
        # same kernels on the same spectra: bit-equal wherever the result has a fixed summation order (belt rings, cap
        # rings whose grid spans one period); a cap ring whose grid spans several periods folds 3-4 terms per coefficient
        # with atomic additions, so there only to rounding
        belt = slice(int(geom.offset[nside + 16]), int(geom.offset[3 * nside - 17]))
        assert np.array_equal(multi[k][:, belt], single[:, belt]), name
        assert frms(multi[k], single) <= 1e-7, name
        ref = direct.direct_sum(geom, tab, tmax, x.astype(np.float64), out_rings=rings)
        got = take_rings(geom, multi[k], rings)
        if name == "disc":        # the Fourier scheme only suppresses ringing in the caps: exact in the belt
            ref_eq = direct.direct_sum(geom, tab, tmax, x.astype(np.float64), out_rings=eq_rings)
            assert frms(take_rings(geom, multi[k], eq_rings), ref_eq) <= 1e-6
        else:
            assert frms(got, ref) <= (3e-5 if name.startswith("mexhat") else 1e-5), name
    # argument errors: a plan twice, plans of different pixelizations
    with pytest.raises(arkcos.ArkcosError):
        arkcos.arkcos_convolve_multi([plans[0], plans[0]], d_in.data_ptr(), d_out.data_ptr(), nmaps, st)
    other = arkcos.Plan(("healpix", 128), kernels[0][1], kernels[0][2], arkcos.F32, max_nmaps=nmaps)
    with pytest.raises(arkcos.ArkcosError):
        arkcos.arkcos_convolve_multi([plans[0], other], d_in.data_ptr(), d_out.data_ptr(), nmaps, st)


@pytest.mark.parametrize("tc", [0, 1], ids=["tensor_cores", "fp32_only"])
def test_repeatability(tc):
    """Two calls on one plan give the same bits wherever the summation order is fixed: everywhere for a plan whose cap
    grids span a single period (here: all rings of 512+ pixels at nside 512 with a Gaussian), and on belt rings always.
    The fold of a grid spanning several periods (rings next to the poles; hard-edged kernels) adds 3-4 terms per
    coefficient atomically: equal to rounding only (documented in DESIGN.md section 5)."""
    nside = 512
    geom = geometry.healpix_ring(nside)
    px = np.sqrt(4 * np.pi / geom.npix)
    tab, tmax = inputs.gaussian_table(2.91 * px, 3 * 2.91 * px), 3 * 2.91 * px
    x = inputs.white_noise(geom.npix, 8)
    a, plan = gpu_convolve(("healpix", nside), tab, tmax, x, no_tensor_cores=tc)
    b, _ = gpu_convolve(("healpix", nside), tab, tmax, x, plan=plan)
    mp = plan_mprime(plan, geom, tmax)
    # belt rings use their own length as the grid; a cap ring's grid spans one period when M'/2 < N
    single = [r for r in range(geom.nrings) if geom.n[r] == 4 * nside or (geom.n[r] >= 512 and mp[r] // 2 < geom.n[r])]
    assert len(single) > geom.nrings * 0.85
    for r in single:
        assert np.array_equal(a[geom.ring_slice(r)], b[geom.ring_slice(r)]), r
    assert frms(a, b) <= 1e-7


def test_cuda_graph_replay_equals_direct_launches():
    """arkcos_convolve on a non-default stream captures the launches of the first call with a given (d_in, d_out, nmaps,
    stream) into a CUDA graph and replays it afterwards (options.no_cuda_graph = 0).  Replays, re-captures for new buffers
    (more than the four combinations the plan keeps) and a plan that launches directly must agree: bit-equal on the belt,
    to rounding elsewhere (multi-period fold); the first call's own result included."""
    nside, nmaps = 256, 2
    geom = geometry.healpix_ring(nside)
    px = np.sqrt(4 * np.pi / geom.npix)
    tab, tmax = inputs.gaussian_table(2.91 * px, 3 * 2.91 * px), 3 * 2.91 * px
    plan_g = arkcos.Plan(("healpix", nside), tab, tmax, arkcos.F32, max_nmaps=nmaps)
    plan_d = arkcos.Plan(("healpix", nside), tab, tmax, arkcos.F32, max_nmaps=nmaps, no_cuda_graph=1)
    belt = slice(int(geom.offset[nside + 16]), int(geom.offset[3 * nside - 17]))
    s = torch.cuda.Stream()
    outs = []
    with torch.cuda.stream(s):
        xs = [torch.from_numpy(inputs.white_noise_maps(geom.npix, 20 + k, nmaps)).cuda() for k in range(6)]
        os_ = [torch.full_like(x, float("nan")) for x in xs]
        ref = [torch.empty_like(x) for x in xs]
        for rep in range(3):                       # capture, replay, replay; six buffer pairs > four cached graphs
            for x, o in zip(xs, os_):
                plan_g.convolve(x.data_ptr(), o.data_ptr(), nmaps, s.cuda_stream)
            s.synchronize()
            outs.append([o.cpu().numpy() for o in os_])
        for x, r in zip(xs, ref):
            plan_d.convolve(x.data_ptr(), r.data_ptr(), nmaps, s.cuda_stream)
        s.synchronize()
    for k in range(6):
        r = ref[k].cpu().numpy()
        for rep in range(3):
            assert np.array_equal(outs[rep][k][:, belt], r[:, belt]), (rep, k)
            assert frms(outs[rep][k], r) <= 1e-7, (rep, k)
    # one map of a two-map plan through the same stream: another graph
    with torch.cuda.stream(s):
        o1 = torch.empty_like(xs[0][0])
        plan_g.convolve(xs[0][0].data_ptr(), o1.data_ptr(), 1, s.cuda_stream)
        plan_g.convolve(xs[0][0].data_ptr(), o1.data_ptr(), 1, s.cuda_stream)
        s.synchronize()
    assert frms(o1.cpu().numpy(), ref[0][0].cpu().numpy()) <= 1e-7
