"""arkcos_convolve_no_alloc (include/arkcos.h): the convolution with its spectra and pole scratch in the library's static
device array must equal arkcos_convolve, the existing path, on calls in a row that share that array.

Collected last on purpose (the file name sorts after the other test files): the suite runs with pytest -x.
Tolerances are those of tests/test_parity_gpu.py between two runs of the CUDA path: fp32 fractional RMS <= 1e-7
(the fold of multi-period cap rings adds atomically, in any order), fp64 max-norm <= 1e-12.
"""
import numpy as np
import pytest

from paper_1104_0672_b200 import arkcos, inputs

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def frms(a, b):
    a, b = a.double(), b.double()
    return float(torch.sqrt(((a - b) ** 2).sum() / (b ** 2).sum()))


def stream():
    return torch.cuda.current_stream().cuda_stream


def test_no_alloc_entry_point_equals_existing_path_on_calls_in_a_row():
    nside, nmaps = 128, 2
    npix = 12 * nside * nside
    fwhm = 2.0 * np.sqrt(4 * np.pi / npix)
    tmax = 3 * fwhm
    tab = inputs.gaussian_table(fwhm, tmax)
    plan = arkcos.Plan(("healpix", nside), tab, tmax, arkcos.F32, max_nmaps=nmaps)
    names = [name for name, flops, _ in plan.band_kernels() if flops > 0]
    assert any("band_mac_pole_fold_kernel" in n for n in names), names     # the two pole launches and their scratch are on the path
    # a second plan of another pixelization, dtype and size: its call in between leaves its own data in the shared array
    c1 = inputs.config(1)
    tab1, tmax1 = inputs.kernel_table(c1), c1["theta_max"]
    plan64 = arkcos.Plan(c1["pix"], tab1, tmax1, arkcos.F64)
    npix64 = plan64.npix

    xs = [torch.from_numpy(inputs.white_noise_maps(npix, 21 + k, nmaps)).cuda() for k in range(3)]
    y = torch.from_numpy(inputs.white_noise(npix64, 1, dtype=np.float64)).cuda()
    refs = [torch.full_like(x, float("nan")) for x in xs]
    outs = [torch.full_like(x, float("nan")) for x in xs]
    ref64, out64 = torch.full_like(y, float("nan")), torch.full_like(y, float("nan"))
    for x, r in zip(xs, refs):
        plan.convolve(x.data_ptr(), r.data_ptr(), nmaps, stream())
    plan64.convolve(y.data_ptr(), ref64.data_ptr(), 1, stream())
    torch.cuda.synchronize()
    assert all(bool(torch.isfinite(r).all()) for r in refs) and bool(torch.isfinite(ref64).all())

    # two calls in a row on one stream, no synchronisation in between; then the other plan; then the first again
    plan.convolve_no_alloc(xs[0].data_ptr(), outs[0].data_ptr(), nmaps, stream())
    plan.convolve_no_alloc(xs[1].data_ptr(), outs[1].data_ptr(), nmaps, stream())
    plan64.convolve_no_alloc(y.data_ptr(), out64.data_ptr(), 1, stream())
    plan.convolve_no_alloc(xs[2].data_ptr(), outs[2].data_ptr(), nmaps, stream())
    torch.cuda.synchronize()
    for k in range(3):
        assert bool(torch.isfinite(outs[k]).all())
        assert frms(outs[k], refs[k]) <= 1e-7, k
    assert float((out64 - ref64).abs().max() / ref64.abs().max()) <= 1e-12

    # the calls allocate nothing on the device: free memory is what it was (every kernel has run once by now)
    free_before = torch.cuda.mem_get_info()[0]
    for k in range(2):
        outs[k].fill_(float("nan"))
        plan.convolve_no_alloc(xs[k].data_ptr(), outs[k].data_ptr(), nmaps, stream())
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before
    for k in range(2):
        assert frms(outs[k], refs[k]) <= 1e-7, k

    # the existing path is untouched by all this
    again = torch.full_like(xs[0], float("nan"))
    plan.convolve(xs[0].data_ptr(), again.data_ptr(), nmaps, stream())
    torch.cuda.synchronize()
    assert frms(again, refs[0]) <= 1e-7


def test_no_alloc_entry_point_refuses_what_does_not_fit():
    nside, nmaps = 128, 24                        # 2 x 24 maps x 0.79 MB of spectra > 32 MiB
    npix = 12 * nside * nside
    fwhm = 2.0 * np.sqrt(4 * np.pi / npix)
    tab = inputs.gaussian_table(fwhm, 3 * fwhm)
    plan = arkcos.Plan(("healpix", nside), tab, 3 * fwhm, arkcos.F32, max_nmaps=nmaps)
    x = torch.from_numpy(inputs.white_noise_maps(npix, 31, nmaps)).cuda()
    out = torch.full_like(x, float("nan"))
    with pytest.raises(arkcos.ArkcosError) as e:
        plan.convolve_no_alloc(x.data_ptr(), out.data_ptr(), nmaps, stream())
    assert e.value.status == arkcos.INVALID_ARG
    assert "ARKCOS_NO_ALLOC_SCRATCH_BYTES" in str(e.value) and str(arkcos.NO_ALLOC_SCRATCH_BYTES) in str(e.value)
    torch.cuda.synchronize()
    assert bool(torch.isnan(out).all())           # nothing was enqueued
    # the same plan with a number of maps that fits is served
    ref = torch.full_like(x[:4], float("nan"))
    plan.convolve(x.data_ptr(), ref.data_ptr(), 4, stream())
    plan.convolve_no_alloc(x.data_ptr(), out.data_ptr(), 4, stream())
    torch.cuda.synchronize()
    assert frms(out[:4], ref) <= 1e-7
    # argument checks of the existing entry point hold here too
    with pytest.raises(arkcos.ArkcosError):
        plan.convolve_no_alloc(x.data_ptr(), x.data_ptr(), 1, stream())
