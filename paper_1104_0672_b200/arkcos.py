"""Thin ctypes binding of libarkcos.so (include/arkcos.h): same names, argument marshalling only.

Every step of the convolution runs in the library's CUDA kernels.  There is no fallback: if the shared
library is missing or a call fails, an exception is raised.  torch is used by callers for device memory
and streams only; this module takes raw pointers (``tensor.data_ptr()``) and a raw ``cudaStream_t``.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, Structure, byref, c_char_p, c_double, c_float, c_int, c_int64, c_void_p

import numpy as np

ECP, HEALPIX_RING = 0, 1
F32, F64 = 0, 1
OK, INVALID_ARG, UNSUPPORTED, CUDA_ERROR, OUT_OF_MEMORY = 0, -1, -2, -3, -4
NO_ALLOC_SCRATCH_BYTES = 32 << 20      # ARKCOS_NO_ALLOC_SCRATCH_BYTES of include/arkcos.h

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libarkcos.so")


class Pixelization(Structure):
    _fields_ = [("kind", c_int), ("ntheta", c_int), ("nphi", c_int), ("nside", c_int)]


class Kernel(Structure):
    _fields_ = [("table", POINTER(c_double)), ("n", c_int), ("theta_max", c_double)]


class Options(Structure):
    _fields_ = [("variant", c_int), ("ell_nyquist", c_double), ("polar_oversample", c_int), ("max_nmaps", c_int),
                ("cache_kernel_rows", c_int), ("exact_caps", c_int), ("cache_kernel_spectra", c_int), ("no_tensor_cores", c_int),
                ("no_cuda_graph", c_int), ("reserved", c_int * 4)]


class ArkcosError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        lib = _lib()
        super().__init__(f"{where}: {lib.arkcos_strerror(status).decode()} ({status}): "
                         f"{lib.arkcos_last_error().decode()}")


_LIB = None

# every symbol include/arkcos.h declares: name -> (restype, argtypes)
SYMBOLS = {
    "arkcos_plan_create": (c_int, [POINTER(c_void_p), POINTER(Pixelization), POINTER(Kernel), c_int, POINTER(Options)]),
    "arkcos_plan_create_tables_only": (c_int, [POINTER(c_void_p), POINTER(Pixelization), POINTER(Kernel), c_int,
                                               POINTER(Options)]),
    "arkcos_convolve": (c_int, [c_void_p, c_void_p, c_void_p, c_int, c_void_p]),
    "arkcos_convolve_no_alloc": (c_int, [c_void_p, c_void_p, c_void_p, c_int, c_void_p]),
    "arkcos_convolve_multi": (c_int, [POINTER(c_void_p), c_int, c_void_p, c_void_p, c_int, c_void_p]),
    "arkcos_convolve_host": (c_int, [c_void_p, c_void_p, c_void_p, c_int, c_void_p]),
    "arkcos_convolve_host_async": (c_int, [c_void_p, c_void_p, c_void_p, c_int]),
    "arkcos_plan_synchronize": (c_int, [c_void_p]),
    "arkcos_plan_destroy": (c_int, [c_void_p]),
    "arkcos_plan_npix": (c_int64, [c_void_p]),
    "arkcos_plan_nrings": (c_int, [c_void_p]),
    "arkcos_plan_ring_info": (c_int, [c_void_p, c_int, POINTER(c_double), POINTER(c_int), POINTER(c_double),
                                      POINTER(c_int64), POINTER(c_int), POINTER(c_int), POINTER(c_int)]),
    "arkcos_plan_ell_nyquist": (c_double, [c_void_p]),
    "arkcos_plan_stats": (c_int, [c_void_p, POINTER(c_int64), POINTER(c_int64), POINTER(c_double), POINTER(c_double),
                                  POINTER(c_int64)]),
    "arkcos_plan_set_timing": (c_int, [c_void_p, c_int]),
    "arkcos_plan_get_timing": (c_int, [c_void_p, POINTER(c_float)]),
    "arkcos_plan_band_kernels": (c_int, [c_void_p, POINTER(c_int), POINTER(c_char_p), POINTER(c_double), POINTER(c_float)]),
    "arkcos_plan_fft_kernels": (c_int, [c_void_p, POINTER(c_int), POINTER(c_char_p), POINTER(c_double), POINTER(c_float),
                                        POINTER(c_float)]),
    "arkcos_plan_work_model": (c_int, [c_void_p, POINTER(c_double), POINTER(c_double), POINTER(c_double), POINTER(c_int)]),
    "arkcos_plan_tensor_cores": (c_int, [c_void_p, POINTER(c_int), POINTER(c_int)]),
    "arkcos_plan_launches_per_convolve": (c_int, [c_void_p]),
    "arkcos_probe_fp32_peak": (c_int, [POINTER(c_double), c_int]),
    "arkcos_kernel_legendre": (c_int, [POINTER(Kernel), c_double, c_double, c_int, POINTER(c_double)]),
    "arkcos_kernel_truncation_error": (c_int, [POINTER(Kernel), c_double, POINTER(c_double), c_int, POINTER(c_double),
                                               POINTER(c_double)]),
    "arkcos_kernel_choose_cut": (c_int, [POINTER(Kernel), POINTER(c_double), c_int, c_double, c_int, POINTER(c_double),
                                         POINTER(c_double), POINTER(c_double)]),
    "arkcos_kernel_choose_ell_nyquist": (c_int, [POINTER(Kernel), POINTER(c_double), c_int, c_double, POINTER(c_double)]),
    "arkcos_strerror": (c_char_p, [c_int]),
    "arkcos_last_error": (c_char_p, []),
}


def _lib():
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1104_0672_b200.build` "
                              "(there is no CPU fallback)")
        lib = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            f = getattr(lib, name)
            f.restype, f.argtypes = res, args
        _LIB = lib
    return _LIB


def _check(status: int, where: str):
    if status != OK:
        raise ArkcosError(status, where)


def arkcos_strerror(status: int) -> str:
    return _lib().arkcos_strerror(status).decode()


def arkcos_probe_fp32_peak(repeats: int = 10) -> float:
    v = c_double()
    _check(_lib().arkcos_probe_fp32_peak(byref(v), repeats), "arkcos_probe_fp32_peak")
    return v.value


def _kernel(table, theta_max):
    tab = np.ascontiguousarray(table, dtype=np.float64)
    return tab, Kernel(tab.ctypes.data_as(POINTER(c_double)), int(tab.shape[0]), float(theta_max))


def arkcos_kernel_legendre(table, theta_max: float, lmax: int, theta_lo: float = 0.0, theta_hi=None) -> np.ndarray:
    tab, k = _kernel(table, theta_max)
    out = np.empty(lmax + 1)
    _check(_lib().arkcos_kernel_legendre(byref(k), float(theta_lo), float(theta_max if theta_hi is None else theta_hi), int(lmax),
                                         out.ctypes.data_as(POINTER(c_double))), "arkcos_kernel_legendre")
    return out


def arkcos_kernel_truncation_error(table, theta_max: float, theta_cut: float, c_ell):
    """(sigma2, signal2) of Eq. 7 for lmax = len(c_ell) - 1."""
    tab, k = _kernel(table, theta_max)
    cl = np.ascontiguousarray(c_ell, dtype=np.float64)
    s2, sig = c_double(), c_double()
    _check(_lib().arkcos_kernel_truncation_error(byref(k), float(theta_cut), cl.ctypes.data_as(POINTER(c_double)), cl.shape[0] - 1,
                                                 byref(s2), byref(sig)), "arkcos_kernel_truncation_error")
    return s2.value, sig.value


def arkcos_kernel_choose_cut(table, theta_max: float, c_ell, rel_tol: float, ngrid: int = 256):
    """(theta_cut, sigma2, signal2)."""
    tab, k = _kernel(table, theta_max)
    cl = np.ascontiguousarray(c_ell, dtype=np.float64)
    cut, s2, sig = c_double(), c_double(), c_double()
    _check(_lib().arkcos_kernel_choose_cut(byref(k), cl.ctypes.data_as(POINTER(c_double)), cl.shape[0] - 1, float(rel_tol), int(ngrid),
                                           byref(cut), byref(s2), byref(sig)), "arkcos_kernel_choose_cut")
    return cut.value, s2.value, sig.value


def arkcos_kernel_choose_ell_nyquist(table, theta_max: float, c_ell, rel_tol: float) -> float:
    tab, k = _kernel(table, theta_max)
    cl = np.ascontiguousarray(c_ell, dtype=np.float64)
    v = c_double()
    _check(_lib().arkcos_kernel_choose_ell_nyquist(byref(k), cl.ctypes.data_as(POINTER(c_double)), cl.shape[0] - 1, float(rel_tol),
                                                   byref(v)), "arkcos_kernel_choose_ell_nyquist")
    return v.value


class Plan:
    """Owns an ``arkcos_plan*``.  ``pix`` is ("ecp", ntheta, nphi) or ("healpix", nside)."""

    def __init__(self, pix, table, theta_max: float, dtype=F32, *, variant=0, ell_nyquist=0.0, polar_oversample=0,
                 max_nmaps=1, cache_kernel_rows=0, exact_caps=0, cache_kernel_spectra=0, no_tensor_cores=0, no_cuda_graph=0, tables_only=False):
        lib = _lib()
        if pix[0] == "ecp":
            p = Pixelization(ECP, int(pix[1]), int(pix[2]), 0)
        elif pix[0] == "healpix":
            p = Pixelization(HEALPIX_RING, 0, 0, int(pix[1]))
        else:
            raise ValueError(pix)
        tab = np.ascontiguousarray(table, dtype=np.float64)
        k = Kernel(tab.ctypes.data_as(POINTER(c_double)), int(tab.shape[0]), float(theta_max))
        o = Options(int(variant), float(ell_nyquist), int(polar_oversample), int(max_nmaps), int(cache_kernel_rows),
                    int(exact_caps), int(cache_kernel_spectra), int(no_tensor_cores), int(no_cuda_graph))
        self._h = c_void_p()
        self.dtype = dtype
        self.max_nmaps = max(1, int(max_nmaps))
        create = lib.arkcos_plan_create_tables_only if tables_only else lib.arkcos_plan_create
        _check(create(byref(self._h), byref(p), byref(k), int(dtype), byref(o)), "arkcos_plan_create")

    # -- the three calls of the boundary
    def convolve(self, d_in: int, d_out: int, nmaps: int = 1, stream: int = 0):
        """arkcos_convolve: device pointers (ints), raw cudaStream_t (int)."""
        _check(_lib().arkcos_convolve(self._h, c_void_p(d_in), c_void_p(d_out), int(nmaps), c_void_p(stream)),
               "arkcos_convolve")

    def convolve_no_alloc(self, d_in: int, d_out: int, nmaps: int = 1, stream: int = 0):
        """arkcos_convolve_no_alloc: as convolve, scratch in the library's static device array (NO_ALLOC_SCRATCH_BYTES)."""
        _check(_lib().arkcos_convolve_no_alloc(self._h, c_void_p(d_in), c_void_p(d_out), int(nmaps), c_void_p(stream)),
               "arkcos_convolve_no_alloc")

    def convolve_host(self, h_in: int, h_out: int, nmaps: int = 1, stream: int = 0):
        _check(_lib().arkcos_convolve_host(self._h, c_void_p(h_in), c_void_p(h_out), int(nmaps), c_void_p(stream)),
               "arkcos_convolve_host")

    def convolve_host_async(self, h_in: int, h_out: int, nmaps: int = 1):
        """Streaming form: returns once upload, kernels and download are enqueued; finish with synchronize()."""
        _check(_lib().arkcos_convolve_host_async(self._h, c_void_p(h_in), c_void_p(h_out), int(nmaps)),
               "arkcos_convolve_host_async")

    def synchronize(self):
        _check(_lib().arkcos_plan_synchronize(self._h), "arkcos_plan_synchronize")

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h and _LIB is not None:   # _LIB is gone at interpreter exit
            _LIB.arkcos_plan_destroy(self._h)
            self._h = c_void_p()

    __del__ = destroy

    # -- queries
    @property
    def npix(self) -> int:
        return int(_lib().arkcos_plan_npix(self._h))

    @property
    def nrings(self) -> int:
        return int(_lib().arkcos_plan_nrings(self._h))

    @property
    def ell_nyquist(self) -> float:
        return float(_lib().arkcos_plan_ell_nyquist(self._h))

    def ring_info(self, ring: int) -> dict:
        th, n, p0, off = c_double(), c_int(), c_double(), c_int64()
        lo, hi, mp = c_int(), c_int(), c_int()
        _check(_lib().arkcos_plan_ring_info(self._h, ring, byref(th), byref(n), byref(p0), byref(off), byref(lo),
                                            byref(hi), byref(mp)), "arkcos_plan_ring_info")
        return dict(theta=th.value, n=n.value, phi0=p0.value, offset=off.value, band_lo=lo.value, band_hi=hi.value,
                    mprime=mp.value)

    def stats(self) -> dict:
        rp, rs, ws = c_int64(), c_int64(), c_int64()
        mf, ff = c_double(), c_double()
        _check(_lib().arkcos_plan_stats(self._h, byref(rp), byref(rs), byref(mf), byref(ff), byref(ws)),
               "arkcos_plan_stats")
        return dict(ring_pairs=rp.value, row_samples=rs.value, mac_flops=mf.value, fft_flops=ff.value,
                    workspace_bytes=ws.value)

    def tensor_cores(self) -> dict:
        """Whether the band step runs on the tensor cores, with the blocks per launch class and the blocks one SM holds."""
        blocks = (c_int * 3)()
        res = c_int()
        used = _lib().arkcos_plan_tensor_cores(self._h, blocks, byref(res))
        if used < 0:
            raise ArkcosError(used, "arkcos_plan_tensor_cores")
        return dict(used=bool(used), blocks=list(blocks), resident_per_sm=res.value)

    @property
    def launches_per_convolve(self) -> int:
        return int(_lib().arkcos_plan_launches_per_convolve(self._h))

    def set_timing(self, enable):
        _check(_lib().arkcos_plan_set_timing(self._h, int(enable)), "arkcos_plan_set_timing")

    def band_kernels(self, with_timing: bool = False):
        """[(name, model_flops, last_ms or None)] of the band kernels (timing needs set_timing(2) before the call)."""
        n = c_int()
        names = (c_char_p * 9)()
        fl = (c_double * 9)()
        ms = (c_float * 9)()
        _check(_lib().arkcos_plan_band_kernels(self._h, byref(n), names, fl, ms if with_timing else None),
               "arkcos_plan_band_kernels")
        return [(names[k].decode(), fl[k], ms[k] if with_timing else None) for k in range(n.value)]

    def fft_kernels(self, with_timing: bool = False):
        """[(name, pixels, forward_ms or None, inverse_ms or None)] of the ring-FFT launches (timing needs set_timing(2))."""
        n = c_int()
        names = (c_char_p * 9)()
        px = (c_double * 9)()
        f, i = (c_float * 9)(), (c_float * 9)()
        _check(_lib().arkcos_plan_fft_kernels(self._h, byref(n), names, px, f if with_timing else None, i if with_timing else None),
               "arkcos_plan_fft_kernels")
        return [(names[k].decode(), px[k], f[k] if with_timing else None, i[k] if with_timing else None) for k in range(n.value)]

    def work_model(self) -> dict:
        a, b, c, m = c_double(), c_double(), c_double(), c_int()
        _check(_lib().arkcos_plan_work_model(self._h, byref(a), byref(b), byref(c), byref(m)), "arkcos_plan_work_model")
        return dict(band_pair_modes=a.value, fft_flops_min=b.value, tensor_flops=c.value, memsets_per_map=m.value)

    def get_timing(self):
        ms = (c_float * 4)()
        _check(_lib().arkcos_plan_get_timing(self._h, ms), "arkcos_plan_get_timing")
        return dict(rows=ms[0], fft_forward=ms[1], band=ms[2], fft_inverse=ms[3])


def arkcos_convolve_multi(plans, d_in: int, d_out: int, nmaps: int = 1, stream: int = 0):
    """arkcos_convolve_multi: d_out is [len(plans)][nmaps][npix] on the device."""
    arr = (c_void_p * len(plans))(*[p._h for p in plans])
    _check(_lib().arkcos_convolve_multi(arr, len(plans), c_void_p(d_in), c_void_p(d_out), int(nmaps), c_void_p(stream)),
           "arkcos_convolve_multi")


def convolve_torch(plan: Plan, x, out=None):
    """Convenience for tests/bench: x is a CUDA torch tensor [npix] or [nmaps, npix] of the plan's dtype."""
    import torch
    assert x.is_cuda and x.is_contiguous()
    nmaps = 1 if x.dim() == 1 else x.shape[0]
    if out is None:
        out = torch.empty_like(x)
    plan.convolve(x.data_ptr(), out.data_ptr(), nmaps, torch.cuda.current_stream().cuda_stream)
    return out
