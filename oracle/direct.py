"""Oracle #1: the brute-force direct sum, Eq. 6 with pixel weights.

    out(p) = sum_{q : gamma_pq < theta_max} K(gamma_pq) in(q) Omega_q

Two restatements of the same definition live here:

* ``direct_sum``        -- calls ``direct_sum.c`` (plain C, OpenMP over output rings), used for parity and
                           as the timed CPU baseline.  Distance via Eq. 9's haversine form.
* ``direct_sum_numpy``  -- a dozen lines of numpy, distance via arccos of the dot product of unit vectors
                           (the literal "p.q" of PAPER.md:51).  Only for tiny grids; it exists to pin the C
                           routine to something that does not share its formula.

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

from .geometry import RingGeometry

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None


def build(force: bool = False) -> str:
    """Compile direct_sum.c with gcc into oracle/liboracle_direct.so (building the checker is not using it)."""
    src = os.path.join(_HERE, "direct_sum.c")
    so = os.path.join(_HERE, "liboracle_direct.so")
    if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-fopenmp", "-o", so, src, "-lm"])
    return so


def _lib():
    global _LIB
    if _LIB is None:
        lib = ctypes.CDLL(build())
        f = lib.arkcos_oracle_direct_sum
        P = ctypes.c_void_p
        f.argtypes = [ctypes.c_int, P, P, P, P, P, P, ctypes.c_int, ctypes.c_double,
                      P, ctypes.c_int, ctypes.c_int64, P, ctypes.c_int, P, ctypes.c_int]
        f.restype = ctypes.c_int
        _LIB = lib
    return _LIB


def kernel_lerp(table: np.ndarray, theta_max: float, gamma: np.ndarray) -> np.ndarray:
    """K(gamma) by linear interpolation in theta on table[t] = K(t theta_max / (n-1))."""
    table = np.asarray(table, float)
    n = table.shape[0]
    u = np.asarray(gamma, float) * (n - 1) / theta_max
    t = np.clip(np.floor(u).astype(np.int64), 0, n - 2)
    return table[t] + (u - t) * (table[t + 1] - table[t])


def direct_sum(geom: RingGeometry, table, theta_max: float, inp, out_rings=None, nthreads: int = 0,
               return_threads: bool = False):
    """Eq. 6 on the rings ``out_rings`` (default: all).  inp: [npix] or [nmaps, npix].

    Returns [.., sum of ring lengths] with the requested rings concatenated in the order given.
    """
    inp = np.asarray(inp, dtype=np.float64)
    squeeze = inp.ndim == 1
    inp2 = np.ascontiguousarray(inp.reshape(-1, geom.npix))
    nmaps = inp2.shape[0]
    if out_rings is None:
        out_rings = np.arange(geom.nrings)
    out_rings = np.ascontiguousarray(out_rings, dtype=np.int32)
    nout = int(geom.n[out_rings].sum()) if out_rings.size else 0
    out = np.zeros((nmaps, nout))
    table = np.ascontiguousarray(table, dtype=np.float64)
    th = np.ascontiguousarray(geom.theta)
    n = np.ascontiguousarray(geom.n, dtype=np.int64)
    p0 = np.ascontiguousarray(geom.phi0)
    om = np.ascontiguousarray(geom.omega)
    off = np.ascontiguousarray(geom.offset, dtype=np.int64)
    rc = _lib().arkcos_oracle_direct_sum(
        geom.nrings, th.ctypes.data, n.ctypes.data, p0.ctypes.data, om.ctypes.data, off.ctypes.data,
        table.ctypes.data, int(table.shape[0]), float(theta_max),
        inp2.ctypes.data, nmaps, geom.npix, out_rings.ctypes.data, int(out_rings.size),
        out.ctypes.data, int(nthreads))
    if rc < 0:
        raise ValueError(f"arkcos_oracle_direct_sum failed: {rc}")
    res = out[0] if squeeze else out
    return (res, rc) if return_threads else res


def unit_vectors(geom: RingGeometry) -> np.ndarray:
    v = np.empty((geom.npix, 3))
    for i in range(geom.nrings):
        ph = geom.phi(i)
        st, ct = np.sin(geom.theta[i]), np.cos(geom.theta[i])
        v[geom.ring_slice(i)] = np.stack([st * np.cos(ph), st * np.sin(ph), np.full_like(ph, ct)], axis=1)
    return v


def direct_sum_numpy(geom: RingGeometry, table, theta_max: float, inp) -> np.ndarray:
    """Eq. 6 literally: gamma = arccos(n_p . n_q), dense npix x npix.  Tiny grids only."""
    if geom.npix > 6000:
        raise ValueError("direct_sum_numpy is for tiny grids")
    v = unit_vectors(geom)
    gamma = np.arccos(np.clip(v @ v.T, -1.0, 1.0))
    w = np.where(gamma < theta_max, kernel_lerp(table, theta_max, np.minimum(gamma, theta_max)), 0.0)
    omega_q = np.repeat(geom.omega, geom.n)
    inp = np.asarray(inp, float)
    out = (inp.reshape(-1, geom.npix) * omega_q[None, :]) @ w.T      # out[map, p] = sum_q w[p, q] Omega_q in[map, q]
    return out[0] if inp.ndim == 1 else out
