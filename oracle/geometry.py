"""Ring geometry of the pixelizations the paper's algorithm runs on (oracle side, fp64).

"Our algorithm works for any pixelization where pixels are grouped into isolatitude rings"
(PAPER.md:9).  A pixelization is therefore described ring by ring: colatitude theta_i, number of
pixels N_i, azimuth of the first pixel phi0_i (pixel k sits at phi0_i + 2 pi k / N_i), pixel weight
Omega_i (solid angle of one pixel of the ring) and the index of the ring's first pixel in the map.

* ECP (equidistant cylindrical projection): N_theta rings at
  theta_i = (i + 1/2) pi / N_theta, N_phi pixels each at phi_k = 2 pi k / N_phi,
  Omega_i = sin(theta_i) (pi / N_theta) (2 pi / N_phi)        (BASELINE.json configs[0]).
* HEALPix ring scheme: north cap rings n = 1 .. nside-1 with 4 n pixels,
  2 nside + 1 equatorial rings with 4 nside pixels, south cap by mirror; every cap ring is shifted by
  phi0 = pi / (4 n), every other equatorial ring by pi / (4 nside).  The ring
  colatitudes are not printed in the paper; they are the published definition it cites
  (Gorski et al. 2005):  z = 1 - n^2 / (3 nside^2) in the caps,
  z = 4/3 - 2 i / (3 nside) for nside <= i <= 3 nside.  Omega = 4 pi / (12 nside^2).

This file is test infrastructure (see oracle/__init__.py).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class RingGeometry:
    kind: str              # "ecp" | "healpix_ring"
    theta: np.ndarray      # [R] colatitude of ring i (radians), north to south
    n: np.ndarray          # [R] int64, pixels on ring i
    phi0: np.ndarray       # [R] azimuth of pixel 0 of ring i
    omega: np.ndarray      # [R] solid angle of one pixel of ring i
    offset: np.ndarray     # [R+1] int64, map index of pixel 0 of ring i; offset[R] = npix

    @property
    def nrings(self) -> int:
        return int(self.theta.shape[0])

    @property
    def npix(self) -> int:
        return int(self.offset[-1])

    def ring_slice(self, i: int) -> slice:
        return slice(int(self.offset[i]), int(self.offset[i + 1]))

    def phi(self, i: int) -> np.ndarray:
        """Azimuths of the pixels of ring i."""
        return self.phi0[i] + 2.0 * np.pi * np.arange(int(self.n[i])) / float(self.n[i])


def _finish(kind, theta, n, phi0, omega) -> RingGeometry:
    n = np.asarray(n, dtype=np.int64)
    offset = np.zeros(n.shape[0] + 1, dtype=np.int64)
    np.cumsum(n, out=offset[1:])
    return RingGeometry(kind, np.asarray(theta, float), n, np.asarray(phi0, float),
                        np.asarray(omega, float), offset)


def ecp(ntheta: int, nphi: int) -> RingGeometry:
    """ECP grid, BASELINE.json configs[0..1]."""
    i = np.arange(ntheta)
    theta = (i + 0.5) * np.pi / ntheta
    omega = np.sin(theta) * (np.pi / ntheta) * (2.0 * np.pi / nphi)
    return _finish("ecp", theta, np.full(ntheta, nphi), np.zeros(ntheta), omega)


def healpix_ring(nside: int) -> RingGeometry:
    """HEALPix ring scheme, rings i = 1 .. 4 nside - 1 north to south (stored 0-based)."""
    R = 4 * nside - 1
    theta = np.empty(R)
    n = np.empty(R, dtype=np.int64)
    phi0 = np.empty(R)
    for idx in range(R):
        i = idx + 1                       # the paper's / HEALPix's 1-based ring number
        if i < nside:                     # north polar cap, ring n = i has 4 n pixels
            # z = 1 - i^2 / (3 nside^2);  theta = arccos z = 2 asin(sqrt((1 - z) / 2))  (no cancellation)
            theta[idx] = 2.0 * np.arcsin(i / (np.sqrt(6.0) * nside))
            n[idx] = 4 * i
            phi0[idx] = np.pi / (4.0 * i)
        elif i <= 3 * nside:              # equatorial region, 2 nside + 1 rings of 4 nside pixels
            z = 4.0 / 3.0 - 2.0 * i / (3.0 * nside)
            theta[idx] = np.arccos(z)
            n[idx] = 4 * nside
            phi0[idx] = np.pi / (4.0 * nside) if (i - nside) % 2 == 0 else 0.0
        else:                             # south polar cap: mirror image of ring 4 nside - i
            ii = 4 * nside - i
            theta[idx] = np.pi - 2.0 * np.arcsin(ii / (np.sqrt(6.0) * nside))
            n[idx] = 4 * ii
            phi0[idx] = np.pi / (4.0 * ii)
    omega = np.full(R, 4.0 * np.pi / (12.0 * nside * nside))
    return _finish("healpix_ring", theta, n, phi0, omega)


def band(geom: RingGeometry, i: int, theta_max: float) -> np.ndarray:
    """Input rings that can reach output ring i: |theta_i - theta_j| < theta_max.

    The angular distance between two points is never smaller than their colatitude difference, so no
    other ring holds a pixel with gamma < theta_max ('Band').
    """
    return np.nonzero(np.abs(geom.theta - geom.theta[i]) < theta_max)[0]
