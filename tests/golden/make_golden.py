"""Writes tests/golden/point_source_hp8.txt by calling ONLY oracle/ (never the CUDA path):
the response of oracle #1 to a unit point source on HEALPix nside 8 with a Gaussian profile.
Run:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import geometry, direct  # noqa: E402

DEG = np.pi / 180
NSIDE, FWHM, TMAX, NTAB, Q0 = 8, 15 * DEG, 30 * DEG, 65536, 200


def table():
    sigma = FWHM / 2.3548
    t = np.arange(NTAB) * (TMAX / (NTAB - 1))
    return np.exp(-0.5 * (t / sigma) ** 2)


if __name__ == "__main__":
    geom = geometry.healpix_ring(NSIDE)
    x = np.zeros(geom.npix)
    x[Q0] = 1.0
    out = direct.direct_sum(geom, table(), TMAX, x)
    nz = np.nonzero(out)[0]
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "point_source_hp8.txt")
    with open(path, "w") as f:
        f.write("# oracle #1 (Eq. 6, PAPER.md:79): response to a unit source at pixel 200, HEALPix nside 8 (ring order),\n"
                "# Gaussian FWHM 15 deg cut at 30 deg, 65536-point table.  Written by tests/golden/make_golden.py.\n"
                "# pixel  out\n")
        for p in nz:
            f.write(f"{p} {out[p]:.17e}\n")
    print(path, nz.size)
