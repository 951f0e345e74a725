"""CPU oracle for the ARKCoS hybrid ring convolution (Elsner & Wandelt, arXiv:1104.0672).

TEST INFRASTRUCTURE ONLY.  Nothing under ``oracle/`` is part of the product: only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import,
call, link or execute it.  It shares no code with the CUDA path in ``paper_1104_0672_b200/`` and never
imports it.  Everything here is fp64, slow, and written to be checked against the paper by eye.

Modules
-------
geometry    ring geometry of the two pixelizations (ECP; HEALPix ring scheme)
direct      oracle #1, the brute-force direct sum  s_p = sum_q K(p.q) r_q Omega_q  (Eq. 6)
hybrid      oracle #2, the paper's ring-by-ring Fourier scheme with direct DFTs
legendre    Legendre transform of a profile (Eq. 2) and the truncation-error estimate (Eq. 7)

Parity pins (tests/test_oracle_*.py, ``-m "not gpu"``): point-source response, ECP circulant identity
(#2 == #1 to 1e-13), Jacobi-Anger closed form of a kernel row, linearity / phi-shift / mirror /
self-adjointness, Funk-Hecke for l = 0, 1, an independent arccos(dot) restatement of Eq. 6; for legendre the
closed-form K_l of a disc / annulus, the flat-sky Gaussian window, completeness, and Eq. 7 against the brute-force
sum on white noise (tests/test_oracle_legendre.py).
"""
from . import geometry, direct, hybrid, legendre  # noqa: F401
