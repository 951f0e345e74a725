"""Oracle #2: the paper's hybrid scheme, ring by ring, in fp64 with direct DFTs.

"convolving along isolatitude rings ... by means of the convolution theorem, and integrating in the
longitudinal direction in pixel space".  The steps are the paper's
with the anti-ringing modifications of PAPER.md:219 (variant "B", the default) or without them
(variant "A"); the paper's own CPU implementation "mostly for validation purposes" is the
model.  TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

Notation: output ring i, input ring j, N_i pixels on ring i, delta_ij = phi0_i - phi0_j,
kappa_ij(psi) = K(gamma(theta_i, theta_j, psi)) [gamma < theta_max] (Eq. 9),
M_ij = length of the phi grid the kernel row is sampled on.

Step 1  B_j[m] = sum_l in(j,l) exp(-2 pi i m l / N_j),  m = 0 .. N_j-1.
Step 2 for every j in the band of i:
   class E, N_i == N_j == N_max (both rings have the full length: every ECP ring, the HEALPix equatorial rings; DESIGN.md
        reading R11): M_ij = N_i and the row is sampled *with* the offset ("substitute
        cos(phi) with cos(phi - phi0)"): kappa[d] = kappa_ij(delta_ij + 2 pi d / M),
        kt[m] = sum_d kappa[d] exp(-2 pi i m d / M); no phase factor.  This is an exact circulant
        identity (the ECP case of PAPER.md:219 and the HEALPix equatorial region).
   class C, every other pair (a polar-cap ring is involved, including a cap ring paired with itself): M_ij = M'_i (reading R10), the row is
        sampled at delta = 0 and both rings are re-origined by Eq. 8:
        kt[m] <- kt[m] exp(i m delta_ij) for signed |m| < M/2, and the +-M/2 bins carry half the
        Nyquist coefficient each.
   C_i[m] += Omega_j kt[m] B_j[m mod N_j]         variant B: periodic extension ("duplicate")
                                                   variant A: B_j := 0 for |m| > N_j/2 ("zero-pad")
Step 3  variant B: D_i[m mod N_i] += C_i[m] ("add the super-Nyquist modes to the sub-Nyquist modes",
        PAPER.md:219); variant A: keep |m| <= N_i/2 ("truncate ... to the Nyquist frequency").
Step 4  out(i,k) = (1/M) Re sum_m' D_i[m'] exp(2 pi i m' k / N_i).

Where the normalisation comes from: kappa(delta + psi) ~ (1/M) sum_m kt[m] exp(i m psi) (the trigonometric
interpolant through the M samples) put into  out(i,k) = Omega_j sum_l kappa(delta_ij + 2 pi k/N_i - 2 pi l/N_j) in(j,l).
"""
from __future__ import annotations

import numpy as np

from .geometry import RingGeometry, band
from .direct import kernel_lerp

DIRECT_DFT_MAX = 1024     # above this length the DFT step calls the library FFT (same definition)


def dft(x: np.ndarray, sign: int = -1) -> np.ndarray:
    """X[m] = sum_l x[l] exp(sign 2 pi i m l / N) along the last axis, unnormalised."""
    x = np.asarray(x)
    N = x.shape[-1]
    if N > DIRECT_DFT_MAX:
        return np.fft.fft(x, axis=-1) if sign < 0 else np.fft.ifft(x, axis=-1) * N
    ml = np.outer(np.arange(N), np.arange(N)) % N          # exact integer phase index
    W = np.exp(sign * 2j * np.pi * ml / N)
    return x @ W.T


def squared_chord(theta_i: float, theta_j: float, psi: np.ndarray) -> np.ndarray:
    """x = 2 - 2 cos(gamma), Eq. 9 in haversine form."""
    A = 4.0 * np.sin(0.5 * (theta_i - theta_j)) ** 2
    Bc = 4.0 * np.sin(theta_i) * np.sin(theta_j)
    return A + Bc * np.sin(0.5 * psi) ** 2


def kernel_row(theta_i, theta_j, psi, table, theta_max) -> np.ndarray:
    """kappa_ij(psi): the tabulated profile at the angular distance of Eq. 9, zero outside the support."""
    x = squared_chord(theta_i, theta_j, np.asarray(psi, float))
    gamma = 2.0 * np.arcsin(np.minimum(1.0, 0.5 * np.sqrt(x)))
    return np.where(gamma < theta_max, kernel_lerp(table, theta_max, np.minimum(gamma, theta_max)), 0.0)


def mprime_resolving(geom: RingGeometry, theta_max: float, ell_nyq: float) -> np.ndarray:
    """Shortest class-C grid per output ring that resolves wavenumber ell_nyq along the ring (reading R10).

    The paper samples every kernel row on 4 nside points.  Under reading R10 the grid of a
    cap-touching row resolves wavenumber ell_nyq along the ring:  M'_i >= 2 ceil(ell_nyq * smax_i),
    smax_i = max sin(theta) over ring i and its band, never below 8.  Any even M'_i at or above this bound is a valid
    setting of the scheme; which one a plan uses is the plan's parameter ("run it with the plan's
    settings"), passed to hybrid_convolve as ``mprime``.
    """
    out = np.empty(geom.nrings, dtype=np.int64)
    s = np.sin(geom.theta)
    for i in range(geom.nrings):
        smax = s[band(geom, i, theta_max)].max()
        out[i] = max(8, 2 * int(np.ceil(ell_nyq * smax)))
    return out


def is_class_e(geom, i, j) -> bool:
    """Both rings have the full ring length, so their pixels share one phi grid up to the half-pixel offset."""
    nmax = int(geom.n.max())
    return int(geom.n[i]) == nmax and int(geom.n[j]) == nmax


def pair_spectrum(geom, i, j, table, theta_max, M):
    """(signed mode numbers m, kt[m] incl. Eq. 8 phases) of ring pair (i, j) on an M-point grid."""
    delta = geom.phi0[i] - geom.phi0[j]
    d = np.arange(M)
    if is_class_e(geom, i, j) and M == geom.n[i]:                # class E: offset-aware sampling
        kap = kernel_row(geom.theta[i], geom.theta[j], delta + 2.0 * np.pi * d / M, table, theta_max)
        phase_delta = 0.0
    else:                                                         # class C: delta = 0, Eq. 8 on both rings
        kap = kernel_row(geom.theta[i], geom.theta[j], 2.0 * np.pi * d / M, table, theta_max)
        phase_delta = delta
    kt = dft(kap.astype(complex))                                 # kt[m], m = 0 .. M-1
    half = M // 2
    if M % 2 == 0:
        m = np.arange(-half, half + 1)                            # both Nyquist bins, half weight each
        vals = kt[m % M] * np.exp(1j * m * phase_delta)
        vals[0] *= 0.5
        vals[-1] *= 0.5
    else:
        m = np.arange(-half, half + 1)
        vals = kt[m % M] * np.exp(1j * m * phase_delta)
    return m, vals


def hybrid_convolve(geom: RingGeometry, table, theta_max: float, inp, variant: str = "B",
                    mprime=None, out_rings=None) -> np.ndarray:
    """The hybrid scheme on rings ``out_rings`` (default all).  inp: [npix] or [nmaps, npix].

    mprime: int or [R] array, the class-C grid length per *output* ring (default 4 nside-like:
    the longest ring, which is the paper's choice).
    """
    inp = np.asarray(inp, float)
    squeeze = inp.ndim == 1
    maps = inp.reshape(-1, geom.npix)
    nmaps = maps.shape[0]
    if out_rings is None:
        out_rings = np.arange(geom.nrings)
    if mprime is None:
        mprime = int(geom.n.max())
    mprime = np.broadcast_to(np.asarray(mprime, dtype=np.int64), (geom.nrings,))
    table = np.asarray(table, float)

    spec_cache = {}

    def ring_spectrum(j):                                         # step 1
        if j not in spec_cache:
            spec_cache[j] = dft(maps[:, geom.ring_slice(j)].astype(complex))
        return spec_cache[j]

    pieces = []
    for i in out_rings:
        i = int(i)
        Ni = int(geom.n[i])
        D = np.zeros((nmaps, Ni), dtype=complex)
        for j in band(geom, i, theta_max):
            j = int(j)
            Nj = int(geom.n[j])
            M = Ni if is_class_e(geom, i, j) else int(mprime[i])
            m, kt = pair_spectrum(geom, i, j, table, theta_max, M)        # step 2
            Bj = ring_spectrum(j)[:, m % Nj]
            if variant == "A":
                # zero-padded B_j: nothing above ring j's Nyquist frequency, whose own bin is
                # split half/half between +N_j/2 and -N_j/2 when the grid extends past it; output truncated
                # at ring i's Nyquist frequency
                wA = (np.abs(m) < Nj / 2).astype(float)
                wA[np.abs(m) * 2 == Nj] = 0.5 if M > Nj else 1.0
                wA[np.abs(m) > Ni // 2] = 0.0
                Bj = Bj * wA
            elif variant != "B":
                raise ValueError("variant must be 'A' or 'B'")
            C = geom.omega[j] * kt[None, :] * Bj / M
            np.add.at(D, (slice(None), m % Ni), C)                         # step 3 (fold)
        pieces.append(dft(D, sign=+1).real)                                # step 4
    out = np.concatenate(pieces, axis=1) if pieces else np.zeros((nmaps, 0))
    return out[0] if squeeze else out
