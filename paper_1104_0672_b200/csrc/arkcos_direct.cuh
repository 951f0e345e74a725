// Exact direct-space sum on selected output rings (option exact_caps): Eq. 6 of the paper with compact-support pruning
// (the paper itself recomputes pixels by direct sum where the Fourier scheme is not good enough,
// PAPER.md:178).  Used for the HEALPix polar-cap rings and the equatorial rings whose band reaches into a cap: there the
// hybrid scheme only "suppresses" ringing for discontinuous or hard-cut kernels, the direct sum has none.
//
//   out(i,k) = sum_{j in band(i)} Omega_j sum_{l : gamma < theta_max} K(gamma) in(j,l),
//   x = 2 - 2 cos(gamma) = A_ij + B_ij sin^2(dphi / 2)   (Eq. 9),  dphi = phi_jl - phi_ik.
//
// One thread owns output pixel k of northern ring i AND of its mirror image (same weights), for NM maps at
// once (the weights do not depend on the map).  Distances and the profile interpolation are double precision, as in the
// kernel-row generator; the accumulators have the plan's precision.
#pragma once
#include "arkcos_band.cuh"

namespace arkcos {

constexpr int kDirectThreads = 128;

// grid = (blocks of kDirectThreads pixels over the listed rings, map chunks); items: {index into ring_list, first pixel}
template <class T, int NM>
__global__ void __launch_bounds__(kDirectThreads)
direct_rings_kernel(const BandItem* __restrict__ items, const NorthRec* __restrict__ north,
                    const PairRec* __restrict__ pairs, const RingRec* __restrict__ rings, int R,
                    const double* __restrict__ table, int ntab, double theta_max, double xmax,
                    const T* __restrict__ in, T* __restrict__ out, int64_t npix, int nmaps)
{
    const BandItem it = items[blockIdx.x];
    const int i = it.ring, iS = R - 1 - i;
    const RingRec ri = rings[i], riS = rings[iS];
    const int k = it.m0 + (int)threadIdx.x;
    if (k >= ri.n) return;
    const int map0 = (int)blockIdx.y * NM;
    const double tscale = (double)(ntab - 1) / theta_max;
    const double uk = ((double)k + (ri.shifted ? 0.5 : 0.0)) / (double)ri.n;       // azimuth of the pixel in turns
    T accN[NM], accS[NM];
#pragma unroll
    for (int q = 0; q < NM; ++q) { accN[q] = (T)0; accS[q] = (T)0; }
    const NorthRec nr = north[i];
    for (int p = nr.pair_lo; p < nr.pair_hi; ++p) {
        const PairRec pr = pairs[p];
        const RingRec rj = rings[pr.j], rjS = rings[R - 1 - pr.j];
        const int Nj = rj.n;
        const double omega = pr.scale * (double)pr.M;                              // Omega_j
        const double shj = rj.shifted ? 0.5 : 0.0;
        // window of input pixels that can lie inside the support: |dphi| <= psimax (a superset; gamma decides)
        int l0 = 0, cnt = Nj;
        if (pr.B > 0.0) {
            const double ratio = (xmax - pr.A) / pr.B;
            if (ratio < 1.0) {
                const double psimax = 2.0 * asin(sqrt(fmax(ratio, 0.0)));          // radians
                const int hw = (int)floor(psimax * (double)Nj * (0.5 / 3.14159265358979323846)) + 1;
                if (2 * hw + 1 < Nj) {
                    const int lc = (int)floor(uk * (double)Nj - shj + 0.5);
                    l0 = lc - hw;
                    cnt = 2 * hw + 1;
                }
            }
        }
        const T* __restrict__ inN = in + (int64_t)map0 * npix + rj.pix_off;
        const T* __restrict__ inS = in + (int64_t)map0 * npix + rjS.pix_off;
        for (int c = 0; c < cnt; ++c) {
            int l = l0 + c;
            l = l < 0 ? l + Nj : (l >= Nj ? l - Nj : l);
            const double dturn = ((double)l + shj) / (double)Nj - uk;
            const double sh = sinpi(dturn);
            const double gamma = gamma_of_chord2(pr.A + pr.B * sh * sh);
            if (gamma < theta_max) {
                const double uu = gamma * tscale;
                int tt = (int)floor(uu);
                tt = max(0, min(tt, ntab - 2));
                const double f = uu - (double)tt;
                const double k0 = table[tt], k1 = table[tt + 1];
                const T w = (T)((k0 + f * (k1 - k0)) * omega);
#pragma unroll
                for (int q = 0; q < NM; ++q) {
                    if (map0 + q < nmaps) {
                        accN[q] += w * inN[(int64_t)q * npix + l];
                        accS[q] += w * inS[(int64_t)q * npix + l];
                    }
                }
            }
        }
    }
#pragma unroll
    for (int q = 0; q < NM; ++q) {
        if (map0 + q < nmaps) {
            out[(int64_t)(map0 + q) * npix + ri.pix_off + k] = accN[q];
            if (iS != i) out[(int64_t)(map0 + q) * npix + riS.pix_off + k] = accS[q];
        }
    }
}

}  // namespace arkcos
