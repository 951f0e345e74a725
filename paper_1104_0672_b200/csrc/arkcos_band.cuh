// Kernel-row generator and banded per-mode multiply-accumulate (steps 3-6 of the hot path).
//
// For output ring i and input ring j inside the support, the kernel row kappa_ij(psi) = K(gamma(theta_i,theta_j,psi))
// (Eq. 9) is even in psi, so its transform along phi is a cosine series over half a row:
//     G_ij[m] = (Omega_j / M) sum_d kappa(psi_d) cos(m psi_d) = sum_t W_ij[t] cos(m (2t + par) pi / M)
// with W the non-zero half-row samples (weight 2 for a sample that has a mirror image, "only on the first
// 2 nside + 1 pixels of a ring").  The output ring's folded spectrum is
//     Dp_i[m'] = sum_j sum_{m = m' + w N_i or w N_i - m', 0 <= m <= M/2} (+-) G_ij[m] Bp_j[m]  (conjugated for the second family)
// ("multiplied ... summation over n_support elements in the theta-direction", PAPER.md:219 duplicate + fold).
// DESIGN.md "Band kernel" derives the signs; the same G serves ring i and its mirror image in the south
// ("only for the northern hemisphere", "northern and southern hemisphere simultaneously").
#pragma once
#include "arkcos_device.cuh"
#include "arkcos_fft.cuh"

namespace arkcos {

struct PairRec {
    double A, B;       // x = A + B sin^2(psi/2): A = 4 sin^2((theta_i - theta_j)/2), B = 4 sin(theta_i) sin(theta_j)
    double scale;      // Omega_j / M
    int64_t woff;      // first sample of the row in W
    int M;             // length of the phi grid of this row (even)
    int par;           // sample positions psi_t = (2t + par) pi / M ; par = 1: half-step offset
    int cnt;           // stored samples t = 0 .. cnt-1
    int j;             // input ring (northern image)
};

struct NorthRec { int pair_lo, pair_hi; };     // pairs of northern output ring i
struct BandItem { int ring, m0; };             // one block of the band kernel: output ring, first folded mode

// Step 3: evaluate the tabulated profile on the half-row of every ring pair.  The distance is
// computed in double precision for both dtypes.  One block per pair.
template <class T> __global__ void kernel_rows_kernel(const PairRec* __restrict__ pairs, int npairs,
                                                      const double* __restrict__ table, int ntab, double theta_max,
                                                      T* __restrict__ W)
{
    const int p = blockIdx.x;
    if (p >= npairs) return;
    const PairRec pr = pairs[p];
    const double inv2M = 1.0 / (2.0 * (double)pr.M);
    const double tscale = (double)(ntab - 1) / theta_max;
    for (int t = threadIdx.x; t < pr.cnt; t += blockDim.x) {
        const int u = 2 * t + pr.par;
        const double sh = sinpi((double)u * inv2M);                    // sin(psi/2), psi = u pi / M
        const double x = pr.A + pr.B * sh * sh;
        double hx = 0.5 * sqrt(x);
        if (hx > 1.0) hx = 1.0;
        const double gamma = 2.0 * asin(hx);
        double val = 0.0;
        if (gamma < theta_max) {
            const double uu = gamma * tscale;
            int tt = (int)floor(uu);
            tt = max(0, min(tt, ntab - 2));
            const double f = uu - (double)tt;
            const double k0 = table[tt], k1 = table[tt + 1];
            const double mult = (u == 0 || u == pr.M) ? 1.0 : 2.0;
            val = (k0 + f * (k1 - k0)) * pr.scale * mult;
        }
        W[pr.woff + t] = (T)val;
    }
}

// Bp_j extended to any mode m >= 0 from the stored half spectrum b[0 .. N/2] (periodic extension).
template <class T> __device__ __forceinline__ cx<T> ext_mode(const cx<T>* __restrict__ b, int m, int N, int shifted)
{
    const int wj = m / N, r = m - wj * N;
    cx<T> v;
    if (2 * r <= N) v = b[r];
    else {
        v = cconj(b[N - r]);
        if (shifted) v = mk<T>(-v.x, -v.y);
    }
    if (shifted && (wj & 1)) v = mk<T>(-v.x, -v.y);
    return v;
}

// Reference band kernel: one thread per folded output mode m', cosines by rotation re-seeded every RESEED samples.
// grid = (items, nmaps).
template <class T, int RESEED>
__global__ void band_mac_general_kernel(const BandItem* __restrict__ items, const NorthRec* __restrict__ north,
                                        const PairRec* __restrict__ pairs, const T* __restrict__ W,
                                        const RingRec* __restrict__ rings, int R, const cx<T>* __restrict__ specIn,
                                        cx<T>* __restrict__ specOut, int64_t spec_stride)
{
    const BandItem it = items[blockIdx.x];
    const int i = it.ring, iS = R - 1 - i;
    const RingRec ri = rings[i];
    const int Ni = ri.n, mp = it.m0 + (int)threadIdx.x;
    if (2 * mp > Ni) return;
    const cx<T>* __restrict__ in = specIn + (int64_t)blockIdx.y * spec_stride;
    cx<T> accN = mk<T>(0, 0), accS = mk<T>(0, 0);
    const NorthRec nr = north[i];
    for (int p = nr.pair_lo; p < nr.pair_hi; ++p) {
        const PairRec pr = pairs[p];
        const RingRec rj = rings[pr.j], rjS = rings[R - 1 - pr.j];
        const cx<T>* __restrict__ bN = in + rj.spec_off;
        const cx<T>* __restrict__ bS = in + rjS.spec_off;
        const T* __restrict__ w = W + pr.woff;
        const int M = pr.M, Mh = M >> 1;
        for (int fam = 0; fam < 2; ++fam) {
            int wi = fam;
            for (int m = fam ? Ni - mp : mp; m <= Mh; m += Ni, ++wi) {
                // G_ij[m] = sum_t w[t] cos(m (2t + par) pi / M)
                const cx<T> rot = cispi_ratio<T>((uint32_t)((2u * (uint32_t)m) % (2u * (uint32_t)M)), (uint32_t)M);
                T G = 0;
                for (int t0 = 0; t0 < pr.cnt; t0 += RESEED) {
                    const uint64_t q = ((uint64_t)m * (uint64_t)(2 * t0 + pr.par)) % (uint64_t)(2 * M);
                    cx<T> c = cispi_ratio<T>((uint32_t)q, (uint32_t)M);
                    const int t1 = min(pr.cnt, t0 + RESEED);
                    for (int t = t0; t < t1; ++t) {
                        G += w[t] * c.x;
                        c = cmul(c, rot);
                    }
                }
                if (2 * m == M) G *= (T)0.5;                         // the +-M/2 bins carry half the Nyquist term each
                if (ri.shifted && (wi & 1)) G = -G;                   // exp(i m phi0_i) = (-1)^w exp(+-i m' phi0_i)
                cx<T> vN = ext_mode(bN, m, rj.n, rj.shifted);
                cx<T> vS = ext_mode(bS, m, rjS.n, rjS.shifted);
                if (fam) { vN.y = -vN.y; vS.y = -vS.y; }
                accN.x += G * vN.x; accN.y += G * vN.y;
                accS.x += G * vS.x; accS.y += G * vS.y;
            }
        }
    }
    cx<T>* __restrict__ out = specOut + (int64_t)blockIdx.y * spec_stride;
    out[ri.spec_off + mp] = accN;
    if (iS != i) out[rings[iS].spec_off + mp] = accS;
}

}  // namespace arkcos
