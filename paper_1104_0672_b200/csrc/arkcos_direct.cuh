// Exact direct-space sum on selected output rings (option exact_caps): Eq. 6 of the paper with compact-support pruning
// (the paper itself recomputes pixels by direct sum where the Fourier scheme is not good enough,
// PAPER.md:178).  Used for the HEALPix polar-cap rings and the equatorial rings whose band reaches into a cap: there the
// hybrid scheme only "suppresses" ringing for discontinuous or hard-cut kernels, the direct sum has none.
//
//   out(i,k) = sum_{j in band(i)} Omega_j sum_{l : gamma < theta_max} K(gamma) in(j,l),
//   x = 2 - 2 cos(gamma) = A_ij + B_ij sin^2(dphi / 2)   (Eq. 9),  dphi = phi_jl - phi_ik.
//
// A weight K(gamma) Omega_j depends on the map not at all, on the hemisphere not at all and, every HEALPix
// ring having a multiple of four pixels with the same pattern in each quadrant, not on the quadrant: one thread owns output
// pixel k of the first quadrant of northern ring i, its three images k + q N_i/4 and the four of the mirror ring, for NM
// maps at once: 8 NM accumulators per evaluated weight.  Distances and the profile interpolation are double precision, as
// in the kernel-row generator; the accumulators have the plan's precision.
// Along an input ring the azimuth difference advances by a fixed angle, so sin(dphi/2) follows by a plane rotation from
// one sincospi per (thread, ring pair); gamma^2 is a short series in x (the squared chord is small for compact kernels);
// what depends on the ring pair alone (window half-width, rotation step) is computed once per block; UN input pixels are
// evaluated side by side (independent dependency chains); the table holds (K[t], K[t+1] - K[t]) so that a lookup is one
// 16-byte load.
// From four maps on, the input pixels a block needs from one input ring (the union of its threads' windows, for every map,
// hemisphere and quadrant) are staged in shared memory, four maps of one pixel per 16-byte word, and the weights of a thread in
// a thread-private column of shared memory: the inner loop is one 16-byte shared-memory read per four multiply-adds.
#pragma once
#include "arkcos_band.cuh"

namespace arkcos {

constexpr int kDirectThreads = 128;
constexpr int kDirectChunk = 32;              // window pixels whose weights a thread stages at a time (NM >= 4; a multiple of UN)
constexpr int kDirectPairChunk = 64;          // ring pairs whose constants are staged in shared memory at a time
constexpr int kDirectWindow = 224;            // input pixels of one ring a block can stage per stream (NM >= 4)

// sin, cos of pi / N_j; 1 / N_j; window half-width; first pixel and length of the union of the block's windows
struct DirectPairConst { double sd, cd, invn; int hw, lbase, wlen, pad; };

template <class T, int NM> struct DirectCfg {
    static constexpr bool STAGED = NM >= 4;
    static constexpr int VEC = 16 / (int)sizeof(T);                 // maps per 16-byte shared-memory word
    static constexpr int QG = STAGED ? NM / VEC : 1;                // words per staged pixel and (hemisphere, quadrant)
    static constexpr size_t smem = STAGED ? (size_t)8 * NM * kDirectWindow * sizeof(T) : 0;
};

// gamma from the squared chord: gamma^2 = 4 asin^2(sqrt(x)/2) = x + x^2/12 + x^3/90 + x^4/560 + x^5/3150 + x^6/16632 + ...
// (truncation < 1e-17 relative below 2^-9, i.e. gamma < 2.5 degrees); gamma_of_chord2 beyond.
__device__ __forceinline__ double gamma_small_chord2(double x)
{
    if (x < 1.0 / 512.0) {
        double p = 1.0 / 3150.0;
        p = p * x + 1.0 / 560.0;
        p = p * x + 1.0 / 90.0;
        p = p * x + 1.0 / 12.0;
        p = p * x + 1.0;
        return sqrt(x * p);
    }
    return gamma_of_chord2(x);
}

// input pixel of ring j (Nj pixels, half-pixel shift shj) nearest in azimuth to pixel k of a ring of n pixels (shift shi)
__device__ __forceinline__ int direct_window_centre(int k, double shi, int n, int Nj, double shj)
{
    const double uk = ((double)k + shi) / (double)n;
    return (int)floor(uk * (double)Nj - shj + 0.5);
}

// K(gamma) Omega_j of the input pixel whose sin(dphi / 2) is s; 0 outside the support
template <class T>
__device__ __forceinline__ T direct_weight(const PairRec& pr, double s, double omega, const double2* __restrict__ table2, int ntab,
                                           double tscale, double theta_max, bool inside)
{
    const double gamma = gamma_small_chord2(pr.A + pr.B * (s * s));
    const double uu = gamma * tscale;
    const int tt = min((int)uu, ntab - 2);
    const double f = uu - (double)tt;
    const double2 kk = table2[tt];
    return (inside && gamma < theta_max) ? (T)((kk.x + f * kk.y) * omega) : (T)0;
}

// grid = (blocks of kDirectThreads first-quadrant pixels over the listed rings, map chunks); items: {ring, first pixel};
// dynamic shared memory DirectCfg<T, NM>::smem
template <class T, int NM, int UN>
__global__ void __launch_bounds__(kDirectThreads)
direct_rings_kernel(const BandItem* __restrict__ items, const NorthRec* __restrict__ north,
                    const PairRec* __restrict__ pairs, const RingRec* __restrict__ rings, int R,
                    const double2* __restrict__ table2, int ntab, double theta_max, double xmax,
                    const T* __restrict__ in, T* __restrict__ out, int64_t npix, int nmaps)
{
    using C = DirectCfg<T, NM>;
    constexpr bool STAGED = C::STAGED;
    constexpr int VEC = C::VEC, QG = C::QG, SW = kDirectWindow;
    struct __align__(16) Word { T v[VEC]; };
    extern __shared__ __align__(16) unsigned char direct_smem[];
    Word* sIn = reinterpret_cast<Word*>(direct_smem);                              // [(h * 4 + qd) * QG + g][SW]
    __shared__ DirectPairConst sP[kDirectPairChunk];
    __shared__ T sW[STAGED ? kDirectChunk * kDirectThreads : 1];
    const int tid = (int)threadIdx.x;
    const BandItem it = items[blockIdx.x];
    const int i = it.ring, iS = R - 1 - i;
    const RingRec ri = rings[i], riS = rings[iS];
    const int nq = ri.n >> 2;                                                      // pixels per quadrant
    const int k = it.m0 + tid;
    const bool active = k < nq;
    const int map0 = (int)blockIdx.y * NM;
    const int nm = min(NM, nmaps - map0);
    const double tscale = (double)(ntab - 1) / theta_max;
    const double shi = ri.shifted ? 0.5 : 0.0;
    const double uk = ((double)k + shi) / (double)ri.n;                            // azimuth of the pixel in turns
    T acc[2][4][NM];
#pragma unroll
    for (int h = 0; h < 2; ++h)
#pragma unroll
        for (int qd = 0; qd < 4; ++qd)
#pragma unroll
            for (int q = 0; q < NM; ++q) acc[h][qd][q] = (T)0;
    // map q of this thread's chunk; maps beyond the last one alias it (their sums are never stored), so that the inner loops
    // carry no predicate; a pixel is addressed as bq[q][32-bit offset within the map]
    const T* __restrict__ bq[NM];
#pragma unroll
    for (int q = 0; q < NM; ++q) {
        bq[q] = in + (int64_t)(map0 + min(q, nm - 1)) * npix;
        asm volatile("" : "+l"(bq[q]));          // kept in registers: recomputing it per load costs four instructions
    }
    const NorthRec nr = north[i];
    for (int p0 = nr.pair_lo; p0 < nr.pair_hi; p0 += kDirectPairChunk) {
        __syncthreads();
        if (tid < kDirectPairChunk && p0 + tid < nr.pair_hi) {
            const PairRec pr = pairs[p0 + tid];
            const RingRec rj = rings[pr.j];
            const int Nj = rj.n;
            DirectPairConst pc;
            pc.hw = Nj;                                                            // the whole ring
            // window of input pixels that can lie inside the support: |dphi| <= psimax (a superset; gamma decides)
            if (pr.B > 0.0) {
                const double ratio = (xmax - pr.A) / pr.B;
                if (ratio < 1.0) {
                    const double psimax = 2.0 * asin(sqrt(fmax(ratio, 0.0)));      // radians
                    pc.hw = (int)floor(psimax * (double)Nj * (0.5 / 3.14159265358979323846)) + 1;
                }
            }
            pc.invn = 1.0 / (double)Nj;
            sincospi(pc.invn, &pc.sd, &pc.cd);
            pc.lbase = 0;
            pc.wlen = Nj;
            if (2 * pc.hw + 1 < Nj) {                                              // union of the windows of the block's pixels
                const double shj = rj.shifted ? 0.5 : 0.0;
                const int lcA = direct_window_centre(it.m0, shi, ri.n, Nj, shj);
                const int lcB = direct_window_centre(min(it.m0 + kDirectThreads, nq) - 1, shi, ri.n, Nj, shj);
                pc.lbase = lcA - pc.hw;
                pc.wlen = lcB - lcA + 2 * pc.hw + 1;
            }
            pc.pad = 0;
            sP[tid] = pc;
        }
        __syncthreads();
        const int pe = min(p0 + kDirectPairChunk, nr.pair_hi);
        for (int p = p0; p < pe; ++p) {
            const PairRec pr = pairs[p];
            const DirectPairConst pc = sP[p - p0];
            const RingRec rj = rings[pr.j], rjS = rings[R - 1 - pr.j];
            const int Nj = rj.n, nj4 = Nj >> 2;
            const uint32_t offN = (uint32_t)rj.pix_off, offS = (uint32_t)rjS.pix_off;
            const bool in_smem = STAGED && pc.wlen <= SW;                          // the same for every thread of the block
            if (STAGED && in_smem) {
                __syncthreads();                                                   // the previous pair's window has been read
                const uint32_t lbp = (uint32_t)(pc.lbase < 0 ? pc.lbase + Nj : pc.lbase);
                for (int e = tid; e < pc.wlen; e += kDirectThreads) {
#pragma unroll
                    for (int qd = 0; qd < 4; ++qd) {
                        const uint32_t l = (lbp + (uint32_t)e + (uint32_t)(qd * nj4)) % (uint32_t)Nj;
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            const uint32_t o = (h ? offS : offN) + l;
#pragma unroll
                            for (int g = 0; g < QG; ++g) {
                                Word wd;
#pragma unroll
                                for (int v = 0; v < VEC; ++v) wd.v[v] = __ldg(bq[g * VEC + v] + o);
                                sIn[((h * 4 + qd) * QG + g) * SW + e] = wd;
                            }
                        }
                    }
                }
                __syncthreads();
            }
            if (!active) continue;
            const double omega = pr.scale * (double)pr.M;                          // Omega_j
            const double shj = rj.shifted ? 0.5 : 0.0;
            int l0 = 0, cnt = Nj;
            if (2 * pc.hw + 1 < Nj) {
                l0 = direct_window_centre(k, shi, ri.n, Nj, shj) - pc.hw;
                cnt = 2 * pc.hw + 1;
            }
            double s, c;                                                           // sin, cos of dphi / 2 at the window's first pixel
            sincospi(((double)l0 + shj) * pc.invn - uk, &s, &c);
            if constexpr (STAGED) {
                for (int c0 = 0; c0 < cnt; c0 += kDirectChunk) {
                    const int nw = min(kDirectChunk, cnt - c0);
                    for (int cc = 0; cc < nw; cc += UN) {
#pragma unroll
                        for (int e = 0; e < UN; ++e) {
                            sW[(cc + e) * kDirectThreads + tid] = direct_weight<T>(pr, s, omega, table2, ntab, tscale, theta_max, cc + e < nw);
                            const double s1 = s * pc.cd + c * pc.sd;               // next pixel of the input ring
                            c = c * pc.cd - s * pc.sd;
                            s = s1;
                        }
                    }
                    if (in_smem) {
                        const Word* __restrict__ sb = sIn + (l0 - pc.lbase + c0);
#pragma unroll 2
                        for (int cc = 0; cc < nw; ++cc) {
                            const T w = sW[cc * kDirectThreads + tid];
#pragma unroll
                            for (int h = 0; h < 2; ++h)
#pragma unroll
                                for (int qd = 0; qd < 4; ++qd)
#pragma unroll
                                    for (int g = 0; g < QG; ++g) {
                                        const Word wd = sb[((h * 4 + qd) * QG + g) * SW + cc];
#pragma unroll
                                        for (int v = 0; v < VEC; ++v) acc[h][qd][g * VEC + v] += w * wd.v[v];
                                    }
                        }
                    } else {                                                       // window too long for shared memory: from L1 / L2
                        int lb = l0 + c0;
                        lb = lb < 0 ? lb + Nj : (lb >= Nj ? lb - Nj : lb);
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            const uint32_t ro = h ? offS : offN;
#pragma unroll
                            for (int qd = 0; qd < 4; ++qd) {
                                int l = lb + qd * nj4;
                                l = l >= Nj ? l - Nj : l;
#pragma unroll 2
                                for (int cc = 0; cc < nw; ++cc) {
                                    const T w = sW[cc * kDirectThreads + tid];
                                    const uint32_t o = ro + (uint32_t)l;
#pragma unroll
                                    for (int q = 0; q < NM; ++q) acc[h][qd][q] += w * __ldg(bq[q] + o);
                                    ++l;
                                    l = l == Nj ? 0 : l;
                                }
                            }
                        }
                    }
                }
            } else {
                for (int c0 = 0; c0 < cnt; c0 += UN) {
                    T w[UN];
                    int lw[UN];
#pragma unroll
                    for (int e = 0; e < UN; ++e) {
                        w[e] = direct_weight<T>(pr, s, omega, table2, ntab, tscale, theta_max, c0 + e < cnt);
                        int l = l0 + c0 + e;
                        lw[e] = l < 0 ? l + Nj : (l >= Nj ? l - Nj : l);
                        const double s1 = s * pc.cd + c * pc.sd;                   // next pixel of the input ring
                        c = c * pc.cd - s * pc.sd;
                        s = s1;
                    }
#pragma unroll
                    for (int e = 0; e < UN; ++e) {
                        if (w[e] != (T)0) {
                            int l = lw[e];
#pragma unroll
                            for (int qd = 0; qd < 4; ++qd) {
#pragma unroll
                                for (int q = 0; q < NM; ++q) {
                                    acc[0][qd][q] += w[e] * __ldg(bq[q] + (offN + (uint32_t)l));
                                    acc[1][qd][q] += w[e] * __ldg(bq[q] + (offS + (uint32_t)l));
                                }
                                l += nj4;
                                l = l >= Nj ? l - Nj : l;
                            }
                        }
                    }
                }
            }
        }
    }
    if (!active) return;
#pragma unroll
    for (int q = 0; q < NM; ++q) {
        if (q < nm) {
#pragma unroll
            for (int qd = 0; qd < 4; ++qd) {
                out[(int64_t)(map0 + q) * npix + ri.pix_off + k + qd * nq] = acc[0][qd][q];
                if (iS != i) out[(int64_t)(map0 + q) * npix + riS.pix_off + k + qd * nq] = acc[1][qd][q];
            }
        }
    }
}

}  // namespace arkcos
