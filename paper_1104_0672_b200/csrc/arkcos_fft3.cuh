// Ring FFTs, register-resident version for float rings whose transform size Q is 512 .. 4096 (steps 1+2 and 6+7 of the
// hot path; "a real-to-complex Fourier transform ... on each ring", Eq. 8
// "a complex-to-real backward FFT on all output rings").
//
// A ring of N reals is one complex FFT of length L = N/2 plus a split (as in arkcos_fft.cuh).  Here a thread keeps 16
// points of the transform in registers: Q = 16 * 16 * RL (RL = Q/256 = 2..16) is done as radix-16, radix-16, radix-RL
// Stockham passes with two shared-memory exchanges; T = Q/16 threads per block.
//   * power-of-two rings (L = Q: equatorial rings, ECP): one ring per block (ring_fft3_direct1_kernel, 64 registers, four
//     blocks of the largest size per SM, so that the memory phases of some blocks overlap the butterflies of others);
//   * any other length L <= Q (the HEALPix cap rings N = 4i): Bluestein, one ring per block, TWO transforms side by side
//     (twiddles and index arithmetic paid once).  The cyclic convolution of length P = 2Q is split into its even and odd
//     frequency bins,
//         Y[2k] = FFT_Q(a)[k],  Y[2k+1] = FFT_Q(a[n] w_P^n)[k],     y[n] = E[n] + conj(w_P^n) O[n]  (n < Q),
//     (a = chirped input, zero beyond L <= Q; only y[n < L] is needed), so that the two transforms of a block are the
//     even and the odd half, the filter product needs no exchange (the output layout of one transform is the input
//     layout of the next) and chirp, filter and half-bin phases are fused into the loads and stores.
#pragma once
#include "arkcos_fft3.hpp"

namespace arkcos {

// Forward complex DFT of size Q of NB sequences held in registers: in  u[b][r] = x_b[t + T r],  out u[b][q] = X_b[t + T q].
// s: NB arrays of SQ complex numbers (padded indexing e + e/16).  Twiddle tables laid out so that a warp reads whole
// 128-byte lines (the L1 data pipe is the busiest unit of these kernels):
//   tw16[16 r + k] = exp(-2 pi i r k / 256)  (pass 2: lane k = t mod 16),
//   tw3[256 (r - 1) + i] = exp(-2 pi i r i / Q), r = 1 .. RL-1, i < 256  (pass 3, one table per transform size).
// Entry: any earlier readers of s must have passed a barrier.  Exit: results in registers, s free after the next barrier.
template <int LOGQ, int NB>
__device__ __forceinline__ void fft3(cx<float> (&u)[NB][16], cx<float>* __restrict__ s, const cx<float>* __restrict__ tw,
                                     int logPT, const cx<float>* __restrict__ tw16, const cx<float>* __restrict__ tw3)
{
    using F = Fft3<LOGQ>;
    constexpr int T = F::T, RL = F::RL, NC = F::NC, SQ = F::SQ;
    const int t = (int)threadIdx.x;
    // pass 1: radix 16, no twiddles; butterfly t writes X[16 t + q]
#pragma unroll
    for (int b = 0; b < NB; ++b) {
        dft16(u[b]);
#pragma unroll
        for (int q = 0; q < 16; ++q) s[b * SQ + 17 * t + q] = u[b][q];
    }
    // pass 2 twiddles: row k = t mod 16 of the 16 x 16 table
    cx<float> w[16];
#pragma unroll
    for (int r = 1; r < 16; ++r) w[r] = tw16[16 * r + (t & 15)];
    __syncthreads();
    const int ld0 = t + (t >> 4);
#pragma unroll
    for (int b = 0; b < NB; ++b)
#pragma unroll
        for (int r = 0; r < 16; ++r) u[b][r] = s[b * SQ + ld0 + r * (T + T / 16)];
    __syncthreads();
    // pass 2: radix 16, p = 16; butterfly t writes X[16 (t - k) + k + 16 q]
    {
        const int k = t & 15, st0 = 17 * (t - k) + k;
#pragma unroll
        for (int b = 0; b < NB; ++b) {
#pragma unroll
            for (int r = 1; r < 16; ++r) u[b][r] = cmul(u[b][r], w[r]);
            dft16(u[b]);
#pragma unroll
            for (int q = 0; q < 16; ++q) s[b * SQ + st0 + 17 * q] = u[b][q];
        }
    }
    __syncthreads();
#pragma unroll
    for (int b = 0; b < NB; ++b)
#pragma unroll
        for (int r = 0; r < 16; ++r) u[b][r] = s[b * SQ + ld0 + r * (T + T / 16)];
    // pass 3: radix RL, p = 256: butterflies i = t + T c, c < NC, on registers c + NC r'; output layout = input layout
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        const int i = t + T * c;
        cx<float> wl[RL];
#pragma unroll
        for (int r = 1; r < RL; ++r) wl[r] = tw3[256 * (r - 1) + i];
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            cx<float> v[RL];
            v[0] = u[b][c];
#pragma unroll
            for (int r = 1; r < RL; ++r) v[r] = cmul(u[b][c + NC * r], wl[r]);
            dftR<float, RL>(v);
#pragma unroll
            for (int r = 0; r < RL; ++r) u[b][c + NC * r] = v[r];
        }
    }
}

}  // namespace arkcos

namespace arkcos {

// Asynchronous DRAM -> L2 prefetch of [p, p + bytes) (one thread issues it; 16-byte granularity).
__device__ __forceinline__ void prefetch_l2(const void* p, uint32_t bytes)
{
    const uintptr_t a = (uintptr_t)p & ~(uintptr_t)15;
    const uint32_t n = (uint32_t)(((uintptr_t)p + bytes + 15 - a) & ~(uintptr_t)15);
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(a), "r"(n) : "memory");
}

// X[k] of a real ring from the packed transform: zk = Z[k], zc = conj(Z[L-k]); h = exp(-i pi k / N).
__device__ __forceinline__ cx<float> split_fwd(cx<float> zk, cx<float> zc, cx<float> h, int shifted)
{
    const cx<float> e = cscale(zk + zc, 0.5f), o = cscale(zk - zc, 0.5f);
    const cx<float> wo = cmul(cmul(h, h), o);                  // exp(-2 pi i k / N) o
    cx<float> X = mk<float>(e.x + wo.y, e.y - wo.x);           // e - i exp(-2 pi i k / N) o
    if (shifted) X = cmul(X, h);                               // re-origin, Eq. 8
    return X;
}

// conj(Z[k]) of the packed inverse transform from Dp[k] and Dp[L-k]; hk, hl = exp(+i pi k / N), exp(+i pi (L-k) / N).
__device__ __forceinline__ cx<float> pack_inv(cx<float> xk, cx<float> xl, cx<float> hk, cx<float> hl, int shifted)
{
    if (shifted) { xk = cmul(xk, hk); xl = cmul(xl, hl); }
    const cx<float> xc = cconj(xl);
    const cx<float> a = xk + xc, d = xk - xc;
    const cx<float> wd = cmul(cmul(hk, hk), d);                // exp(+2 pi i k / N) d
    return mk<float>(a.x - wd.y, -(a.y + wd.x));               // conj(a + i wd)
}

// Bluestein middle part shared by both directions: u[0][r] = a[t + T r] (chirped input, zero beyond L) on entry;
// on exit g[q] = conj(y[n]), n = t + T q, y = the cyclic convolution of a with the chirp filter (valid for n < L).
template <int LOGQ>
__device__ __forceinline__ void bluestein_core(cx<float> (&u)[2][16], cx<float>* __restrict__ s, const FftLen& f,
                                               const cx<float>* __restrict__ tw, int logPT,
                                               const cx<float>* __restrict__ tw16, const cx<float>* __restrict__ tw3,
                                               const cx<float>* __restrict__ filt)
{
    using F = Fft3<LOGQ>;
    constexpr int T = F::T;
    const int t = (int)threadIdx.x, L = f.L;
    const int shP = logPT - LOGQ - 1;                           // w_P^n = tw[n << shP], P = 2Q
    const float4* __restrict__ fl = reinterpret_cast<const float4*>(filt + f.filt_off);     // (F[2k], F[2k+1])
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const int n = t + T * r;
        u[1][r] = n < L ? cmul(u[0][r], tw[n << shP]) : mk<float>(0.f, 0.f);
    }
    fft3<LOGQ, 2>(u, s, tw, logPT, tw16, tw3);
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const float4 v = fl[t + T * q];
        u[0][q] = cconj(cmul(u[0][q], mk<float>(v.x, v.y)));
        u[1][q] = cconj(cmul(u[1][q], mk<float>(v.z, v.w)));
    }
    __syncthreads();
    fft3<LOGQ, 2>(u, s, tw, logPT, tw16, tw3);                       // u[0] = conj(E), u[1] = conj(O)
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const int n = t + T * q;
        if (n < L) u[0][q] = u[0][q] + cmul(u[1][q], tw[n << shP]);          // conj(y) = conj(E) + w_P^n conj(O)
    }
}

// Steps 1 + 2, Bluestein rings with transform size Q.  grid = (Bluestein jobs, nmaps), block = Q/16 threads.
template <int LOGQ>
__global__ void __launch_bounds__(Fft3<LOGQ>::T, Fft3<LOGQ>::MINB)
ring_fft3_forward_kernel(const float* __restrict__ in, int64_t npix, cx<float>* __restrict__ spec, int64_t spec_stride,
                         const RingRec* __restrict__ rings, const FftJob* __restrict__ jobs,
                         const FftLen* __restrict__ lens, const cx<float>* __restrict__ tw, int logPT,
                         const cx<float>* __restrict__ tw16, const cx<float>* __restrict__ tw3,
                         const cx<float>* __restrict__ filt, const cx<float>* __restrict__ chirp,
                         const cx<float>* __restrict__ phase, int ahead)
{
    using F = Fft3<LOGQ>;
    constexpr int T = F::T;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<float>* s = reinterpret_cast<cx<float>*>(smem_raw);
    const int t = (int)threadIdx.x;
    const FftJob& job = jobs[blockIdx.x];
    const RingRec r0 = job.r0;
    const FftLen f = job.f;
    const int L = f.L;
    const float* __restrict__ map = in + (int64_t)blockIdx.y * npix;
    cx<float>* __restrict__ out = spec + (int64_t)blockIdx.y * spec_stride;
    if (t == 32 && blockIdx.x + ahead < gridDim.x) {            // the block that follows this one on the SM: inputs -> L2
        const FftJob& nx = jobs[blockIdx.x + ahead];
        prefetch_l2(map + nx.r0.pix_off, (uint32_t)nx.r0.n * 4u);
        if (nx.has1) prefetch_l2(map + nx.r1.pix_off, (uint32_t)nx.r1.n * 4u);
        if (!nx.f.pow2) prefetch_l2(chirp + nx.f.chirp_off, (uint32_t)nx.f.L * 8u);
    }
    const cx<float>* __restrict__ ph = phase + f.ph_off;
    cx<float> u[2][16];
    {
        const cx<float>* __restrict__ x0 = reinterpret_cast<const cx<float>*>(map + r0.pix_off);
        const cx<float>* __restrict__ cw = chirp + f.chirp_off;
        if (t == 0) {
            prefetch_l2(filt + f.filt_off, (uint32_t)(2 * F::Q * sizeof(cx<float>)));
            prefetch_l2(ph, (uint32_t)((L + 1) * sizeof(cx<float>)));
        }
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const int n = t + T * r;
            u[0][r] = n < L ? cmul(x0[n], cw[n]) : mk<float>(0.f, 0.f);
        }
        bluestein_core<LOGQ>(u, s, f, tw, logPT, tw16, tw3, filt);
        // phases of the split: loaded now (into the registers of the odd half), used after the exchange
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const int k = t + T * q;
            u[1][q] = ph[k < L ? k : L];
        }
        __syncthreads();
        // Z[n] = chirp[n] y[n]
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const int n = t + T * q;
            if (n < L) {
                u[0][q] = cmul(cw[n], cconj(u[0][q]));
                s[phys(n)] = u[0][q];
            }
        }
        __syncthreads();
        cx<float>* __restrict__ o = out + r0.spec_off;
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const int k = t + T * q;
            if (k < L) {
                const cx<float> zc = cconj(s[phys(k == 0 ? 0 : L - k)]);
                o[k] = split_fwd(u[0][q], zc, u[1][q], r0.shifted);
            }
        }
        if (t == 0) o[L] = split_fwd(u[0][0], cconj(u[0][0]), ph[L], r0.shifted);
    }
}

// Steps 6 + 7, Bluestein rings with transform size Q.  grid = (Bluestein jobs, nmaps), block = Q/16 threads.
template <int LOGQ>
__global__ void __launch_bounds__(Fft3<LOGQ>::T, Fft3<LOGQ>::MINB)
ring_fft3_inverse_kernel(const cx<float>* __restrict__ spec, int64_t spec_stride, float* __restrict__ outmap, int64_t npix,
                         const RingRec* __restrict__ rings, const FftJob* __restrict__ jobs,
                         const FftLen* __restrict__ lens, const cx<float>* __restrict__ tw, int logPT,
                         const cx<float>* __restrict__ tw16, const cx<float>* __restrict__ tw3,
                         const cx<float>* __restrict__ filt, const cx<float>* __restrict__ chirp,
                         const cx<float>* __restrict__ phase, int ahead)
{
    using F = Fft3<LOGQ>;
    constexpr int T = F::T;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<float>* s = reinterpret_cast<cx<float>*>(smem_raw);
    const int t = (int)threadIdx.x;
    const FftJob& job = jobs[blockIdx.x];
    const RingRec r0 = job.r0;
    const FftLen f = job.f;
    const int L = f.L;
    const cx<float>* __restrict__ D = spec + (int64_t)blockIdx.y * spec_stride;
    float* __restrict__ map = outmap + (int64_t)blockIdx.y * npix;
    if (t == 32 && blockIdx.x + ahead < gridDim.x) {            // the block that follows this one on the SM: inputs -> L2
        const FftJob& nx = jobs[blockIdx.x + ahead];
        prefetch_l2(D + nx.r0.spec_off, (uint32_t)(nx.r0.n / 2 + 1) * 8u);
        if (nx.has1) prefetch_l2(D + nx.r1.spec_off, (uint32_t)(nx.r1.n / 2 + 1) * 8u);
        if (!nx.f.pow2) prefetch_l2(chirp + nx.f.chirp_off, (uint32_t)nx.f.L * 8u);
        prefetch_l2(phase + nx.f.ph_off, (uint32_t)(nx.f.L + 1) * 8u);      // the inverse needs the phases with its first loads
    }
    const cx<float>* __restrict__ ph = phase + f.ph_off;
    cx<float> u[2][16];
    {
        const cx<float>* __restrict__ cw = chirp + f.chirp_off;
        if (t == 0) prefetch_l2(filt + f.filt_off, (uint32_t)(2 * F::Q * sizeof(cx<float>)));
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const int k = t + T * r;
            cx<float> v = mk<float>(0.f, 0.f);
            if (k < L) {
                const cx<float> hk = cconj(ph[k]), hl = mk<float>(hk.y, hk.x);     // exp(i pi (L-k)/N) = i conj(exp(i pi k/N))
                v = cmul(pack_inv(D[r0.spec_off + k], D[r0.spec_off + L - k], hk, hl, r0.shifted), cw[k]);
            }
            u[0][r] = v;
        }
        bluestein_core<LOGQ>(u, s, f, tw, logPT, tw16, tw3, filt);
        // z'[n] = chirp[n] y[n]; out = conj(z') = conj(chirp[n]) conj(y[n])
        cx<float>* __restrict__ o0 = reinterpret_cast<cx<float>*>(map + r0.pix_off);
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const int n = t + T * q;
            if (n < L) o0[n] = cmulc(u[0][q], cw[n]);
        }
    }
}

}  // namespace arkcos

namespace arkcos {

// exp(-i pi q / 32), q = 0 .. 15 (an immediate once the loop over q is unrolled).  A power-of-two ring has N = 32 T, so the
// half-angle phase of the split at k = t + T q is exp(-i pi k / N) = exp(-i pi t / N) exp(-i pi q / 32): one table load per thread.
__device__ __forceinline__ cx<float> phase_step(int q)
{
    constexpr float c[16] = {1.000000000e+00f, 9.951847267e-01f, 9.807852804e-01f, 9.569403357e-01f, 9.238795325e-01f, 8.819212643e-01f,
                             8.314696123e-01f, 7.730104534e-01f, 7.071067812e-01f, 6.343932842e-01f, 5.555702330e-01f, 4.713967368e-01f,
                             3.826834324e-01f, 2.902846773e-01f, 1.950903220e-01f, 9.801714033e-02f};
    return mk<float>(c[q], q == 0 ? 0.f : -c[16 - q]);      // sin(pi q / 32) = cos(pi (16 - q) / 32)
}

// Power-of-two rings, ONE transform per block (block b works on ring b & 1 of direct job b >> 1): twice as many resident
// blocks at half the registers, so that the load / store phases of some blocks overlap the butterflies of the others.
template <int LOGQ, bool FWD>
__global__ void __launch_bounds__(Fft3<LOGQ>::T, 2 * Fft3<LOGQ>::MINB)
ring_fft3_direct1_kernel(const float* __restrict__ in, float* __restrict__ outmap, int64_t npix,
                         cx<float>* __restrict__ spec, int64_t spec_stride, const FftJob* __restrict__ jobs,
                         const cx<float>* __restrict__ tw, int logPT, const cx<float>* __restrict__ tw16,
                         const cx<float>* __restrict__ tw3, const cx<float>* __restrict__ phase)
{
    using F = Fft3<LOGQ>;
    constexpr int T = F::T;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<float>* s = reinterpret_cast<cx<float>*>(smem_raw);
    const int t = (int)threadIdx.x;
    const FftJob& job = jobs[blockIdx.x >> 1];
    if ((blockIdx.x & 1) && !job.has1) return;
    const RingRec rr = (blockIdx.x & 1) ? job.r1 : job.r0;
    const int L = job.f.L;
    const cx<float>* __restrict__ ph = phase + job.f.ph_off;
    cx<float>* __restrict__ sp = spec + (int64_t)blockIdx.y * spec_stride + rr.spec_off;
    const cx<float> pht = ph[t];                                               // exp(-i pi t / N)
    cx<float> u[1][16];
    if (FWD) {
        const cx<float>* __restrict__ x0 = reinterpret_cast<const cx<float>*>(in + (int64_t)blockIdx.y * npix + rr.pix_off);
#pragma unroll
        for (int r = 0; r < 16; ++r) u[0][r] = x0[t + T * r];
        fft3<LOGQ, 1>(u, s, tw, logPT, tw16, tw3);
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 16; ++q) s[phys(t + T * q)] = u[0][q];
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const int k = t + T * q;
            const cx<float> zc = cconj(s[phys(k == 0 ? 0 : L - k)]);
            sp[k] = split_fwd(u[0][q], zc, cmul(pht, phase_step(q)), rr.shifted);
        }
        if (t == 0) sp[L] = split_fwd(u[0][0], cconj(u[0][0]), ph[L], rr.shifted);
    } else {
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const int k = t + T * r;
            const cx<float> hk = cconj(cmul(pht, phase_step(r)));              // exp(+i pi k / N)
            u[0][r] = pack_inv(sp[k], sp[L - k], hk, mk<float>(hk.y, hk.x), rr.shifted);   // exp(i pi (L-k)/N) = i conj(hk)
        }
        fft3<LOGQ, 1>(u, s, tw, logPT, tw16, tw3);
        cx<float>* __restrict__ o0 = reinterpret_cast<cx<float>*>(outmap + (int64_t)blockIdx.y * npix + rr.pix_off);
#pragma unroll
        for (int q = 0; q < 16; ++q) o0[t + T * q] = cconj(u[0][q]);
    }
}

}  // namespace arkcos

namespace arkcos {

// Power-of-two rings of twice the largest transform size (L = 2 Q = 8192 complex points: the belt of HEALPix nside 4096, ECP
// rings of 16384 pixels; PAPER.md:231 names nside 4096 as the next size).  One ring per block as TWO size-Q transforms side by
// side - the even and the odd samples of the packed ring (decimation in time) - and one radix-2 step in registers,
//     Z[k] = E[k] + w^k O[k],   Z[k + Q] = E[k] - w^k O[k],   w = exp(-2 pi i / 2Q),
// with the split / packing of the real ring as in the other kernels.  grid = (jobs, nmaps), block = Q/16 threads, job.r0 only.
template <bool FWD>
__global__ void __launch_bounds__(Fft3<12>::T, Fft3<12>::MINB)
ring_fft3_direct2_kernel(const float* __restrict__ in, float* __restrict__ outmap, int64_t npix,
                         cx<float>* __restrict__ spec, int64_t spec_stride, const FftJob* __restrict__ jobs,
                         const cx<float>* __restrict__ tw, int logPT, const cx<float>* __restrict__ tw16,
                         const cx<float>* __restrict__ tw3, const cx<float>* __restrict__ phase)
{
    using F = Fft3<12>;
    constexpr int T = F::T, Q = F::Q, L = 2 * Q;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<float>* s = reinterpret_cast<cx<float>*>(smem_raw);
    const int t = (int)threadIdx.x;
    const FftJob& job = jobs[blockIdx.x];
    const RingRec rr = job.r0;
    const cx<float>* __restrict__ ph = phase + job.f.ph_off;                   // exp(-i pi k / N), k = 0 .. L
    cx<float>* __restrict__ sp = spec + (int64_t)blockIdx.y * spec_stride + rr.spec_off;
    const int shW = logPT - 13;                                                // w^k = tw[k << shW]
    cx<float> u[2][16];
    if (FWD) {
        const cx<float>* __restrict__ x0 = reinterpret_cast<const cx<float>*>(in + (int64_t)blockIdx.y * npix + rr.pix_off);
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const int m = t + T * r;
            u[0][r] = x0[2 * m];
            u[1][r] = x0[2 * m + 1];
        }
        fft3<12, 2>(u, s, tw, logPT, tw16, tw3);
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const cx<float> wo = cmul(tw[(t + T * q) << shW], u[1][q]);
            u[1][q] = u[0][q] - wo;                                            // Z[k + Q]
            u[0][q] = u[0][q] + wo;                                            // Z[k]
        }
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            s[phys(t + T * q)] = u[0][q];
            s[phys(t + T * q + Q)] = u[1][q];
        }
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const int k = t + T * q;
            sp[k] = split_fwd(u[0][q], cconj(s[phys(k == 0 ? 0 : L - k)]), ph[k], rr.shifted);
            sp[k + Q] = split_fwd(u[1][q], cconj(s[phys(Q - k)]), ph[k + Q], rr.shifted);
        }
        if (t == 0) sp[L] = split_fwd(u[0][0], cconj(u[0][0]), ph[L], rr.shifted);
    } else {
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const int k0 = 2 * (t + T * r), k1 = k0 + 1;
            const cx<float> h0 = cconj(ph[k0]), h1 = cconj(ph[k1]);            // exp(+i pi k / N); exp(i pi (L-k)/N) = i conj(h)
            u[0][r] = pack_inv(sp[k0], sp[L - k0], h0, mk<float>(h0.y, h0.x), rr.shifted);
            u[1][r] = pack_inv(sp[k1], sp[L - k1], h1, mk<float>(h1.y, h1.x), rr.shifted);
        }
        fft3<12, 2>(u, s, tw, logPT, tw16, tw3);
        cx<float>* __restrict__ o0 = reinterpret_cast<cx<float>*>(outmap + (int64_t)blockIdx.y * npix + rr.pix_off);
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const int k = t + T * q;
            const cx<float> wo = cmul(tw[k << shW], u[1][q]);
            o0[k] = cconj(u[0][q] + wo);
            o0[k + Q] = cconj(u[0][q] - wo);
        }
    }
}

}  // namespace arkcos

namespace arkcos {

// Size-8192 transforms of one sequence held as u[0][.] / u[1][.] by 256 threads, built from two size-4096 transforms side by
// side.  Two layouts: "blocked" u[0][q] = x[k], u[1][q] = x[k + Q], k = t + T q, and "interleaved" u[0][r] = x[2m],
// u[1][r] = x[2m + 1], m = t + T r.  Decimation in time takes interleaved input to blocked output, decimation in frequency
// blocked input to interleaved output, so a transform pair (forward, pointwise product, forward again) needs no reordering.
// Entry: earlier readers of s have passed a barrier.  w = exp(-2 pi i / 8192) = tw[1 << shW].
__device__ __forceinline__ void fft8192_dit(cx<float> (&u)[2][16], cx<float>* __restrict__ s, const cx<float>* __restrict__ tw,
                                            int logPT, const cx<float>* __restrict__ tw16, const cx<float>* __restrict__ tw3)
{
    constexpr int T = Fft3<12>::T;
    const int t = (int)threadIdx.x, shW = logPT - 13;
    fft3<12, 2>(u, s, tw, logPT, tw16, tw3);
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const cx<float> wo = cmul(tw[(t + T * q) << shW], u[1][q]);
        u[1][q] = u[0][q] - wo;
        u[0][q] = u[0][q] + wo;
    }
}
__device__ __forceinline__ void fft8192_dif(cx<float> (&u)[2][16], cx<float>* __restrict__ s, const cx<float>* __restrict__ tw,
                                            int logPT, const cx<float>* __restrict__ tw16, const cx<float>* __restrict__ tw3)
{
    constexpr int T = Fft3<12>::T;
    const int t = (int)threadIdx.x, shW = logPT - 13;
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const cx<float> a = u[0][q], b = u[1][q];
        u[0][q] = a + b;
        u[1][q] = cmul(a - b, tw[(t + T * q) << shW]);
    }
    fft3<12, 2>(u, s, tw, logPT, tw16, tw3);
}

// One half (even bins: half = 0, odd bins: half = 1) of the Bluestein convolution of length P = 16384 for a ring of
// 4096 < L <= 8192 complex points: on entry u = the chirped input (interleaved layout, zero beyond L; for half 1 already
// multiplied by w_P^n); on exit u = conj(E[n]) or conj(O[n]) (interleaved layout), cf. bluestein_core.
__device__ __forceinline__ void bluestein16k_half(cx<float> (&u)[2][16], cx<float>* __restrict__ s, int half, const cx<float>* __restrict__ fl,
                                                  const cx<float>* __restrict__ tw, int logPT, const cx<float>* __restrict__ tw16,
                                                  const cx<float>* __restrict__ tw3)
{
    constexpr int T = Fft3<12>::T, Q = Fft3<12>::Q;
    const int t = (int)threadIdx.x;
    fft8192_dit(u, s, tw, logPT, tw16, tw3);
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const int k = t + T * q;                                               // filter table: F[2k], F[2k + 1] side by side
        u[0][q] = cconj(cmul(u[0][q], fl[2 * k + half]));
        u[1][q] = cconj(cmul(u[1][q], fl[2 * (k + Q) + half]));
    }
    __syncthreads();
    fft8192_dif(u, s, tw, logPT, tw16, tw3);
}

// Steps 1 + 2 / 6 + 7 for Bluestein rings of 4096 < L <= 8192 complex points (the long cap rings of HEALPix nside 4096): the two
// halves of the convolution one after the other, the first one parked in the ring's own output row meanwhile (spectrum row of
// L + 1 coefficients / map ring of L pixel pairs; every thread reads back what it wrote).  grid = (jobs, nmaps), 256 threads.
template <bool FWD>
__global__ void __launch_bounds__(Fft3<12>::T, Fft3<12>::MINB)
ring_fft3_bluestein2_kernel(const float* __restrict__ in, float* __restrict__ outmap, int64_t npix,
                            cx<float>* __restrict__ spec, int64_t spec_stride, const FftJob* __restrict__ jobs,
                            const cx<float>* __restrict__ tw, int logPT, const cx<float>* __restrict__ tw16,
                            const cx<float>* __restrict__ tw3, const cx<float>* __restrict__ filt,
                            const cx<float>* __restrict__ chirp, const cx<float>* __restrict__ phase)
{
    using F = Fft3<12>;
    constexpr int T = F::T;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<float>* s = reinterpret_cast<cx<float>*>(smem_raw);
    const int t = (int)threadIdx.x;
    const FftJob& job = jobs[blockIdx.x];
    const RingRec r0 = job.r0;
    const FftLen f = job.f;
    const int L = f.L;
    const int shP = logPT - 14;                                                // w_P^n = tw[n << shP], P = 16384
    const cx<float>* __restrict__ ph = phase + f.ph_off;
    const cx<float>* __restrict__ cw = chirp + f.chirp_off;
    const cx<float>* __restrict__ fl = filt + f.filt_off;
    cx<float>* __restrict__ sp = spec + (int64_t)blockIdx.y * spec_stride + r0.spec_off;
    cx<float> u[2][16];
    if (FWD) {
        const cx<float>* __restrict__ x0 = reinterpret_cast<const cx<float>*>(in + (int64_t)blockIdx.y * npix + r0.pix_off);
        cx<float>* park = sp;                                                  // conj(E[n]), n < L
#pragma unroll 1
        for (int half = 0; half < 2; ++half) {
#pragma unroll
            for (int r = 0; r < 16; ++r) {
#pragma unroll
                for (int b = 0; b < 2; ++b) {
                    const int n = 2 * (t + T * r) + b;
                    cx<float> a = n < L ? cmul(x0[n], cw[n]) : mk<float>(0.f, 0.f);
                    if (half == 1 && n < L) a = cmul(a, tw[n << shP]);
                    u[b][r] = a;
                }
            }
            if (half == 1) __syncthreads();
            bluestein16k_half(u, s, half, fl, tw, logPT, tw16, tw3);
            if (half == 0) {
#pragma unroll
                for (int r = 0; r < 16; ++r)
#pragma unroll
                    for (int b = 0; b < 2; ++b) {
                        const int n = 2 * (t + T * r) + b;
                        if (n < L) park[n] = u[b][r];
                    }
            }
        }
        __syncthreads();
        // conj(y) = conj(E) + w_P^n conj(O);  Z[n] = chirp[n] y[n]
#pragma unroll
        for (int r = 0; r < 16; ++r)
#pragma unroll
            for (int b = 0; b < 2; ++b) {
                const int n = 2 * (t + T * r) + b;
                if (n < L) {
                    const cx<float> cy = park[n] + cmul(u[b][r], tw[n << shP]);
                    s[phys(n)] = cmul(cw[n], cconj(cy));
                }
            }
        __syncthreads();
        for (int k = t; k < L; k += T)
            sp[k] = split_fwd(s[phys(k)], cconj(s[phys(k == 0 ? 0 : L - k)]), ph[k], r0.shifted);
        if (t == 0) sp[L] = split_fwd(s[phys(0)], cconj(s[phys(0)]), ph[L], r0.shifted);
    } else {
        cx<float>* __restrict__ o0 = reinterpret_cast<cx<float>*>(outmap + (int64_t)blockIdx.y * npix + r0.pix_off);
#pragma unroll 1
        for (int half = 0; half < 2; ++half) {
#pragma unroll
            for (int r = 0; r < 16; ++r) {
#pragma unroll
                for (int b = 0; b < 2; ++b) {
                    const int k = 2 * (t + T * r) + b;
                    cx<float> v = mk<float>(0.f, 0.f);
                    if (k < L) {
                        const cx<float> hk = cconj(ph[k]), hl = mk<float>(hk.y, hk.x);     // exp(i pi (L-k)/N) = i conj(exp(i pi k/N))
                        v = cmul(pack_inv(sp[k], sp[L - k], hk, hl, r0.shifted), cw[k]);
                        if (half == 1) v = cmul(v, tw[k << shP]);
                    }
                    u[b][r] = v;
                }
            }
            if (half == 1) __syncthreads();
            bluestein16k_half(u, s, half, fl, tw, logPT, tw16, tw3);
            if (half == 0) {
#pragma unroll
                for (int r = 0; r < 16; ++r)
#pragma unroll
                    for (int b = 0; b < 2; ++b) {
                        const int n = 2 * (t + T * r) + b;
                        if (n < L) o0[n] = u[b][r];                            // parked in the ring's own pixels
                    }
            }
        }
        // z'[n] = chirp[n] y[n]; out = conj(z') = conj(chirp[n]) conj(y[n])
#pragma unroll
        for (int r = 0; r < 16; ++r)
#pragma unroll
            for (int b = 0; b < 2; ++b) {
                const int n = 2 * (t + T * r) + b;
                if (n < L) o0[n] = cmulc(o0[n] + cmul(u[b][r], tw[n << shP]), cw[n]);
            }
    }
}

}  // namespace arkcos
