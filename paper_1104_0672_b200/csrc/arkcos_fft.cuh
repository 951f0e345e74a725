// Ring FFTs of libarkcos: real FFT of every isolatitude ring and its inverse (steps 1 and 7 of the hot path,
// PAPER.md:125 "a real-to-complex Fourier transform of length n_FFT on each ring", "a complex-to-real
// backward FFT on all output rings"), fused with the re-origin phase of Eq. 8.
//
// A ring of N reals (N even) is transformed as one complex FFT of length L = N/2 plus an O(N) split.  Power-of-two L:
// Stockham radix-8 passes held in registers, exchanged through padded shared memory.  Any other L (HEALPix cap rings,
// N = 4n): Bluestein's chirp-z with a power-of-two convolution length P >= 2L-1; chirps, phases and the filter
// spectrum come from tables built once per distinct ring length at plan time.
#pragma once
#include "arkcos_device.cuh"

namespace arkcos {

constexpr int kFftThreads = 512;

// shared-memory index padding: one extra slot every 16 complex numbers keeps the radix-8 scatter conflict-free
__device__ __forceinline__ int phys(int e) { return e + (e >> 4); }
__host__ __device__ inline size_t fft_smem_elems(int P) { return (size_t)P + (size_t)(P >> 4) + 1; }

template <class T> __device__ __forceinline__ cx<T> mul_mi(cx<T> a) { return mk<T>(a.y, -a.x); }     // a * (-i)

template <class T> __device__ __forceinline__ void dft2(cx<T>* u)
{
    const cx<T> a = u[0] + u[1], b = u[0] - u[1];
    u[0] = a; u[1] = b;
}
template <class T> __device__ __forceinline__ void dft4(cx<T>* u)
{
    const cx<T> s02 = u[0] + u[2], d02 = u[0] - u[2], s13 = u[1] + u[3], d13 = mul_mi(u[1] - u[3]);
    u[0] = s02 + s13; u[2] = s02 - s13; u[1] = d02 + d13; u[3] = d02 - d13;
}
template <class T> __device__ __forceinline__ void dft8(cx<T>* u)
{
    const T h = (T)0.70710678118654752440;
    cx<T> a[8];
#pragma unroll
    for (int n = 0; n < 4; ++n) { a[n] = u[n] + u[n + 4]; a[n + 4] = u[n] - u[n + 4]; }
    a[5] = mk<T>(h * (a[5].x + a[5].y), h * (a[5].y - a[5].x));          // * exp(-i pi/4)
    a[6] = mul_mi(a[6]);                                                  // * exp(-i pi/2)
    a[7] = mk<T>(h * (a[7].y - a[7].x), -h * (a[7].x + a[7].y));         // * exp(-3 i pi/4)
    dft4(a);
    dft4(a + 4);
    u[0] = a[0]; u[2] = a[1]; u[4] = a[2]; u[6] = a[3];
    u[1] = a[4]; u[3] = a[5]; u[5] = a[6]; u[7] = a[7];
}
template <class T> __device__ __forceinline__ void dft16(cx<T>* u)
{
    // 16 = 4 x 4: DFT4 over n1 (stride 4), twiddle exp(-2 pi i n0 k1 / 16), DFT4 over n0; X[k1 + 4 k0]
    const T c1 = (T)0.92387953251128675613, s1 = (T)0.38268343236508977173, h = (T)0.70710678118654752440;
    cx<T> a[4][4];
#pragma unroll
    for (int n0 = 0; n0 < 4; ++n0) {
        cx<T> t[4] = {u[n0], u[n0 + 4], u[n0 + 8], u[n0 + 12]};
        dft4(t);
#pragma unroll
        for (int k1 = 0; k1 < 4; ++k1) a[n0][k1] = t[k1];
    }
    // twiddles w^(n0 k1), w = exp(-i pi / 8)
    const cx<T> w1 = mk<T>(c1, -s1), w2 = mk<T>(h, -h), w3 = mk<T>(s1, -c1), w6 = mk<T>(-h, -h), w9 = mk<T>(-c1, s1);
    a[1][1] = cmul(a[1][1], w1); a[1][2] = cmul(a[1][2], w2); a[1][3] = cmul(a[1][3], w3);
    a[2][1] = cmul(a[2][1], w2); a[2][2] = mul_mi(a[2][2]);   a[2][3] = cmul(a[2][3], w6);
    a[3][1] = cmul(a[3][1], w3); a[3][2] = cmul(a[3][2], w6); a[3][3] = cmul(a[3][3], w9);
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) {
        cx<T> t[4] = {a[0][k1], a[1][k1], a[2][k1], a[3][k1]};
        dft4(t);
#pragma unroll
        for (int k0 = 0; k0 < 4; ++k0) u[k1 + 4 * k0] = t[k0];
    }
}
template <class T, int R> __device__ __forceinline__ void dftR(cx<T>* u)
{
    if (R == 16) dft16(u); else if (R == 8) dft8(u); else if (R == 4) dft4(u); else dft2(u);
}

// One Stockham pass of radix R over the N = 2^logN points in s (padded indexing), p = 2^logp = product of the radices
// of the passes already done.  tw[k] = exp(-2 pi i k / PT), k = 0 .. PT-1.
template <class T, int R, int BPT>
__device__ __forceinline__ void stockham_pass(cx<T>* s, int logN, int logp, const cx<T>* __restrict__ tw, int logPT)
{
    constexpr int logR = R == 16 ? 4 : (R == 8 ? 3 : (R == 4 ? 2 : 1));
    const int nb = 1 << (logN - logR), p = 1 << logp;
    const int sh = logPT - logp - logR;                     // exp(-2 pi i r k / (p R)) = tw[(r k) << sh]
    cx<T> u[BPT][R];
    cx<T> w1[BPT], w2[BPT], w4[BPT], w8[BPT];
    // twiddle loads first (global, L1-resident), so their latency overlaps the shared-memory gather
#pragma unroll
    for (int b = 0; b < BPT; ++b) {
        const int i = (int)threadIdx.x + b * kFftThreads;
        if (i < nb && logp > 0) {
            const int k = i & (p - 1);
            w1[b] = tw[k << sh];
            if (R >= 4) w2[b] = tw[(2 * k) << sh];
            if (R >= 8) w4[b] = tw[(4 * k) << sh];
            if (R >= 16) w8[b] = tw[(8 * k) << sh];
        }
    }
    const bool wide_in = nb >= 16, wide_out = p >= 16;      // strides that are multiples of 16 keep the padding affine
#pragma unroll
    for (int b = 0; b < BPT; ++b) {
        const int i = (int)threadIdx.x + b * kFftThreads;
        if (i < nb) {
            if (wide_in) {
                const int base = phys(i), stride = nb + (nb >> 4);
#pragma unroll
                for (int r = 0; r < R; ++r) u[b][r] = s[base + r * stride];
            } else {
#pragma unroll
                for (int r = 0; r < R; ++r) u[b][r] = s[phys(i + r * nb)];
            }
        }
    }
    __syncthreads();
#pragma unroll
    for (int b = 0; b < BPT; ++b) {
        const int i = (int)threadIdx.x + b * kFftThreads;
        if (i < nb) {
            const int k = i & (p - 1);
            if (logp > 0) {
                cx<T> w[R];
                w[1] = w1[b];
                if (R >= 4) { w[2] = w2[b]; w[3] = cmul(w[1], w[2]); }
                if (R >= 8) {
                    w[4] = w4[b];
#pragma unroll
                    for (int r = 5; r < 8; ++r) w[r] = cmul(w[4], w[r - 4]);
                }
                if (R >= 16) {
                    w[8] = w8[b];
#pragma unroll
                    for (int r = 9; r < 16; ++r) w[r] = cmul(w[8], w[r - 8]);
                }
#pragma unroll
                for (int r = 1; r < R; ++r) u[b][r] = cmul(u[b][r], w[r]);
            }
            dftR<T, R>(u[b]);
            const int j = ((i - k) << logR) + k;
            if (wide_out) {
                const int base = phys(j), stride = p + (p >> 4);
#pragma unroll
                for (int q = 0; q < R; ++q) s[base + q * stride] = u[b][q];
            } else {
#pragma unroll
                for (int q = 0; q < R; ++q) s[phys(j + q * p)] = u[b][q];
            }
        }
    }
    __syncthreads();
}

// Forward complex DFT, natural order in and out, of the 2^logN points in s (padded indexing), in place.
// BPT >= 2^logN / (8 * kFftThreads).  s must be synchronised on entry; it is synchronised on return.
// Radix plan: radix-8 passes, the remainder absorbed by radix-16 passes (3a+1 = 3(a-1)+4, 3a+2 = 3(a-2)+4+4).
template <class T, int BPT> __device__ void fft_pow2(cx<T>* s, int logN, const cx<T>* __restrict__ tw, int logPT)
{
    constexpr int B16 = BPT > 1 ? BPT / 2 : 1;
    int logp = 0;
    int n16 = logN % 3;                                   // number of radix-16 passes wanted
    if (logN < 4 * n16) n16 = 0;                          // too short: finish with a radix-4 / radix-2 pass instead
    const int n8 = (logN - 4 * n16) / 3;
    for (int a = 0; a < n8; ++a, logp += 3) stockham_pass<T, 8, BPT>(s, logN, logp, tw, logPT);
    for (int a = 0; a < n16; ++a, logp += 4) stockham_pass<T, 16, B16>(s, logN, logp, tw, logPT);
    if (logN - logp == 2) stockham_pass<T, 4, 2 * BPT>(s, logN, logp, tw, logPT);
    else if (logN - logp == 1) stockham_pass<T, 2, 4 * BPT>(s, logN, logp, tw, logPT);
}

// Description of one FFT length (one per distinct ring length; device table built at plan time).
struct FftLen {
    int L;             // complex length = N/2
    int logP;          // pow2: P = L; Bluestein: P = smallest power of two >= 2L-1
    int pow2;          // 1: direct power-of-two transform
    int pad;
    int64_t filt_off;  // Bluestein: offset of the filter spectrum FFT_P(b)/P in the filter table
    int64_t chirp_off; // Bluestein: offset of chirp[n] = exp(-i pi n^2 / L), n < L, in the chirp table
    int64_t ph_off;    // offset of ph[k] = exp(-i pi k / N), k = 0 .. L, in the phase table
};

// Forward complex DFT of length L of the natural-order data in s[phys(0 .. L-1)]; the result replaces it.
// Bluestein: X[k] = w[k] sum_n (z[n] w[n]) conj(w[k-n]),  w[n] = exp(-i pi n^2 / L), as a cyclic convolution of length P.
// pre_chirped: the caller already multiplied the input by w[n] and zero-padded s up to P.
template <class T, int BPT>
__device__ void fft_len(cx<T>* s, const FftLen& f, const cx<T>* __restrict__ tw, int logPT,
                        const cx<T>* __restrict__ filt, const cx<T>* __restrict__ chirp)
{
    fft_pow2<T, BPT>(s, f.logP, tw, logPT);
    if (f.pow2) return;
    const int L = f.L, P = 1 << f.logP;
    const cx<T>* __restrict__ fl = filt + f.filt_off;
    const cx<T>* __restrict__ cw = chirp + f.chirp_off;
    // inverse transform of Y F as conj(FFT(conj(Y F)))
    for (int k = threadIdx.x; k < P; k += kFftThreads) s[phys(k)] = cconj(cmul(s[phys(k)], fl[k]));
    __syncthreads();
    fft_pow2<T, BPT>(s, f.logP, tw, logPT);
    for (int k = threadIdx.x; k < L; k += kFftThreads) s[phys(k)] = cmul(cconj(s[phys(k)]), cw[k]);
    __syncthreads();
}

// Plan time: filter spectrum of Bluestein's convolution, one length per block:
// b[n] = exp(+i pi n^2 / L) for |n| < L placed circularly on P points; filt = FFT_P(b) / P.
template <class T, int BPT>
__global__ void __launch_bounds__(kFftThreads, sizeof(T) == 4 ? 2 : 1)
bluestein_filter_kernel(const FftLen* __restrict__ lens, const int* __restrict__ which, const cx<T>* __restrict__ tw,
                        int logPT, const cx<T>* __restrict__ chirp, cx<T>* __restrict__ filt)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* s = reinterpret_cast<cx<T>*>(smem_raw);
    const FftLen f = lens[which[blockIdx.x]];
    const int L = f.L, P = 1 << f.logP;
    const cx<T>* __restrict__ cw = chirp + f.chirp_off;
    for (int n = threadIdx.x; n < P; n += kFftThreads) {
        cx<T> v = mk<T>(0, 0);
        if (n < L) v = cconj(cw[n]);
        else if (n > P - L) v = cconj(cw[P - n]);
        s[phys(n)] = v;
    }
    __syncthreads();
    fft_pow2<T, BPT>(s, f.logP, tw, logPT);
    const T inv = (T)1 / (T)P;
    for (int k = threadIdx.x; k < P; k += kFftThreads) filt[f.filt_off + k] = cscale(s[phys(k)], inv);
}

// Per-ring record used by the FFT kernels and the band kernel.
struct RingRec {
    int64_t pix_off;   // first pixel of the ring in a map
    int64_t spec_off;  // first coefficient of the ring in a spectrum array (ring r holds N/2+1 coefficients)
    int n;             // pixels on the ring
    int shifted;       // 1: phi0 = pi / n, 0: phi0 = 0
    int len_id;        // index into the FftLen table
    int pad;
};

// Step 1 + 2: Bp_j[k] = exp(-i k phi0_j) sum_l in(j,l) exp(-2 pi i k l / N_j), k = 0 .. N_j/2.
// grid = (rings, nmaps); block b works on ring order[b] (longest transforms first).
template <class T, int BPT>
__global__ void __launch_bounds__(kFftThreads, sizeof(T) == 4 ? 2 : 1)
ring_fft_forward_kernel(const T* __restrict__ in, int64_t npix, cx<T>* __restrict__ spec, int64_t spec_stride,
                        const RingRec* __restrict__ rings, const int* __restrict__ order,
                        const FftLen* __restrict__ lens, const cx<T>* __restrict__ tw, int logPT,
                        const cx<T>* __restrict__ filt, const cx<T>* __restrict__ chirp, const cx<T>* __restrict__ phase)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* s = reinterpret_cast<cx<T>*>(smem_raw);
    const RingRec r = rings[order[blockIdx.x]];
    const FftLen f = lens[r.len_id];
    const int N = r.n, L = N >> 1, P = 1 << f.logP;
    const cx<T>* __restrict__ x = reinterpret_cast<const cx<T>*>(in + (int64_t)blockIdx.y * npix + r.pix_off);
    if (f.pow2) {
        for (int l = threadIdx.x; l < L; l += kFftThreads) s[phys(l)] = x[l];          // z[l] = x[2l] + i x[2l+1]
    } else {
        const cx<T>* __restrict__ cw = chirp + f.chirp_off;
        for (int l = threadIdx.x; l < P; l += kFftThreads) s[phys(l)] = l < L ? cmul(x[l], cw[l]) : mk<T>(0, 0);
    }
    __syncthreads();
    fft_len<T, BPT>(s, f, tw, logPT, filt, chirp);
    cx<T>* __restrict__ out = spec + (int64_t)blockIdx.y * spec_stride + r.spec_off;
    const cx<T>* __restrict__ ph = phase + f.ph_off;
    for (int k = threadIdx.x; k <= L; k += kFftThreads) {
        const cx<T> zk = s[phys(k == L ? 0 : k)];
        const cx<T> zc = cconj(s[phys(k == 0 ? 0 : L - k)]);
        const cx<T> e = cscale(zk + zc, (T)0.5), o = cscale(zk - zc, (T)0.5);
        const cx<T> h = ph[k];                         // exp(-i pi k / N)
        const cx<T> wo = cmul(cmul(h, h), o);          // exp(-2 pi i k / N) o
        cx<T> X = mk<T>(e.x + wo.y, e.y - wo.x);       // X[k] = e - i exp(-2 pi i k / N) o
        if (r.shifted) X = cmul(X, h);
        out[k] = X;
    }
}

// Step 6 + 7: out(i,k) = sum_{m'} D_i[m'] exp(2 pi i m' k / N_i) with D_i[m'] = exp(+i m' phi0_i) Dp_i[m'] for
// m' = 0 .. N_i/2 and Hermitian symmetry for the rest.  grid = (rings, nmaps).
template <class T, int BPT>
__global__ void __launch_bounds__(kFftThreads, sizeof(T) == 4 ? 2 : 1)
ring_fft_inverse_kernel(const cx<T>* __restrict__ spec, int64_t spec_stride, T* __restrict__ outmap, int64_t npix,
                        const RingRec* __restrict__ rings, const int* __restrict__ order,
                        const FftLen* __restrict__ lens, const cx<T>* __restrict__ tw, int logPT,
                        const cx<T>* __restrict__ filt, const cx<T>* __restrict__ chirp, const cx<T>* __restrict__ phase)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* s = reinterpret_cast<cx<T>*>(smem_raw);
    const RingRec r = rings[order[blockIdx.x]];
    const FftLen f = lens[r.len_id];
    const int N = r.n, L = N >> 1, P = 1 << f.logP;
    const cx<T>* __restrict__ D = spec + (int64_t)blockIdx.y * spec_stride + r.spec_off;
    const cx<T>* __restrict__ ph = phase + f.ph_off;
    const cx<T>* __restrict__ cw = chirp + f.chirp_off;
    for (int k = threadIdx.x; k < (f.pow2 ? L : P); k += kFftThreads) {
        cx<T> v = mk<T>(0, 0);
        if (k < L) {
            cx<T> xk = D[k], xl = D[L - k];
            const cx<T> hk = cconj(ph[k]), hl = cconj(ph[L - k]);      // exp(+i pi k / N)
            if (r.shifted) { xk = cmul(xk, hk); xl = cmul(xl, hl); }
            const cx<T> xc = cconj(xl);
            const cx<T> a = xk + xc, d = xk - xc;
            const cx<T> wd = cmul(cmul(hk, hk), d);                    // exp(+2 pi i k / N) d
            // Z[k] = a + i wd ; the inverse transform is done as conj(FFT(conj Z))
            v = mk<T>(a.x - wd.y, -(a.y + wd.x));
            if (!f.pow2) v = cmul(v, cw[k]);
        }
        s[phys(k)] = v;
    }
    __syncthreads();
    fft_len<T, BPT>(s, f, tw, logPT, filt, chirp);
    cx<T>* __restrict__ o = reinterpret_cast<cx<T>*>(outmap + (int64_t)blockIdx.y * npix + r.pix_off);
    for (int n = threadIdx.x; n < L; n += kFftThreads) {
        const cx<T> z = s[phys(n)];
        o[n] = mk<T>(z.x, -z.y);                                       // out[2n], out[2n+1]
    }
}

}  // namespace arkcos
