// Ring FFTs of libarkcos: real FFT of every isolatitude ring and its inverse (steps 1 and 7 of the hot path,
// PAPER.md:125 "a real-to-complex Fourier transform of length n_FFT on each ring", "a complex-to-real
// backward FFT on all output rings"), fused with the re-origin phase of Eq. 8.
//
// A ring of N reals (N even) is transformed as one complex FFT of length L = N/2 plus an O(N) split.  Power-of-two L:
// radix-2 butterflies in shared memory.  Any other L (HEALPix cap rings, N = 4n): Bluestein's chirp-z with a
// power-of-two convolution length P >= 2L-1, whose filter spectrum is computed once per distinct L at plan time.
#pragma once
#include "arkcos_device.cuh"

namespace arkcos {

// ---- complex FFT, in place in shared memory, P = 2^logP points ------------------------------------------------------
// tw[k] = exp(-2 pi i k / PT), k = 0 .. PT/2-1, PT = 2^logPT >= P (global memory, read through L1).

// decimation in frequency: natural order in, bit-reversed order out, kernel exp(-i...)
template <class T> __device__ void fft_dif(cx<T>* s, int logP, const cx<T>* __restrict__ tw, int logPT)
{
    const int half = 1 << (logP - 1);
    for (int lh = logP - 1; lh >= 0; --lh) {
        const int h = 1 << lh;
        for (int b = threadIdx.x; b < half; b += blockDim.x) {
            const int pos = b & (h - 1);
            const int i0 = ((b >> lh) << (lh + 1)) | pos;
            const cx<T> a = s[i0], c = s[i0 + h];
            s[i0] = a + c;
            s[i0 + h] = cmul(a - c, tw[pos << (logPT - 1 - lh)]);
        }
        __syncthreads();
    }
}

// decimation in time with the conjugate twiddles: bit-reversed order in, natural order out, kernel exp(+i...)
template <class T> __device__ void ifft_dit(cx<T>* s, int logP, const cx<T>* __restrict__ tw, int logPT)
{
    const int half = 1 << (logP - 1);
    for (int lh = 0; lh < logP; ++lh) {
        const int h = 1 << lh;
        for (int b = threadIdx.x; b < half; b += blockDim.x) {
            const int pos = b & (h - 1);
            const int i0 = ((b >> lh) << (lh + 1)) | pos;
            const cx<T> a = s[i0], c = cmulc(s[i0 + h], tw[pos << (logPT - 1 - lh)]);
            s[i0] = a + c;
            s[i0 + h] = a - c;
        }
        __syncthreads();
    }
}

__device__ __forceinline__ int bitrev(int k, int logP) { return (int)(__brev((unsigned)k) >> (32 - logP)); }

// Description of one FFT length (one per distinct ring length; device table built at plan time).
struct FftLen {
    int L;            // complex length = N/2
    int logP;         // pow2: P = L; Bluestein: P = smallest power of two >= 2L-1
    int pow2;         // 1: direct power-of-two transform
    int pad;
    int64_t filt_off; // Bluestein: offset of the filter spectrum (bit-reversed order, scaled by 1/P) in the filter table
};

// chirp w[n] = exp(-i pi n^2 / L), n < L <= 8192 (n^2 fits 32 bits)
template <class T> __device__ __forceinline__ cx<T> chirp(uint32_t n, uint32_t L)
{
    const uint32_t r = (n * n) % (2u * L);
    return cispi_ratio<T>(r == 0 ? 0u : 2u * L - r, L);
}

// Forward complex DFT of s[0..L-1] (natural order), X[k] = sum_n s[n] exp(-2 pi i n k / L).
// On return X[k] is at s[fft_out_index(k)].  All threads of the block must call it; s must hold P elements and be
// synchronised on entry; it is synchronised on return.
template <class T> __device__ void fft_len(cx<T>* s, const FftLen& f, const cx<T>* __restrict__ tw, int logPT,
                                           const cx<T>* __restrict__ filt)
{
    if (f.pow2) {
        if (f.logP > 0) fft_dif(s, f.logP, tw, logPT);
        return;
    }
    const int L = f.L, P = 1 << f.logP;
    for (int n = threadIdx.x; n < P; n += blockDim.x)
        s[n] = n < L ? cmul(s[n], chirp<T>(n, L)) : mk<T>(0, 0);
    __syncthreads();
    fft_dif(s, f.logP, tw, logPT);
    const cx<T>* __restrict__ fl = filt + f.filt_off;
    for (int k = threadIdx.x; k < P; k += blockDim.x) s[k] = cmul(s[k], fl[k]);
    __syncthreads();
    ifft_dit(s, f.logP, tw, logPT);
    for (int k = threadIdx.x; k < L; k += blockDim.x) s[k] = cmul(s[k], chirp<T>(k, L));
    __syncthreads();
}
__device__ __forceinline__ int fft_out_index(int k, const FftLen& f) { return f.pow2 ? bitrev(k, f.logP) : k; }

// Plan time: filter spectrum of Bluestein's convolution for one length per block:
// b[n] = exp(+i pi n^2 / L) for |n| < L placed circularly on P points; filt = DIF-FFT(b) / P (bit-reversed order).
template <class T> __global__ void bluestein_filter_kernel(const FftLen* __restrict__ lens, const int* __restrict__ which,
                                                           const cx<T>* __restrict__ tw, int logPT, cx<T>* __restrict__ filt)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* s = reinterpret_cast<cx<T>*>(smem_raw);
    const FftLen f = lens[which[blockIdx.x]];
    const int L = f.L, P = 1 << f.logP;
    for (int n = threadIdx.x; n < P; n += blockDim.x) {
        cx<T> v = mk<T>(0, 0);
        if (n < L) v = cconj(chirp<T>(n, L));
        else if (n > P - L) v = cconj(chirp<T>(P - n, L));
        s[n] = v;
    }
    __syncthreads();
    fft_dif(s, f.logP, tw, logPT);
    const T inv = (T)1 / (T)P;
    for (int k = threadIdx.x; k < P; k += blockDim.x) filt[f.filt_off + k] = cscale(s[k], inv);
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
// grid = (rings, nmaps), one ring per block.
template <class T> __global__ void ring_fft_forward_kernel(const T* __restrict__ in, int64_t npix, cx<T>* __restrict__ spec,
                                                           int64_t spec_stride, const RingRec* __restrict__ rings,
                                                           const FftLen* __restrict__ lens, const cx<T>* __restrict__ tw,
                                                           int logPT, const cx<T>* __restrict__ filt)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* s = reinterpret_cast<cx<T>*>(smem_raw);
    const RingRec r = rings[blockIdx.x];
    const FftLen f = lens[r.len_id];
    const int N = r.n, L = N >> 1;
    const cx<T>* __restrict__ x = reinterpret_cast<const cx<T>*>(in + (int64_t)blockIdx.y * npix + r.pix_off);
    for (int l = threadIdx.x; l < L; l += blockDim.x) s[l] = x[l];          // z[l] = x[2l] + i x[2l+1]
    __syncthreads();
    fft_len(s, f, tw, logPT, filt);
    cx<T>* __restrict__ out = spec + (int64_t)blockIdx.y * spec_stride + r.spec_off;
    for (int k = threadIdx.x; k <= L; k += blockDim.x) {
        const cx<T> zk = s[fft_out_index(k == L ? 0 : k, f)];
        const cx<T> zc = cconj(s[fft_out_index(k == 0 ? 0 : L - k, f)]);
        const cx<T> e = cscale(zk + zc, (T)0.5), o = cscale(zk - zc, (T)0.5);
        // X[k] = e - i exp(-2 pi i k / N) o
        const cx<T> w = cispi_ratio<T>(k == 0 ? 0u : (uint32_t)(2 * N - 2 * k), (uint32_t)N);   // exp(-i pi 2k / N)
        const cx<T> wo = cmul(w, o);
        cx<T> X = mk<T>(e.x + wo.y, e.y - wo.x);
        if (r.shifted) X = cmul(X, cispi_ratio<T>(k == 0 ? 0u : (uint32_t)(2 * N - k), (uint32_t)N));  // exp(-i pi k / N)
        out[k] = X;
    }
}

// Step 6 + 7: out(i,k) = sum_{m'} D_i[m'] exp(2 pi i m' k / N_i) with D_i[m'] = exp(+i m' phi0_i) Dp_i[m'] for
// m' = 0 .. N_i/2 and Hermitian symmetry for the rest.  grid = (rings, nmaps).
template <class T> __global__ void ring_fft_inverse_kernel(const cx<T>* __restrict__ spec, int64_t spec_stride,
                                                           T* __restrict__ outmap, int64_t npix,
                                                           const RingRec* __restrict__ rings, const FftLen* __restrict__ lens,
                                                           const cx<T>* __restrict__ tw, int logPT,
                                                           const cx<T>* __restrict__ filt)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* s = reinterpret_cast<cx<T>*>(smem_raw);
    const RingRec r = rings[blockIdx.x];
    const FftLen f = lens[r.len_id];
    const int N = r.n, L = N >> 1;
    const cx<T>* __restrict__ D = spec + (int64_t)blockIdx.y * spec_stride + r.spec_off;
    for (int k = threadIdx.x; k < L; k += blockDim.x) {
        cx<T> xk = D[k], xl = D[L - k];
        if (r.shifted) {
            xk = cmul(xk, cispi_ratio<T>((uint32_t)k, (uint32_t)N));
            xl = cmul(xl, cispi_ratio<T>((uint32_t)(L - k), (uint32_t)N));
        }
        const cx<T> xc = cconj(xl);
        const cx<T> a = xk + xc, d = xk - xc;
        const cx<T> wd = cmul(cispi_ratio<T>((uint32_t)(2 * k), (uint32_t)N), d);          // exp(+2 pi i k / N) d
        // Z[k] = a + i wd ; the inverse transform is done as conj(FFT(conj Z))
        s[k] = mk<T>(a.x - wd.y, -(a.y + wd.x));
    }
    __syncthreads();
    fft_len(s, f, tw, logPT, filt);
    cx<T>* __restrict__ o = reinterpret_cast<cx<T>*>(outmap + (int64_t)blockIdx.y * npix + r.pix_off);
    for (int n = threadIdx.x; n < L; n += blockDim.x) {
        const cx<T> z = s[fft_out_index(n, f)];
        o[n] = mk<T>(z.x, -z.y);                                                             // out[2n], out[2n+1]
    }
}

}  // namespace arkcos
