// Band kernels for plans with cached kernel spectra (options.cache_kernel_spectra): the row transforms
//     G_ij[m] = sum_t W_ij[t] cos(m (2t + par) pi / M),   m = 0 .. M/2,
// of all northern ring pairs are computed once at plan time and kept in HBM (the same beam is applied to
// the maps of many detectors), so that a convolution only streams them: the band step becomes
// bandwidth-bound (4 bytes of G per (pair, mode) against 12-20 FMAs), row length no longer matters, and NM maps that
// share the kernel are accumulated from one read of G.  Structure and index conventions are those of
// band_mac_eq_kernel / band_mac_capchunk_kernel (arkcos_band.cuh); goff[p] is the first float4 of pair p's row in Gc.
#pragma once
#include "arkcos_band.cuh"

namespace arkcos {

constexpr uint32_t kNoPair = 0xffffffffu;

// Plan time: one block row per pair.  grid = (pairs, ceil((M/2 + 1) / 256)), 256 threads.
__global__ void __launch_bounds__(256)
kernel_spectra_kernel(const PairRec* __restrict__ pairs, const float* __restrict__ W, const uint32_t* __restrict__ goff,
                      float* __restrict__ Gc)
{
    const PairRec pr = pairs[blockIdx.x];
    const int M = pr.M, Mh = M >> 1, m = (int)blockIdx.y * 256 + (int)threadIdx.x;
    if (m > Mh) return;
    const float* __restrict__ w = W + pr.woff;
    const uint32_t twoM = 2u * (uint32_t)M;
    const cx<float> rot = cispi_ratio<float>((2u * (uint32_t)m) % twoM, (uint32_t)M);
    float G = 0.f;
    cx<float> c = mk<float>(1.f, 0.f);
    for (int t = 0; t < pr.cnt; ++t) {
        if ((t & 7) == 0) {
            const uint64_t q = ((uint64_t)m * (uint64_t)(2 * t + pr.par)) % (uint64_t)twoM;
            c = cispi_ratio<float>((uint32_t)q, (uint32_t)M);
        } else c = cmul(c, rot);
        G = fmaf(w[t], c.x, G);
    }
    Gc[(size_t)goff[blockIdx.x] * 4 + m] = G;
}

// Class-E runs (equatorial belt, ECP) from cached spectra.  grid = (mode blocks of 256, chunks, ceil(nmaps / NM)),
// block = 256 / MT threads with MT adjacent modes each: <NM = 4, MT = 1> reads G once for four maps with the accumulators
// of <NM = 2, MT = 2> (G is what the kernel streams from HBM: 4 bytes per (pair, mode) and NM maps).
// Dynamic shared memory: kCachedSlots x NM x 2 x 256 coefficients.
constexpr int kCachedSlots = 4;
template <int NM> constexpr size_t cached_smem_bytes() { return (size_t)kCachedSlots * NM * 2 * 256 * sizeof(float2); }
template <int TI, int NM, int MT>
__global__ void __launch_bounds__(256 / MT)
band_mac_eq_cached_kernel(const EqChunk* __restrict__ chunks, const NorthRec* __restrict__ north,
                          const PairRec* __restrict__ pairs, const uint32_t* __restrict__ goff,
                          const float* __restrict__ Gc, const RingRec* __restrict__ rings, int R,
                          const cx<float>* __restrict__ specIn, cx<float>* __restrict__ specOut, int64_t spec_stride,
                          int nmaps)
{
    constexpr int NT = 256 / MT;
    __shared__ uint32_t sG[TI * kEqJMax];                          // [ii][jj]: row of pair (i0 + ii, jlo + jj) or kNoPair
    __shared__ int2 sJ[kEqJMax];                                   // spectrum offsets of input ring jlo + jj (N, S)
    extern __shared__ __align__(16) unsigned char cached_smem[];
    // in-flight input-ring coefficients: [slot][map][hemisphere][256 modes]
    float2 (*sB)[NM][2][256] = reinterpret_cast<float2 (*)[NM][2][256]>(cached_smem);
    const EqChunk ch = chunks[blockIdx.y];
    const int M = rings[ch.i0].n, Mh = M >> 1;
    const int m0 = (int)blockIdx.x * 256 + MT * (int)threadIdx.x;
    const int m0c = min(m0, Mh - MT);
    const int map0 = (int)blockIdx.z * NM;
    const cx<float>* __restrict__ in0 = specIn + (int64_t)map0 * spec_stride + m0c;
    cx<float>* __restrict__ out = specOut + (int64_t)map0 * spec_stride;
    const float* __restrict__ Gm = Gc + m0c;

    for (int tile = 0; tile < ch.n; tile += TI) {
        const int nti = min(TI, ch.n - tile), i0 = ch.i0 + tile;
        const int p_first = north[i0].pair_lo, p_last = north[i0 + nti - 1].pair_hi;
        const int jlo = pairs[p_first].j, jw = pairs[p_last - 1].j - jlo + 1;
        __syncthreads();
        for (int k = threadIdx.x; k < TI * kEqJMax; k += NT) sG[k] = kNoPair;
        for (int jj = threadIdx.x; jj < jw; jj += NT)
            sJ[jj] = make_int2((int)rings[jlo + jj].spec_off, (int)rings[R - 1 - jlo - jj].spec_off);
        __syncthreads();
        for (int p = p_first + (int)threadIdx.x; p < p_last; p += NT) {
            int ii = 0;
#pragma unroll
            for (int q = 1; q < TI; ++q) ii += (q < nti && p >= north[i0 + q].pair_lo) ? 1 : 0;
            sG[ii * kEqJMax + (pairs[p].j - jlo)] = goff[p];
        }
        __syncthreads();
        cx<float> acc[NM][TI][2][MT];
#pragma unroll
        for (int q = 0; q < NM; ++q)
#pragma unroll
            for (int ii = 0; ii < TI; ++ii)
#pragma unroll
                for (int h = 0; h < 2; ++h)
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) acc[q][ii][h][mt] = mk<float>(0.f, 0.f);
        auto fetch = [&](int jj) {
            if (jj < jw) {
                const int2 off = sJ[jj];
#pragma unroll
                for (int q = 0; q < NM; ++q) {
                    if (map0 + q < nmaps) {
                        if (MT == 2) {
                            cp_async16(&sB[jj & 3][q][0][MT * threadIdx.x], in0 + (int64_t)q * spec_stride + off.x);
                            cp_async16(&sB[jj & 3][q][1][MT * threadIdx.x], in0 + (int64_t)q * spec_stride + off.y);
                        } else {
                            cp_async8(&sB[jj & 3][q][0][threadIdx.x], in0 + (int64_t)q * spec_stride + off.x);
                            cp_async8(&sB[jj & 3][q][1][threadIdx.x], in0 + (int64_t)q * spec_stride + off.y);
                        }
                    }
                }
            }
            cp_async_commit();
        };
        auto loadG = [&](int jj, float2 (&g)[TI]) {
#pragma unroll
            for (int ii = 0; ii < TI; ++ii) {
                const uint32_t o = sG[ii * kEqJMax + min(jj, jw - 1)];
                if (MT == 2) g[ii] = o != kNoPair ? *reinterpret_cast<const float2*>(Gm + (size_t)o * 4) : make_float2(0.f, 0.f);
                else g[ii] = make_float2(o != kNoPair ? Gm[(size_t)o * 4] : 0.f, 0.f);
            }
        };
        fetch(0); fetch(1); fetch(2);
        float2 gn[TI];
        loadG(0, gn);
        for (int jj = 0; jj < jw; ++jj) {
            float2 g[TI];
#pragma unroll
            for (int ii = 0; ii < TI; ++ii) g[ii] = gn[ii];
            loadG(jj + 1, gn);
            fetch(jj + 3);
            cp_async_wait<3>();
#pragma unroll
            for (int q = 0; q < NM; ++q) {
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const float2 b0 = sB[jj & 3][q][h][MT * threadIdx.x];
                    const float2 b1 = MT == 2 ? sB[jj & 3][q][h][MT * threadIdx.x + MT - 1] : b0;
#pragma unroll
                    for (int ii = 0; ii < TI; ++ii) {
                        const float2 a0 = ffma2(make_float2(g[ii].x, g[ii].x), b0, make_float2(acc[q][ii][h][0].x, acc[q][ii][h][0].y));
                        acc[q][ii][h][0] = mk<float>(a0.x, a0.y);
                        if (MT == 2) {
                            const float2 a1 = ffma2(make_float2(g[ii].y, g[ii].y), b1,
                                                    make_float2(acc[q][ii][h][MT - 1].x, acc[q][ii][h][MT - 1].y));
                            acc[q][ii][h][MT - 1] = mk<float>(a1.x, a1.y);
                        }
                    }
                }
            }
        }
#pragma unroll
        for (int ii = 0; ii < TI; ++ii) {
            if (ii < nti && m0 < Mh) {
                const int i = i0 + ii, iS = R - 1 - i;
                const int64_t offN = rings[i].spec_off, offS = rings[iS].spec_off;
#pragma unroll
                for (int q = 0; q < NM; ++q) {
                    if (map0 + q >= nmaps) continue;
                    cx<float>* o = out + (int64_t)q * spec_stride;
                    if (MT == 2) {
                        *reinterpret_cast<float4*>(o + offN + m0) =
                            make_float4(acc[q][ii][0][0].x, acc[q][ii][0][0].y, acc[q][ii][0][MT - 1].x, acc[q][ii][0][MT - 1].y);
                        if (iS != i)
                            *reinterpret_cast<float4*>(o + offS + m0) =
                                make_float4(acc[q][ii][1][0].x, acc[q][ii][1][0].y, acc[q][ii][1][MT - 1].x, acc[q][ii][1][MT - 1].y);
                    } else {
                        o[offN + m0] = acc[q][ii][0][0];
                        if (iS != i) o[offS + m0] = acc[q][ii][1][0];
                    }
                }
            }
        }
    }
}


// Runs of cap rings with one grid length M' from cached spectra (see band_mac_capchunk_kernel for the extension of the
// input coefficients and the fold).  grid = (items, ceil(nmaps / NM)).
// block = 256 / MT threads, MT adjacent modes each (an item is a block of 256 modes either way).
template <int TI, int NM, bool MULTI, int MT>
__global__ void __launch_bounds__(256 / MT)
band_mac_capchunk_cached_kernel(const CapChunkItem* __restrict__ items, const CapChunk* __restrict__ chunks,
                                const NorthRec* __restrict__ north, const PairRec* __restrict__ pairs,
                                const uint32_t* __restrict__ goff, const float* __restrict__ Gc,
                                const RingRec* __restrict__ rings, int R, const cx<float>* __restrict__ specIn,
                                cx<float>* __restrict__ specOut, int64_t spec_stride, int nmaps)
{
    constexpr int NT = 256 / MT;
    __shared__ uint32_t sG[TI * kEqJMax];
    __shared__ int4 sJ[kEqJMax];                                   // input ring jlo + jj: spectrum offsets (N, S), N_j, shifted
    const CapChunkItem it = items[blockIdx.x];
    const CapChunk ch = chunks[it.chunk];
    const int M = ch.M, Mh = M >> 1;
    const int m0 = it.bx * 256 + MT * (int)threadIdx.x;      // modes m0 .. m0 + MT - 1 (MT = 2: m0 even)
    const int mA = min(m0, Mh), mB = min(m0 + MT - 1, Mh);
    const int map0 = (int)blockIdx.y * NM;
    const cx<float>* __restrict__ in = specIn + (int64_t)map0 * spec_stride;
    cx<float>* __restrict__ out = specOut + (int64_t)map0 * spec_stride;
    const float* __restrict__ Gm = Gc + (MT == 2 ? min(m0, Mh & ~1) : min(m0, Mh));          // rows are padded to a multiple of 4 floats
    // periodic extension of the stored half spectrum of a ring (N_j, shifted flag in bit 31, magic = ceil(2^32 / N_j)):
    // m = w N_j + r; above N_j/2 the coefficient is the conjugate of the one at N_j - r; a shifted ring changes sign on
    // reflection and on every odd period (reading R8)
    // (MULTI = false: the plan guarantees M'/2 < N_j and M'/2 < N_i for every ring involved, period 0 only)
    auto ext_index = [](int m, int nj_sh, uint32_t magic) {
        const int Nj = nj_sh & 0x7fffffff, w = MULTI ? (int)__umulhi((uint32_t)m, magic) : 0, r = m - w * Nj;
        return 2 * r > Nj ? Nj - r : r;
    };
    auto ext_value = [](cx<float> b, int m, int nj_sh, uint32_t magic) {
        const int Nj = nj_sh & 0x7fffffff, w = MULTI ? (int)__umulhi((uint32_t)m, magic) : 0, r = m - w * Nj;
        const bool refl = 2 * r > Nj;
        if (refl) b.y = -b.y;
        if (nj_sh < 0 && (refl != ((w & 1) != 0))) { b.x = -b.x; b.y = -b.y; }
        return b;
    };

    for (int tile = 0; tile < ch.n; tile += TI) {
        const int nti = min(TI, ch.n - tile), i0 = ch.i0 + tile;
        const int p_first = north[i0].pair_lo, p_last = north[i0 + nti - 1].pair_hi;
        const int jlo = pairs[p_first].j, jw = pairs[p_last - 1].j - jlo + 1;
        __syncthreads();
        for (int k = threadIdx.x; k < TI * kEqJMax; k += NT) sG[k] = kNoPair;
        for (int jj = threadIdx.x; jj < jw; jj += NT) {
            const RingRec rj = rings[jlo + jj];
            sJ[jj] = make_int4((int)rj.spec_off, (int)rings[R - 1 - jlo - jj].spec_off, rj.n | (rj.shifted ? (int)0x80000000 : 0),
                               MULTI ? (int)(uint32_t)((0x100000000ull + (uint64_t)rj.n - 1ull) / (uint64_t)rj.n) : 0);
        }
        __syncthreads();
        for (int p = p_first + (int)threadIdx.x; p < p_last; p += NT) {
            int ii = 0;
#pragma unroll
            for (int q = 1; q < TI; ++q) ii += (q < nti && p >= north[i0 + q].pair_lo) ? 1 : 0;
            sG[ii * kEqJMax + (pairs[p].j - jlo)] = goff[p];
        }
        __syncthreads();
        cx<float> acc[NM][TI][2][MT];
#pragma unroll
        for (int q = 0; q < NM; ++q)
#pragma unroll
            for (int ii = 0; ii < TI; ++ii)
#pragma unroll
                for (int h = 0; h < 2; ++h)
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) acc[q][ii][h][mt] = mk<float>(0.f, 0.f);
        cx<float> nx[NM][2][MT];
        float2 gn[TI];
        auto fetch = [&](int jj) {
            const int jc = min(jj, jw - 1);
            const int4 rj = sJ[jc];
            const int ia = ext_index(mA, rj.z, (uint32_t)rj.w), ib = ext_index(mB, rj.z, (uint32_t)rj.w);
#pragma unroll
            for (int q = 0; q < NM; ++q) {
                const cx<float>* __restrict__ b = in + (int64_t)(map0 + q < nmaps ? q : 0) * spec_stride;
                nx[q][0][0] = b[rj.x + ia];
                nx[q][1][0] = b[rj.y + ia];
                if (MT == 2) { nx[q][0][MT - 1] = b[rj.x + ib]; nx[q][1][MT - 1] = b[rj.y + ib]; }
            }
#pragma unroll
            for (int ii = 0; ii < TI; ++ii) {
                const uint32_t o = sG[ii * kEqJMax + jc];
                if (MT == 2) gn[ii] = o != kNoPair ? *reinterpret_cast<const float2*>(Gm + (size_t)o * 4) : make_float2(0.f, 0.f);
                else gn[ii] = make_float2(o != kNoPair ? Gm[(size_t)o * 4] : 0.f, 0.f);
            }
        };
        fetch(0);
        for (int jj = 0; jj < jw; ++jj) {
            const int4 rj = sJ[jj];
            cx<float> v[NM][2][MT];
            float2 g[TI];
#pragma unroll
            for (int q = 0; q < NM; ++q)
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    v[q][h][0] = ext_value(nx[q][h][0], mA, rj.z, (uint32_t)rj.w);
                    if (MT == 2) v[q][h][MT - 1] = ext_value(nx[q][h][MT - 1], mB, rj.z, (uint32_t)rj.w);
                }
#pragma unroll
            for (int ii = 0; ii < TI; ++ii) g[ii] = gn[ii];
            fetch(jj + 1);
#pragma unroll
            for (int q = 0; q < NM; ++q)
#pragma unroll
                for (int h = 0; h < 2; ++h)
#pragma unroll
                    for (int ii = 0; ii < TI; ++ii) {
                        const float2 a0 = ffma2(make_float2(g[ii].x, g[ii].x), make_float2(v[q][h][0].x, v[q][h][0].y),
                                                make_float2(acc[q][ii][h][0].x, acc[q][ii][h][0].y));
                        acc[q][ii][h][0] = mk<float>(a0.x, a0.y);
                        if (MT == 2) {
                            const float2 a1 = ffma2(make_float2(g[ii].y, g[ii].y), make_float2(v[q][h][MT - 1].x, v[q][h][MT - 1].y),
                                                    make_float2(acc[q][ii][h][MT - 1].x, acc[q][ii][h][MT - 1].y));
                            acc[q][ii][h][MT - 1] = mk<float>(a1.x, a1.y);
                        }
                    }
        }
#pragma unroll
        for (int ii = 0; ii < TI; ++ii) {
            if (ii < nti) {
                const int i = i0 + ii, iS = R - 1 - i;
                const RingRec ri = rings[i];
                const int64_t offS = rings[iS].spec_off;
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    const int m = m0 + mt;
                    if (m > Mh) continue;
                    const float hw = (2 * m == M) ? 0.5f : 1.f;
                    const int w = MULTI ? m / ri.n : 0, r = m - w * ri.n;
                    const float s0 = (ri.shifted && (w & 1)) ? -1.f : 1.f, s1 = ri.shifted ? -s0 : s0;
#pragma unroll
                    for (int q = 0; q < NM; ++q) {
                        if (map0 + q >= nmaps) continue;
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            if (h == 1 && iS == i) continue;
                            float2* dst = reinterpret_cast<float2*>(out + (int64_t)q * spec_stride + (h ? offS : ri.spec_off));
                            const float tx = hw * acc[q][ii][h][mt].x, ty = hw * acc[q][ii][h][mt].y;
                            if (2 * r <= ri.n) atomicAdd(dst + r, make_float2(s0 * tx, s0 * ty));
                            if (2 * r >= ri.n) atomicAdd(dst + (ri.n - r), make_float2(s1 * tx, -s1 * ty));
                            if (MULTI && r == 0 && w > 0) atomicAdd(dst, make_float2(s0 * tx, -s0 * ty));     // m = -w N_i folds onto 0 as well
                        }
                    }
                }
            }
        }
    }
}

}  // namespace arkcos
