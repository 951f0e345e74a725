// Band step on the 5th-generation tensor cores (steps 4-6 of the hot path for float plans).
//
// The kernel-row phi-transform ("the FFT of the kernel": the dominant cost of the paper's
// implementation) is a pruned cosine sum over the few non-zero samples of the half row,
//     G_ij[m] = sum_u W_ij[u] cos(pi m u s / M),      u = 0 .. K-1  (s = 1: half-step positions included, s = 2: integer grid)
// i.e. for a tile of ring pairs and a tile of modes the dense contraction  G[m, pair] = C[m, u] W[pair, u].  Here it runs
// as tcgen05.mma kind::tf32 with the accumulator in tensor memory: one block owns 128 consecutive modes (TMEM lanes)
// for a whole run of output rings, builds the cosine operand C once, and per tile of TI = 4 output rings stages the rows
// of the up to 32 input rings of the tile's window as the B operand (column = 4 * input ring + output ring, missing
// pairs are zero rows).  FP32 accuracy comes from the 3xTF32 split  C W = C_hi W_lo + C_lo W_hi + C_hi W_hi  with the
// two small terms issued first (measured on B200: 1.1e-7 fractional RMS for K = 24, the level of an FP32 FMA chain;
// in the other order the accumulator's truncation leaves 2.9e-7).
// What stays on the FP32 pipe is the multiply-accumulate over input rings: thread = lane = mode m
// reads G for one input ring and the tile's four output rings with tcgen05.ld and the coefficient Bp_j[m] of ring j and
// of its mirror image from a thread-private shared-memory window that slides with the tile (each coefficient is
// fetched from L2 once per run of rings, by cp.async, while the tensor core works).
//
// KIND 0: class-E rings, half-step parity alternates (HEALPix belt);  1: class-E rings, integer grid (ECP);
// KIND 2: runs of cap rings with one M', single period (M'/2 < N of every ring involved);  3: several periods.
// The fold of the cap kinds and all sign rules are those of band_mac_capchunk_kernel (arkcos_band.cuh).
#pragma once
#include "arkcos_band.cuh"

namespace arkcos {

constexpr int kTcThreads = 128;            // one thread per TMEM lane
constexpr int kTcTI = 4;                   // output rings per tile
constexpr int kTcJW = 32;                  // input rings a tile's window can hold
constexpr int kTcN = kTcTI * kTcJW;        // accumulator columns
constexpr int kTcK = 24;                   // sample positions u per row
constexpr int kTcChunkRings = 24;          // longest run of cap rings handed to one block
constexpr size_t kTcSmemBytes = (size_t)(2 * (kTcK / 4) * 128 + 2 * (kTcK / 4) * kTcN + kTcJW * 128) * 16;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ float tf32_rn(float x)
{
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return __uint_as_float(r);
}

// Shared-memory matrix descriptor, K-major, no swizzle: 8-row x 16-byte core matrices, `sbo` bytes between 8-row groups,
// `lbo` bytes between the two 16-byte chunks along K of one MMA (K = 8 tf32 values).
__device__ __forceinline__ uint64_t tc_smem_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo)
{
    return (uint64_t)((saddr >> 4) & 0x3fffu) | ((uint64_t)((lbo >> 4) & 0x3fffu) << 16) | ((uint64_t)((sbo >> 4) & 0x3fffu) << 32) |
           ((uint64_t)1 << 46);
}

__device__ __forceinline__ void tc_mma_tf32(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}\n"
        ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
}

__device__ __forceinline__ void tc_ld16(uint32_t (&g)[16], uint32_t taddr)
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                 : "=r"(g[0]), "=r"(g[1]), "=r"(g[2]), "=r"(g[3]), "=r"(g[4]), "=r"(g[5]), "=r"(g[6]), "=r"(g[7]), "=r"(g[8]),
                   "=r"(g[9]), "=r"(g[10]), "=r"(g[11]), "=r"(g[12]), "=r"(g[13]), "=r"(g[14]), "=r"(g[15])
                 : "r"(taddr));
}

template <int KIND>
__global__ void __launch_bounds__(kTcThreads, 2)
band_mac_tc_kernel(const CapChunkItem* __restrict__ items, const CapChunk* __restrict__ chunks,
                   const NorthRec* __restrict__ north, const PairRec* __restrict__ pairs, const float* __restrict__ W,
                   const RingRec* __restrict__ rings, int R, const cx<float>* __restrict__ specIn,
                   cx<float>* __restrict__ specOut, int64_t spec_stride)
{
    constexpr bool CAP = KIND >= 2, MULTI = KIND == 3, ALT = KIND == 0;
    constexpr int TI = kTcTI, JW = kTcJW, N = kTcN, K = kTcK, KC = K / 4;
    static_assert(TI == 4, "column = 4 * input ring + output ring");
    extern __shared__ __align__(128) unsigned char tc_smem[];
    float4* sA = reinterpret_cast<float4*>(tc_smem);            // [hi / lo][KC][128 modes]: cos(pi m u s / M), u = 4 kc .. 4 kc + 3
    float4* sB = sA + 2 * KC * 128;                              // [hi / lo][KC][N columns]: row samples of the tile's ring pairs
    float4* sV = sB + 2 * KC * N;                                // [JW slots][128 threads]: (Bp_j[m], Bp_jS[m]) of window ring j
    __shared__ __align__(8) uint64_t bar;
    __shared__ uint32_t s_tmem;
    __shared__ int4 sJ[JW];                                      // window ring: spectrum offsets (N, S), N_j | shifted << 31, magic
    __shared__ int sPlo[TI], sJ0[TI], sNp[TI], sUmax;

    const int t = (int)threadIdx.x, warp = t >> 5;
    const CapChunkItem it = items[blockIdx.x];
    const CapChunk ch = chunks[it.chunk];
    const int M = ch.M, Mh = M >> 1;
    const int m_raw = it.bx * 128 + t, m = min(m_raw, Mh);
    const cx<float>* __restrict__ in = specIn + (int64_t)blockIdx.y * spec_stride;
    cx<float>* __restrict__ out = specOut + (int64_t)blockIdx.y * spec_stride;

    // ---- A operand: the cosines of this block's 128 modes, split into TF32 hi + lo ------------------------------------
    {
        const uint32_t twoM = 2u * (uint32_t)M, step = ALT ? 1u : 2u;
        const cx<float> rot = cispi_ratio<float>(((uint32_t)m * step) % twoM, (uint32_t)M);
        cx<float> c = mk<float>(1.f, 0.f);
        float hi[4], lo[4];
#pragma unroll
        for (int u = 0; u < K; ++u) {
            if ((u & 3) == 0) c = cispi_ratio<float>(((uint32_t)m * step * (uint32_t)u) % twoM, (uint32_t)M);
            else c = cmul(c, rot);
            hi[u & 3] = tf32_rn(c.x);
            lo[u & 3] = tf32_rn(c.x - hi[u & 3]);
            if ((u & 3) == 3) {
                sA[(u >> 2) * 128 + t] = make_float4(hi[0], hi[1], hi[2], hi[3]);
                sA[(KC + (u >> 2)) * 128 + t] = make_float4(lo[0], lo[1], lo[2], lo[3]);
            }
        }
    }
    for (int k = t; k < JW * 128; k += kTcThreads) sV[k] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (t == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&bar)));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "r"(N));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = s_tmem;
    // instruction descriptor: D = f32, A = B = tf32, both K-major, N >> 3 at bit 17, M >> 4 at bit 24
    constexpr uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);

    // periodic extension of a stored half spectrum (reading R8): m = w N_j + r; above N_j/2 the conjugate of N_j - r
    auto ext_index = [](int mm, int nj_sh, uint32_t magic) {
        const int Nj = nj_sh & 0x7fffffff, w = MULTI ? (int)__umulhi((uint32_t)mm, magic) : 0, r = mm - w * Nj;
        return 2 * r > Nj ? Nj - r : r;
    };

    uint32_t phase = 0;
    int jhave = -1;                                              // highest ring whose coefficients sit in the window
    for (int tile = 0; tile < ch.n; tile += TI) {
        const int nti = min(TI, ch.n - tile), i0 = ch.i0 + tile;
        const int p_first = north[i0].pair_lo, p_last = north[i0 + nti - 1].pair_hi;
        const int jlo = pairs[p_first].j, jhi = pairs[p_last - 1].j, jw = jhi - jlo + 1;
        const int jnew = max(jhave + 1, jlo);
        __syncthreads();        // the previous tile is done with the accumulator, the B operand and the tile records
        if (t < TI) {
            const NorthRec nr = north[i0 + min(t, nti - 1)];
            sPlo[t] = nr.pair_lo;
            sJ0[t] = pairs[nr.pair_lo].j;
            sNp[t] = t < nti ? nr.pair_hi - nr.pair_lo : 0;
        }
        if (t == 0) sUmax = 1;
        for (int j = jnew + t; j <= jhi; j += kTcThreads) {
            const RingRec rj = rings[j];
            sJ[j & (JW - 1)] = make_int4((int)rj.spec_off, (int)rings[R - 1 - j].spec_off, rj.n | (rj.shifted ? (int)0x80000000 : 0),
                                         MULTI ? (int)(uint32_t)((0x100000000ull + (uint64_t)rj.n - 1ull) / (uint64_t)rj.n) : 0);
        }
        __syncthreads();
        // ---- B operand: one column per ring pair of the tile, TF32 hi + lo; missing pairs and the tails are zero ------
        {
            int umax = 0;
            for (int idx = t; idx < N * KC; idx += kTcThreads) {
                const int kc = idx / N, c = idx - kc * N, jj = c >> 2, ii = c & 3;
                const int pj = jlo + jj - sJ0[ii];
                float4 w = make_float4(0.f, 0.f, 0.f, 0.f);
                if (pj >= 0 && pj < sNp[ii]) {
                    const PairRec& pr = pairs[sPlo[ii] + pj];
                    const int cnt = pr.cnt, cnt4 = (cnt + 3) & ~3;
                    if (ALT) {
                        const int par = pr.par;
                        if (kc == 0) umax = max(umax, 2 * cnt - 1 + par);
                        if (2 * kc < cnt4) {
                            const float2 ww = *reinterpret_cast<const float2*>(W + pr.woff + 2 * kc);
                            w = par ? make_float4(0.f, ww.x, 0.f, ww.y) : make_float4(ww.x, 0.f, ww.y, 0.f);
                        }
                    } else {
                        if (kc == 0) umax = max(umax, cnt);
                        if (4 * kc < cnt4) w = *reinterpret_cast<const float4*>(W + pr.woff + 4 * kc);
                    }
                }
                const float4 h = make_float4(tf32_rn(w.x), tf32_rn(w.y), tf32_rn(w.z), tf32_rn(w.w));
                sB[kc * N + c] = h;
                sB[(KC + kc) * N + c] = make_float4(tf32_rn(w.x - h.x), tf32_rn(w.y - h.y), tf32_rn(w.z - h.z), tf32_rn(w.w - h.w));
            }
            if (umax > 1) atomicMax(&sUmax, umax);
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (t == 0) {
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const int ksteps = min(K / 8, (sUmax + 7) >> 3);
            const uint32_t a0 = smem_u32(sA), b0 = smem_u32(sB);
            uint32_t acc_flag = 0;
#pragma unroll
            for (int s = 0; s < 3; ++s) {                        // (hi, lo), (lo, hi), then (hi, hi): small terms first
                const int ha = s == 1 ? 1 : 0, hb = s == 0 ? 1 : 0;
                for (int ks = 0; ks < ksteps; ++ks) {
                    const uint64_t da = tc_smem_desc(a0 + (uint32_t)((ha * KC + 2 * ks) * 128 * 16), 128 * 16, 128);
                    const uint64_t db = tc_smem_desc(b0 + (uint32_t)((hb * KC + 2 * ks) * N * 16), N * 16, 128);
                    tc_mma_tf32(tmem, da, db, idesc, acc_flag);
                    acc_flag = 1;
                }
            }
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&bar)) : "memory");
        }
        // ---- window: coefficients of the rings that enter with this tile, fetched while the tensor core works ---------
        for (int j = jnew; j <= jhi; ++j) {
            const int4 rj = sJ[j & (JW - 1)];
            const int idx = CAP ? ext_index(m, rj.z, (uint32_t)rj.w) : m;
            float4* dst = sV + (j & (JW - 1)) * 128 + t;
            cp_async8(dst, in + rj.x + idx);
            cp_async8(reinterpret_cast<char*>(dst) + 8, in + rj.y + idx);
        }
        cp_async_commit();
        jhave = jhi;
        {
            uint32_t done = 0;
            while (!done)
                asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                             : "=r"(done) : "r"(smem_u32(&bar)), "r"(phase) : "memory");
            phase ^= 1u;
        }
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        cp_async_wait<0>();

        // ---- multiply-accumulate over the window's input rings ---------------------------------------------------------
        float2 acc[TI][2];
#pragma unroll
        for (int ii = 0; ii < TI; ++ii) acc[ii][0] = acc[ii][1] = make_float2(0.f, 0.f);
        const uint32_t tbase = tmem + ((uint32_t)(warp * 32) << 16);
        for (int jj0 = 0; jj0 < jw; jj0 += 4) {
            uint32_t g[16];
            tc_ld16(g, tbase + (uint32_t)(jj0 * TI));
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                if (jj0 + q < jw) {
                    const int slot = (jlo + jj0 + q) & (JW - 1);
                    float4 v = sV[slot * 128 + t];
                    if (CAP) {
                        // reflection conjugates; a shifted ring changes sign on reflection and on every odd period
                        const int4 rj = sJ[slot];
                        const int Nj = rj.z & 0x7fffffff, w = MULTI ? (int)__umulhi((uint32_t)m, (uint32_t)rj.w) : 0, r = m - w * Nj;
                        const bool refl = 2 * r > Nj;
                        const uint32_t sre = (rj.z < 0 && (refl != ((w & 1) != 0))) ? 0x80000000u : 0u;
                        const uint32_t sim = sre ^ (refl ? 0x80000000u : 0u);
                        v.x = __uint_as_float(__float_as_uint(v.x) ^ sre); v.y = __uint_as_float(__float_as_uint(v.y) ^ sim);
                        v.z = __uint_as_float(__float_as_uint(v.z) ^ sre); v.w = __uint_as_float(__float_as_uint(v.w) ^ sim);
                    }
#pragma unroll
                    for (int ii = 0; ii < TI; ++ii) {
                        const float G = __uint_as_float(g[q * TI + ii]);
                        acc[ii][0] = ffma2(make_float2(G, G), make_float2(v.x, v.y), acc[ii][0]);
                        acc[ii][1] = ffma2(make_float2(G, G), make_float2(v.z, v.w), acc[ii][1]);
                    }
                }
            }
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");

        // ---- output: class E stores its mode; cap runs fold onto the ring's own modes --------------------
#pragma unroll
        for (int ii = 0; ii < TI; ++ii) {
            if (ii < nti) {
                const int i = i0 + ii, iS = R - 1 - i;
                const RingRec ri = rings[i];
                const int64_t offS = rings[iS].spec_off;
                if (!CAP) {
                    out[ri.spec_off + m] = mk<float>(acc[ii][0].x, acc[ii][0].y);
                    if (iS != i) out[offS + m] = mk<float>(acc[ii][1].x, acc[ii][1].y);
                } else if (m_raw <= Mh) {
                    const float hw = (2 * m == M) ? 0.5f : 1.f;          // the +-M/2 bins carry half the Nyquist term each
                    const int w = MULTI ? m / ri.n : 0, r = m - w * ri.n;
                    const float s0 = (ri.shifted && (w & 1)) ? -1.f : 1.f, s1 = ri.shifted ? -s0 : s0;
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        if (h == 1 && iS == i) continue;
                        float2* dst = reinterpret_cast<float2*>(out + (h ? offS : ri.spec_off));
                        const float tx = hw * acc[ii][h].x, ty = hw * acc[ii][h].y;
                        if (2 * r <= ri.n) atomicAdd(dst + r, make_float2(s0 * tx, s0 * ty));
                        if (2 * r >= ri.n) atomicAdd(dst + (ri.n - r), make_float2(s1 * tx, -s1 * ty));
                        if (MULTI && r == 0 && w > 0) atomicAdd(dst, make_float2(s0 * tx, -s0 * ty));     // m = -w N_i folds onto 0 as well
                    }
                }
            }
        }
    }
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(N));
}

}  // namespace arkcos
