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
#include "arkcos_band_tc.hpp"

namespace arkcos {

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

__device__ __forceinline__ void tc_commit(uint64_t* bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void tc_ld16(uint32_t (&g)[16], uint32_t taddr)
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                 : "=r"(g[0]), "=r"(g[1]), "=r"(g[2]), "=r"(g[3]), "=r"(g[4]), "=r"(g[5]), "=r"(g[6]), "=r"(g[7]), "=r"(g[8]),
                   "=r"(g[9]), "=r"(g[10]), "=r"(g[11]), "=r"(g[12]), "=r"(g[13]), "=r"(g[14]), "=r"(g[15])
                 : "r"(taddr));
}

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t done = 0;
    while (!done)
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
}

// Warp-specialised: the producer warpgroup (threads 256 .. 383, thread = accumulator column) converts the rows of tile
// k + 1 into the B operand (two stages) and its first thread issues the MMAs of both blocks of modes into TMEM stage
// (k + 1) & 1, while the two consumer warpgroups (thread = mode) multiply-accumulate tile k out of TMEM stage k & 1.
// mbarriers: full[s] (MMAs of the stage done), empty[s] (all eight consumer warps have read the stage), rows[s] (the MMAs
// that read B-operand stage s are done).
template <int KIND, class CFG>
__global__ void __launch_bounds__(CFG::threads, 1)
band_mac_tc_kernel(const TcItem* __restrict__ items, const TcChunk* __restrict__ chunks, const TcTile* __restrict__ tiles,
                   const uint32_t* __restrict__ cols, const TcRing* __restrict__ ringtab, const float* __restrict__ W, int R,
                   const cx<float>* __restrict__ specIn, cx<float>* __restrict__ specOut, int64_t spec_stride)
{
    constexpr bool CAP = KIND >= 2, MULTI = KIND == 3, ALT = KIND == 0;
    constexpr int TI = CFG::TI, JW = CFG::JW, N = CFG::N, K = CFG::K, KC = K / 4, MT = CFG::MT;
    constexpr int kTcConsumers = CFG::consumers, kTcProducers = CFG::producers;
    constexpr int kTmemCols = 2 * MT * N <= 256 ? 256 : 512;       // two stages of MT x N accumulator columns (a power of two)
    static_assert(TI == 4, "column = 4 * input ring + output ring");
    extern __shared__ __align__(128) unsigned char tc_smem[];
    float4* sA = reinterpret_cast<float4*>(tc_smem);            // [block of modes][hi / lo][KC][128 modes]: cos(pi m u s / M), u = 4 kc .. 4 kc + 3
    float4* sB = sA + MT * 2 * KC * 128;                         // [stage][hi / lo][KC][N columns]: row samples of the tile's ring pairs
    float4* sV = sB + 2 * 2 * KC * N;                            // [block of modes][JW slots][128 threads]: (Bp_j[m], Bp_jS[m]) of window ring j
    __shared__ __align__(8) uint64_t bar_full[2], bar_empty[2], bar_rows[2];
    __shared__ uint32_t s_tmem;
    __shared__ int sUmax[2];
    __shared__ TcTile sTiles[kTcMaxTiles];                       // records of the run's tiles and of the rings of their windows
    __shared__ TcRing sRings[kTcMaxWindow];

    const int t = (int)threadIdx.x, warp = t >> 5;
    const TcItem it = items[blockIdx.x];
    const TcChunk ch = chunks[it.chunk];
    const int M = ch.M, Mh = M >> 1;
    const int ntiles = (ch.n + TI - 1) / TI;
    const bool producer = t >= kTcConsumers;
    const int wg = t >> 7, l128 = t & 127;                       // consumer: block of modes, lane within it
    const int m_raw = (it.bx * MT + wg) * 128 + l128, m = min(m_raw, Mh);

    const cx<float>* __restrict__ in = specIn + (int64_t)blockIdx.y * spec_stride;
    cx<float>* __restrict__ out = specOut + (int64_t)blockIdx.y * spec_stride;
    const uint32_t sv0 = smem_u32(sV + wg * JW * 128 + l128);      // this thread's slot 0; slot s at + 2048 s bytes
    // periodic extension of a stored half spectrum (reading R8): m = w N_j + r; above N_j/2 the conjugate of N_j - r
    auto ext_index = [](int mm, int nj_sh, uint32_t magic) {
        const int Nj = nj_sh & 0x7fffffff, w = MULTI ? (int)__umulhi((uint32_t)mm, magic) : 0, r = mm - w * Nj;
        return 2 * r > Nj ? Nj - r : r;
    };
    auto fetch_ring = [&](int j, const TcRing& rj) {
        const int idx = CAP ? ext_index(m, rj.n_sh, rj.magic) : m;
        const uint32_t dst = sv0 + 2048u * (uint32_t)(j % JW);
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(in + rj.offN + idx) : "memory");
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst + 8u), "l"(in + rj.offS + idx) : "memory");
    };
    if (!producer) {
        // ---- A operand: the cosines of this warpgroup's 128 modes, split into TF32 hi + lo ----------------------------
        float4* sAw = sA + wg * 2 * KC * 128;
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
                sAw[(u >> 2) * 128 + l128] = make_float4(hi[0], hi[1], hi[2], hi[3]);
                sAw[(KC + (u >> 2)) * 128 + l128] = make_float4(lo[0], lo[1], lo[2], lo[3]);
            }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        // the window starts out finite: accumulator columns past the tile's window are exact zeros, but 0 * garbage is not
        for (int sl = 0; sl < JW; ++sl) sV[(wg * JW + sl) * 128 + l128] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    const int jbase = tiles[ch.tile0].jlo;                      // first ring of the run's first window
    if (producer) {
        const int c = t - kTcConsumers;
        const int4* __restrict__ src = reinterpret_cast<const int4*>(tiles + ch.tile0);
        int4* dst = reinterpret_cast<int4*>(sTiles);
        for (int q = c; q < ntiles * (int)(sizeof(TcTile) / 16); q += kTcProducers) dst[q] = src[q];
        const int jlast = tiles[ch.tile0 + ntiles - 1].jhi;
        const int4* __restrict__ rsrc = reinterpret_cast<const int4*>(ringtab + jbase);
        int4* rdst = reinterpret_cast<int4*>(sRings);
        for (int q = c; q <= jlast - jbase; q += kTcProducers) rdst[q] = rsrc[q];
    }
    if (t == 0) {
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            mbar_init(&bar_full[s], 1);
            mbar_init(&bar_empty[s], kTcConsumers / 32);
            mbar_init(&bar_rows[s], 1);
            sUmax[s] = 1;
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == kTcConsumers / 32) {                             // the first producer warp owns the tensor-memory allocation
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "r"(kTmemCols));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = s_tmem;

    if (producer) {
        // =================================== rows -> B operand -> MMAs =========================================
        const int c = t - kTcConsumers;
        // instruction descriptor: D = f32, A = B = tf32, both K-major, N >> 3 at bit 17, M >> 4 at bit 24
        constexpr uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
        // Rows travel two tiles ahead of their conversion: the raw samples of tile k sit in buffer k & 1, which is refilled
        // with tile k + 2 once tile k has been converted (the loads have a whole tile to arrive); column words three ahead.
        float4 raw[2][KC];
        auto load_row = [&](float4 (&dst)[KC], uint32_t cw) {
            const bool have = cw != kTcNoPair;
            const int cnt4 = have ? (int)(((cw >> 25) & 63u) + 3u) & ~3 : 0;
            const float* __restrict__ w = W + (size_t)(cw & 0x1ffffffu) * 4;
    #pragma unroll
            for (int kc = 0; kc < KC; ++kc) {
                dst[kc] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (ALT) {                                       // two samples per group of four positions (see convert)
                    if (2 * kc < cnt4) {
                        const float2 ww = *reinterpret_cast<const float2*>(w + 2 * kc);
                        dst[kc].x = ww.x;
                        dst[kc].y = ww.y;
                    }
                } else if (4 * kc < cnt4) dst[kc] = *reinterpret_cast<const float4*>(w + 4 * kc);
            }
        };
        const uint32_t* __restrict__ colp = cols + (size_t)ch.tile0 * N + c;
        auto col_word = [&](int k) { return k < ntiles ? colp[(size_t)k * N] : kTcNoPair; };
        uint32_t cwv[2] = {col_word(0), col_word(1)};            // column words of the tiles whose rows sit in raw[0], raw[1]
        uint32_t cw_ahead = col_word(2);                         // column word of the tile loaded next
        load_row(raw[0], cwv[0]);
        load_row(raw[1], cwv[1]);
        auto tile_step = [&](int k, float4 (&rw)[KC], uint32_t& colw) {
            const int s = k & 1;
            const uint32_t ph = (uint32_t)(k >> 1) & 1u;
            mbar_wait(&bar_rows[s], ph ^ 1u);                    // the MMAs of tile k - 2 have read this stage
            float4* sBs = sB + s * 2 * KC * N;
            if (colw != kTcNoPair) {
                const int cnt = (int)((colw >> 25) & 63u);
                const int used = ALT ? 2 * cnt - 1 + (int)(colw >> 31) : cnt;      // sample positions u the row occupies
                if (used > 8) atomicMax(&sUmax[s], used);
            }
#pragma unroll
            for (int kc = 0; kc < KC; ++kc) {
                float4 w = rw[kc];
                // half-step parity alternates: positions u = 4 kc .. 4 kc + 3 hold samples 2 kc, 2 kc + 1 at parity par
                if (ALT) w = (colw >> 31) ? make_float4(0.f, w.x, 0.f, w.y) : make_float4(w.x, 0.f, w.y, 0.f);
                const float4 h = make_float4(tf32_rn(w.x), tf32_rn(w.y), tf32_rn(w.z), tf32_rn(w.w));
                sBs[kc * N + c] = h;
                sBs[(KC + kc) * N + c] = make_float4(tf32_rn(w.x - h.x), tf32_rn(w.y - h.y), tf32_rn(w.z - h.z), tf32_rn(w.w - h.w));
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            asm volatile("bar.sync 1, %0;" ::"n"(kTcProducers) : "memory");
            if (c == 0) {
                mbar_wait(&bar_empty[s], ph ^ 1u);               // the consumers have read TMEM stage s (tile k - 2)
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const int ksteps = min(K / 8, (sUmax[s] + 7) >> 3);
                sUmax[s] = 1;
                // descriptors differ by the start address only (bits 0-13, in units of 16 bytes; shared memory is < 256 KB,
                // so adding an offset never carries out of the field): one add per operand and product
                const uint64_t da0 = tc_smem_desc(smem_u32(sA), 128 * 16, 128), db0 = tc_smem_desc(smem_u32(sBs), N * 16, 128);
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    uint32_t acc_flag = 0;
                    const uint32_t d = tmem + (uint32_t)((s * MT + mt) * N);
#pragma unroll
                    for (int sp = 0; sp < 3; ++sp) {             // (hi, lo), (lo, hi), then (hi, hi): small terms first
                        const int ha = sp == 1 ? 1 : 0, hb = sp == 0 ? 1 : 0;
#pragma unroll
                        for (int ks = 0; ks < K / 8; ++ks) {
                            if (ks < ksteps) {
                                const uint64_t da = da0 + (uint64_t)((((mt * 2 + ha) * KC + 2 * ks) * 128 * 16) >> 4);
                                const uint64_t db = db0 + (uint64_t)((((hb * KC + 2 * ks) * N * 16)) >> 4);
                                tc_mma_tf32(d, da, db, idesc, acc_flag);
                                acc_flag = 1;
                            }
                        }
                    }
                }
                tc_commit(&bar_full[s]);
                tc_commit(&bar_rows[s]);
            }
            // this buffer takes the rows of tile k + 2 (issued behind the fence, which waits for loads in flight)
            if (k + 2 < ntiles) {
                colw = cw_ahead;
                load_row(rw, colw);
                cw_ahead = col_word(k + 3);
            }
        };
        for (int k = 0; k < ntiles; k += 2) {
            tile_step(k, raw[0], cwv[0]);
            if (k + 1 < ntiles) tile_step(k + 1, raw[1], cwv[1]);
        }
        // the first producer warp frees the tensor memory as soon as the consumers have read the last two tiles (they
        // go on to write their results; the block does not meet again)
        if (warp == kTcConsumers / 32) {
            for (int k = max(ntiles - 2, 0); k < ntiles; ++k) mbar_wait(&bar_empty[k & 1], (uint32_t)(k >> 1) & 1u);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            __syncwarp();
            asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(kTmemCols));
        }
    } else {
        // =================================== multiply-accumulate over input rings ==============================
        TcTile tl = sTiles[0];
        // first tile: its whole window enters
        for (int j0 = tl.jlo; j0 <= tl.jhi; j0 += 4) {
            TcRing rr[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) rr[q] = sRings[min(j0 + q, tl.jhi) - jbase];
#pragma unroll
            for (int q = 0; q < 4; ++q) if (j0 + q <= tl.jhi) fetch_ring(j0 + q, rr[q]);
        }
        cp_async_commit();
        int jhave = tl.jhi;                                      // highest ring whose coefficients sit in (or travel to) the window
        int nold = 0;                                            // rings of the tile's window that were there before this tile
        for (int k = 0; k < ntiles; ++k) {
            const int s = k & 1;
            const uint32_t ph = (uint32_t)(k >> 1) & 1u;
            const TcTile cur = tl;
            const int jlo = cur.jlo, jw = cur.jhi - jlo + 1;
            // records of the next tile and of the rings that enter the window with it: loaded now, used after this tile
            TcRing nx[4];
            if (k + 1 < ntiles) {
                tl = sTiles[k + 1];
#pragma unroll
                for (int q = 0; q < 4; ++q) nx[q] = sRings[min(jhave + 1 + q, tl.jhi) - jbase];
            }
            bool landed = false;
            mbar_wait(&bar_full[s], ph);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");

            float2 acc[TI][2];
#pragma unroll
            for (int ii = 0; ii < TI; ++ii) acc[ii][0] = acc[ii][1] = make_float2(0.f, 0.f);
            const uint32_t tbase = tmem + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)((s * MT + wg) * N);
            uint32_t soff = (uint32_t)(jlo % JW) * 2048u;                // byte offset of the slot of ring jlo + jj
            // cap runs: the periodic extension conjugates on reflection, and a shifted ring changes sign on reflection and on
            // every odd period (reading R8): applied once, in place, when the coefficients of a ring have landed
            auto land = [&]() {
                cp_async_wait<0>();
                landed = true;
                if (CAP) {
                    for (int jj = nold; jj < jw; ++jj) {
                        const TcRing rj = sRings[jlo + jj - jbase];
                        const int Nj = rj.n_sh & 0x7fffffff, w = MULTI ? (int)__umulhi((uint32_t)m, rj.magic) : 0, r = m - w * Nj;
                        const bool refl = 2 * r > Nj;
                        const uint32_t sre = (rj.n_sh < 0 && (refl != ((w & 1) != 0))) ? 0x80000000u : 0u;
                        const uint32_t sim = sre ^ (refl ? 0x80000000u : 0u);
                        if (sre | sim) {
                            const uint32_t a = sv0 + 2048u * (uint32_t)((jlo + jj) % JW);
                            uint32_t x, y, z, ww;
                            asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(x), "=r"(y), "=r"(z), "=r"(ww) : "r"(a));
                            asm volatile("st.shared.v4.b32 [%4], {%0, %1, %2, %3};" ::"r"(x ^ sre), "r"(y ^ sim), "r"(z ^ sre), "r"(ww ^ sim), "r"(a) : "memory");
                        }
                    }
                }
            };
            auto load_v = [&](float4 (&v)[4], int jj0) {
                if (!landed && jj0 + 4 > nold) land();
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v[q].x), "=f"(v[q].y), "=f"(v[q].z), "=f"(v[q].w) : "r"(sv0 + soff));
                    soff += 2048u;
                    if (soff == JW * 2048u) soff = 0u;
                }
            };
            auto mac4 = [&](const uint32_t (&g)[16], const float4 (&v)[4]) {
#pragma unroll
                for (int q = 0; q < 4; ++q) {
#pragma unroll
                    for (int ii = 0; ii < TI; ++ii) {
                        const float G = __uint_as_float(g[q * TI + ii]);
                        acc[ii][0] = ffma2(make_float2(G, G), make_float2(v[q].x, v[q].y), acc[ii][0]);
                        acc[ii][1] = ffma2(make_float2(G, G), make_float2(v[q].z, v[q].w), acc[ii][1]);
                    }
                }
            };
            {
                // groups of four input rings, the accumulator columns and coefficients of the next group in flight
                uint32_t ga[16], gb[16];
                float4 va[4], vb[4];
                tc_ld16(ga, tbase);
                load_v(va, 0);
                for (int jj0 = 0; jj0 < jw; jj0 += 8) {
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    tc_ld16(gb, tbase + (uint32_t)(min(jj0 + 4, JW - 4) * TI));
                    load_v(vb, jj0 + 4);
                    mac4(ga, va);
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    tc_ld16(ga, tbase + (uint32_t)(min(jj0 + 8, JW - 4) * TI));
                    load_v(va, jj0 + 8);
                    if (jj0 + 4 < jw) mac4(gb, vb);
                }
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                if (!landed) land();
            }
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncwarp();
            if ((t & 31) == 0) mbar_arrive(&bar_empty[s]);       // this warp is done with TMEM stage s

            // the rings that enter with the next tile take slots whose rings no later tile reads
            if (k + 1 < ntiles) {
                nold = jhave + 1 - tl.jlo;
#pragma unroll
                for (int q = 0; q < 4; ++q) if (jhave + 1 + q <= tl.jhi) fetch_ring(jhave + 1 + q, nx[q]);
                for (int j = jhave + 5; j <= tl.jhi; ++j) fetch_ring(j, sRings[j - jbase]);
                cp_async_commit();
                jhave = max(jhave, tl.jhi);
            }

            // ---- output: class E stores its mode; cap runs fold onto the ring's own modes ----------------
#pragma unroll
            for (int ii = 0; ii < TI; ++ii) {
                if (ii < cur.nti) {
                    const int i = cur.i0 + ii, iS = R - 1 - i;
                    const int offN = cur.offN[ii], offS = cur.offS[ii];
                    if (!CAP) {
                        if (m_raw < Mh) {                                 // (the Nyquist bin of class-E rings is served elsewhere)
                            out[offN + m] = mk<float>(acc[ii][0].x, acc[ii][0].y);
                            if (iS != i) out[offS + m] = mk<float>(acc[ii][1].x, acc[ii][1].y);
                        }
                    } else if (m_raw <= Mh) {
                        const int Ni = cur.n_sh[ii] & 0x7fffffff;
                        const bool shifted = cur.n_sh[ii] < 0;
                        const float hw = (2 * m == M) ? 0.5f : 1.f;      // the +-M/2 bins carry half the Nyquist term each
                        const int w = MULTI ? m / Ni : 0, r = m - w * Ni;
                        const float s0 = (shifted && (w & 1)) ? -1.f : 1.f, s1 = shifted ? -s0 : s0;
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            if (h == 1 && iS == i) continue;
                            float2* dst = reinterpret_cast<float2*>(out + (h ? offS : offN));
                            const float tx = hw * acc[ii][h].x, ty = hw * acc[ii][h].y;
                            if (2 * r <= Ni) atomicAdd(dst + r, make_float2(s0 * tx, s0 * ty));
                            if (2 * r >= Ni) atomicAdd(dst + (Ni - r), make_float2(s1 * tx, -s1 * ty));
                            if (MULTI && r == 0 && w > 0) atomicAdd(dst, make_float2(s0 * tx, -s0 * ty));     // m = -w N_i folds onto 0 as well
                        }
                    }
                }
            }
        }
    }
}

}  // namespace arkcos
