// Tensor-core band kernel (arkcos_band_tc.cuh): tile geometry, plan-time tables and the host-side launch interface.
// The kernels are compiled in their own translation unit (arkcos_band_tc.cu).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "arkcos_device.cuh"

namespace arkcos {

// Tile geometry.  A block owns MT blocks of 128 modes (TMEM lanes), a tile is TI = 4 output rings whose window of input
// rings has at most JW rings (accumulator column = 4 * input ring + output ring), a row has at most K sample positions.
// Two instantiations: narrow windows (two blocks of modes per thread block) and wide windows / long rows (one).
template <int MT_, int JW_, int K_> struct TcCfgT {
    static constexpr int MT = MT_, JW = JW_, K = K_, TI = 4, N = TI * JW_, KC = K_ / 4;
    static constexpr int consumers = 128 * MT_;        // multiply-accumulate threads: thread = mode
    static constexpr int producers = N;                // B-operand threads: thread = accumulator column; its thread 0 issues the MMAs
    static constexpr int threads = consumers + producers;
    // cosine operand per block of modes, two stages of the row operand, coefficient window per block of modes
    static constexpr size_t smem_bytes = (size_t)(MT_ * 2 * KC * 128 + 2 * 2 * KC * N + MT_ * JW_ * 128) * 16;
    static_assert(N % 32 == 0 && N <= 256 && K_ % 8 == 0 && 2 * MT_ * N <= 512, "tile geometry");
};
using TcCfgNarrow = TcCfgT<2, 32, 24>;     // windows of up to 32 rings, rows of up to 24 positions (Gaussian-like kernels)
using TcCfgWide = TcCfgT<1, 40, 40>;       // windows of up to 40 rings, rows of up to 40 positions (wide hard-cut kernels)
struct TcGeom { int mt, jw, k, n, threads; size_t smem_bytes; };       // the chosen instantiation, for the host
inline TcGeom tc_geom(int cfg)
{
    return cfg == 0 ? TcGeom{TcCfgNarrow::MT, TcCfgNarrow::JW, TcCfgNarrow::K, TcCfgNarrow::N, TcCfgNarrow::threads, TcCfgNarrow::smem_bytes}
                    : TcGeom{TcCfgWide::MT, TcCfgWide::JW, TcCfgWide::K, TcCfgWide::N, TcCfgWide::threads, TcCfgWide::smem_bytes};
}
constexpr int kTcTI = 4;                   // output rings per tile
constexpr int kTcChunkRings = 48;          // longest run of cap rings handed to one block
constexpr int kTcMaxTiles = 16;            // tiles of the longest run (class-E runs: 64 rings); their records live in shared memory
constexpr int kTcMaxWindow = kTcMaxTiles * kTcTI + TcCfgWide::JW;   // input rings the tiles of one run can touch

// Plan-time tables of the tensor-core band kernel (no pointer chasing through the ring-pair table inside the kernel):
// a run of rings, its tiles of up to TI output rings, per tile one word per accumulator column, and two words per ring.
struct TcChunk { int i0, n, M, multi, tile0; };       // run of output rings i0 .. i0 + n - 1 with one grid length M; first tile
struct TcItem { int chunk, bx; };                      // one thread block: run, block of 128 * MT modes
struct __align__(16) TcTile {                          // window of input rings, first output ring, output rings of the tile,
    int jlo, jhi, i0, nti;                             // and per output ring its spectrum offsets (ring, mirror image) and N_i | shifted << 31
    int offN[4], offS[4], n_sh[4];
};
struct TcRing { int offN, offS, n_sh; uint32_t magic; };   // spectrum offsets of ring j and of its mirror image, N_j | shifted << 31, ceil(2^32 / N_j)
// column word: bits 0-24 first sample of the row in W (units of four floats), bits 25-30 samples, bit 31 half-step parity;
// 0xffffffff: no such ring pair (zero row)
constexpr uint32_t kTcNoPair = 0xffffffffu;

// Shared-memory limit and carve-out of the instantiations of geometry cfg (0 narrow, 1 wide); *blocks_per_sm = resident blocks
// per SM.  Returns a cudaError_t.
int tc_setup(int cfg, int* blocks_per_sm);

// KIND as in arkcos_band_tc.cuh (0 class-E alternating parity, 1 class-E integer grid, 2 cap runs single period, 3 several).
void tc_launch(int cfg, int kind, unsigned nitems, unsigned nmaps, cudaStream_t st, const TcItem* items, const TcChunk* chunks,
               const TcTile* tiles, const uint32_t* cols, const TcRing* ringtab, const float* W, int R,
               const cx<float>* specIn, cx<float>* specOut, int64_t spec_stride);

}  // namespace arkcos
