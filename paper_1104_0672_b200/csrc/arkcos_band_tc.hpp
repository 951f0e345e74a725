// Tensor-core band kernel (arkcos_band_tc.cuh): tile geometry, plan-time tables and the host-side launch interface.
// The kernels are compiled in their own translation unit (arkcos_band_tc.cu).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "arkcos_device.cuh"

namespace arkcos {

constexpr int kTcMT = 2;                   // blocks of 128 modes (TMEM lanes) per thread block, one consumer warpgroup each
constexpr int kTcConsumers = 128 * kTcMT;  // multiply-accumulate threads: thread = mode
constexpr int kTcProducers = 128;          // B-operand threads: thread = accumulator column; its thread 0 issues the MMAs
constexpr int kTcThreads = kTcConsumers + kTcProducers;
constexpr int kTcTI = 4;                   // output rings per tile
constexpr int kTcJW = 32;                  // input rings a tile's window can hold
constexpr int kTcN = kTcTI * kTcJW;        // accumulator columns per block of modes
constexpr int kTcK = 24;                   // sample positions u per row
constexpr int kTcChunkRings = 48;          // longest run of cap rings handed to one block
constexpr int kTcMaxTiles = 16;            // tiles of the longest run (class-E runs: 64 rings); their records live in shared memory
constexpr int kTcMaxWindow = kTcMaxTiles * kTcTI + kTcJW;   // input rings the tiles of one run can touch
// cosine operand per block of modes, two stages of the row operand, coefficient window per block of modes
constexpr size_t kTcSmemBytes = (size_t)(kTcMT * 2 * (kTcK / 4) * 128 + 2 * 2 * (kTcK / 4) * kTcN + kTcMT * kTcJW * 128) * 16;

// Plan-time tables of the tensor-core band kernel (no pointer chasing through the ring-pair table inside the kernel):
// a run of rings, its tiles of up to TI output rings, per tile one word per accumulator column, and two words per ring.
struct TcChunk { int i0, n, M, multi, tile0; };       // run of output rings i0 .. i0 + n - 1 with one grid length M; first tile
struct TcItem { int chunk, bx; };                      // one thread block: run, block of 128 * kTcMT modes
struct __align__(16) TcTile {                          // window of input rings, first output ring, output rings of the tile,
    int jlo, jhi, i0, nti;                             // and per output ring its spectrum offsets (ring, mirror image) and N_i | shifted << 31
    int offN[4], offS[4], n_sh[4];
};
struct TcRing { int offN, offS, n_sh; uint32_t magic; };   // spectrum offsets of ring j and of its mirror image, N_j | shifted << 31, ceil(2^32 / N_j)
// column word: bits 0-24 first sample of the row in W (units of four floats), bits 25-30 samples, bit 31 half-step parity;
// 0xffffffff: no such ring pair (zero row)
constexpr uint32_t kTcNoPair = 0xffffffffu;

// Shared-memory limit and carve-out of the four instantiations; *blocks_per_sm = resident blocks per SM.  Returns a cudaError_t.
int tc_setup(int* blocks_per_sm);

// KIND as in arkcos_band_tc.cuh (0 class-E alternating parity, 1 class-E integer grid, 2 cap runs single period, 3 several).
void tc_launch(int kind, unsigned nitems, unsigned nmaps, cudaStream_t st, const TcItem* items, const TcChunk* chunks,
               const TcTile* tiles, const uint32_t* cols, const TcRing* ringtab, const float* W, int R,
               const cx<float>* specIn, cx<float>* specOut, int64_t spec_stride);

}  // namespace arkcos
