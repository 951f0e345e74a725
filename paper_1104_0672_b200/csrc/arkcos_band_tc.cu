// Translation unit of the tensor-core band kernels (arkcos_band_tc.cuh) and their launch interface (arkcos_band_tc.hpp).
#include "arkcos_band_tc.cuh"

namespace arkcos {

namespace {

template <class CFG> int setup(int* blocks_per_sm)
{
    const void* fn[4] = {(const void*)band_mac_tc_kernel<0, CFG>, (const void*)band_mac_tc_kernel<1, CFG>,
                         (const void*)band_mac_tc_kernel<2, CFG>, (const void*)band_mac_tc_kernel<3, CFG>};
    for (const void* f : fn) {
        cudaError_t e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CFG::smem_bytes);
        if (e != cudaSuccess) return (int)e;
        // a block needs nearly all of an SM's shared memory
        e = cudaFuncSetAttribute(f, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
        if (e != cudaSuccess) return (int)e;
    }
    return (int)cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, band_mac_tc_kernel<0, CFG>, CFG::threads, CFG::smem_bytes);
}

template <class CFG>
void launch(int kind, unsigned nitems, unsigned nmaps, cudaStream_t st, const TcItem* items, const TcChunk* chunks, const TcTile* tiles,
            const uint32_t* cols, const TcRing* ringtab, const float* W, int R, const cx<float>* specIn, cx<float>* specOut,
            int64_t spec_stride)
{
    const dim3 grid(nitems, nmaps);
    switch (kind) {
        case 0: band_mac_tc_kernel<0, CFG><<<grid, CFG::threads, CFG::smem_bytes, st>>>(items, chunks, tiles, cols, ringtab, W, R, specIn, specOut, spec_stride); break;
        case 1: band_mac_tc_kernel<1, CFG><<<grid, CFG::threads, CFG::smem_bytes, st>>>(items, chunks, tiles, cols, ringtab, W, R, specIn, specOut, spec_stride); break;
        case 2: band_mac_tc_kernel<2, CFG><<<grid, CFG::threads, CFG::smem_bytes, st>>>(items, chunks, tiles, cols, ringtab, W, R, specIn, specOut, spec_stride); break;
        default: band_mac_tc_kernel<3, CFG><<<grid, CFG::threads, CFG::smem_bytes, st>>>(items, chunks, tiles, cols, ringtab, W, R, specIn, specOut, spec_stride); break;
    }
}

}  // namespace

int tc_setup(int cfg, int* blocks_per_sm) { return cfg == 0 ? setup<TcCfgNarrow>(blocks_per_sm) : setup<TcCfgWide>(blocks_per_sm); }

void tc_launch(int cfg, int kind, unsigned nitems, unsigned nmaps, cudaStream_t st, const TcItem* items, const TcChunk* chunks,
               const TcTile* tiles, const uint32_t* cols, const TcRing* ringtab, const float* W, int R,
               const cx<float>* specIn, cx<float>* specOut, int64_t spec_stride)
{
    if (cfg == 0) launch<TcCfgNarrow>(kind, nitems, nmaps, st, items, chunks, tiles, cols, ringtab, W, R, specIn, specOut, spec_stride);
    else launch<TcCfgWide>(kind, nitems, nmaps, st, items, chunks, tiles, cols, ringtab, W, R, specIn, specOut, spec_stride);
}

}  // namespace arkcos
