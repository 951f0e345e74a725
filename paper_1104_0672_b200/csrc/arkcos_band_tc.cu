// Translation unit of the tensor-core band kernels (arkcos_band_tc.cuh) and their launch interface (arkcos_band_tc.hpp).
#include "arkcos_band_tc.cuh"

namespace arkcos {

int tc_setup(int* blocks_per_sm)
{
    const void* fn[4] = {(const void*)band_mac_tc_kernel<0>, (const void*)band_mac_tc_kernel<1>, (const void*)band_mac_tc_kernel<2>,
                         (const void*)band_mac_tc_kernel<3>};
    for (const void* f : fn) {
        cudaError_t e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kTcSmemBytes);
        if (e != cudaSuccess) return (int)e;
        // a block needs nearly all of an SM's shared memory
        e = cudaFuncSetAttribute(f, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
        if (e != cudaSuccess) return (int)e;
    }
    return (int)cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, band_mac_tc_kernel<0>, kTcThreads, kTcSmemBytes);
}

void tc_launch(int kind, unsigned nitems, unsigned nmaps, cudaStream_t st, const TcItem* items, const TcChunk* chunks,
               const TcTile* tiles, const uint32_t* cols, const TcRing* ringtab, const float* W, int R,
               const cx<float>* specIn, cx<float>* specOut, int64_t spec_stride)
{
    const dim3 grid(nitems, nmaps);
    switch (kind) {
        case 0: band_mac_tc_kernel<0><<<grid, kTcThreads, kTcSmemBytes, st>>>(items, chunks, tiles, cols, ringtab, W, R, specIn, specOut, spec_stride); break;
        case 1: band_mac_tc_kernel<1><<<grid, kTcThreads, kTcSmemBytes, st>>>(items, chunks, tiles, cols, ringtab, W, R, specIn, specOut, spec_stride); break;
        case 2: band_mac_tc_kernel<2><<<grid, kTcThreads, kTcSmemBytes, st>>>(items, chunks, tiles, cols, ringtab, W, R, specIn, specOut, spec_stride); break;
        default: band_mac_tc_kernel<3><<<grid, kTcThreads, kTcSmemBytes, st>>>(items, chunks, tiles, cols, ringtab, W, R, specIn, specOut, spec_stride); break;
    }
}

}  // namespace arkcos

