// Translation unit of the register-resident ring FFT kernels (arkcos_fft3.cuh) and their launch interface (arkcos_fft3.hpp).
#include "arkcos_fft3.cuh"

namespace arkcos {

namespace {

template <int LOGQ> cudaError_t set_smem()
{
    const int full = (int)Fft3<LOGQ>::smem_bytes;
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(ring_fft3_forward_kernel<LOGQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, full)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ring_fft3_inverse_kernel<LOGQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, full)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ring_fft3_direct1_kernel<LOGQ, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, full / 2)) != cudaSuccess) return e;
    return cudaFuncSetAttribute(ring_fft3_direct1_kernel<LOGQ, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, full / 2);
}

template <int LOGQ, bool FWD>
void launch_direct(const FftJob* jobs, unsigned njobs, unsigned nmaps, cudaStream_t st, const Fft3Args& a)
{
    ring_fft3_direct1_kernel<LOGQ, FWD><<<dim3(2u * njobs, nmaps), Fft3<LOGQ>::T, Fft3<LOGQ>::smem_bytes / 2, st>>>(
        a.in, a.outmap, a.npix, a.spec, a.spec_stride, jobs, a.tw, a.logPT, a.tw16, a.tw3, a.phase);
}

template <int LOGQ, bool FWD>
void launch_bluestein(const FftJob* jobs, unsigned njobs, unsigned nmaps, cudaStream_t st, const Fft3Args& a, int sm_count)
{
    const int ahead = sm_count * Fft3<LOGQ>::MINB;             // resident blocks: the one that will take this block's slot
    const dim3 grid(njobs, nmaps);
    if constexpr (FWD)
        ring_fft3_forward_kernel<LOGQ><<<grid, Fft3<LOGQ>::T, Fft3<LOGQ>::smem_bytes, st>>>(
            a.in, a.npix, a.spec, a.spec_stride, nullptr, jobs, nullptr, a.tw, a.logPT, a.tw16, a.tw3, a.filt, a.chirp, a.phase, ahead);
    else
        ring_fft3_inverse_kernel<LOGQ><<<grid, Fft3<LOGQ>::T, Fft3<LOGQ>::smem_bytes, st>>>(
            a.spec, a.spec_stride, a.outmap, a.npix, nullptr, jobs, nullptr, a.tw, a.logPT, a.tw16, a.tw3, a.filt, a.chirp, a.phase, ahead);
}

}  // namespace

int fft3_setup()
{
    cudaError_t e;
    if ((e = set_smem<9>()) != cudaSuccess) return (int)e;
    if ((e = set_smem<10>()) != cudaSuccess) return (int)e;
    if ((e = set_smem<11>()) != cudaSuccess) return (int)e;
    if ((e = set_smem<12>()) != cudaSuccess) return (int)e;
    const int full = (int)Fft3<12>::smem_bytes;
    if ((e = cudaFuncSetAttribute(ring_fft3_direct2_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, full)) != cudaSuccess) return (int)e;
    if ((e = cudaFuncSetAttribute(ring_fft3_direct2_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, full)) != cudaSuccess) return (int)e;
    if ((e = cudaFuncSetAttribute(ring_fft3_bluestein2_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, full)) != cudaSuccess) return (int)e;
    return (int)cudaFuncSetAttribute(ring_fft3_bluestein2_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, full);
}

void fft3_launch_bluestein2(bool fwd, const FftJob* jobs, unsigned njobs, unsigned nmaps, cudaStream_t st, const Fft3Args& a)
{
    const dim3 grid(njobs, nmaps);
    if (fwd)
        ring_fft3_bluestein2_kernel<true><<<grid, Fft3<12>::T, Fft3<12>::smem_bytes, st>>>(
            a.in, a.outmap, a.npix, a.spec, a.spec_stride, jobs, a.tw, a.logPT, a.tw16, a.tw3, a.filt, a.chirp, a.phase);
    else
        ring_fft3_bluestein2_kernel<false><<<grid, Fft3<12>::T, Fft3<12>::smem_bytes, st>>>(
            a.in, a.outmap, a.npix, a.spec, a.spec_stride, jobs, a.tw, a.logPT, a.tw16, a.tw3, a.filt, a.chirp, a.phase);
}

void fft3_launch_direct2(bool fwd, const FftJob* jobs, unsigned njobs, unsigned nmaps, cudaStream_t st, const Fft3Args& a)
{
    const dim3 grid(njobs, nmaps);
    if (fwd)
        ring_fft3_direct2_kernel<true><<<grid, Fft3<12>::T, Fft3<12>::smem_bytes, st>>>(
            a.in, a.outmap, a.npix, a.spec, a.spec_stride, jobs, a.tw, a.logPT, a.tw16, a.tw3, a.phase);
    else
        ring_fft3_direct2_kernel<false><<<grid, Fft3<12>::T, Fft3<12>::smem_bytes, st>>>(
            a.in, a.outmap, a.npix, a.spec, a.spec_stride, jobs, a.tw, a.logPT, a.tw16, a.tw3, a.phase);
}

#define ARKCOS_FFT3_DISPATCH(fn, ...)                                       \
    switch (logq) {                                                         \
        case 9: fwd ? fn<9, true>(__VA_ARGS__) : fn<9, false>(__VA_ARGS__); break;    \
        case 10: fwd ? fn<10, true>(__VA_ARGS__) : fn<10, false>(__VA_ARGS__); break; \
        case 11: fwd ? fn<11, true>(__VA_ARGS__) : fn<11, false>(__VA_ARGS__); break; \
        default: fwd ? fn<12, true>(__VA_ARGS__) : fn<12, false>(__VA_ARGS__); break; \
    }

void fft3_launch_direct(int logq, bool fwd, const FftJob* jobs, unsigned njobs, unsigned nmaps, cudaStream_t st, const Fft3Args& a)
{
    ARKCOS_FFT3_DISPATCH(launch_direct, jobs, njobs, nmaps, st, a)
}

void fft3_launch_bluestein(int logq, bool fwd, const FftJob* jobs, unsigned njobs, unsigned nmaps, cudaStream_t st, const Fft3Args& a,
                           int sm_count)
{
    ARKCOS_FFT3_DISPATCH(launch_bluestein, jobs, njobs, nmaps, st, a, sm_count)
}

}  // namespace arkcos
