// Register-resident ring FFT kernels (arkcos_fft3.cuh): job records, transform geometry and the host-side launch
// interface.  The kernels are compiled in their own translation unit (arkcos_fft3.cu).
#pragma once
#include "arkcos_fft.cuh"

namespace arkcos {

// One job, self-contained (copies of the ring and length records, so a block needs a single table read):
// power-of-two rings: two rings, served by two blocks (has1 = 0: only r0); Bluestein: r0 only.
struct FftJob { RingRec r0, r1; FftLen f; int has1, pad; };

template <int LOGQ> struct Fft3 {
    static constexpr int Q = 1 << LOGQ, T = Q / 16, RL = Q / 256, NC = 16 / RL, SQ = Q + Q / 16;
    static constexpr int MINB = 512 / T;
    static constexpr size_t smem_bytes = 2 * (size_t)SQ * sizeof(cx<float>);
};

// Arguments shared by the launches of one direction.
struct Fft3Args {
    const float* in;            // forward: maps [nmaps][npix]
    float* outmap;              // inverse: maps
    int64_t npix;
    cx<float>* spec;            // forward: written; inverse: read
    int64_t spec_stride;
    const cx<float>*tw, *tw16, *tw3, *filt, *chirp, *phase;
    int logPT;
};

int fft3_setup();               // shared-memory limits of all instantiations; returns a cudaError_t
// power-of-two rings: `njobs` job records of two rings each, one transform per block
void fft3_launch_direct(int logq, bool fwd, const FftJob* jobs, unsigned njobs, unsigned nmaps, cudaStream_t st, const Fft3Args& a);
// power-of-two rings of 8192 complex points: one ring (job.r0) per block, two size-4096 transforms and a radix-2 step
void fft3_launch_direct2(bool fwd, const FftJob* jobs, unsigned njobs, unsigned nmaps, cudaStream_t st, const Fft3Args& a);
// Bluestein rings of 4096 < L <= 8192 complex points: one ring (job.r0) per block, eight size-4096 transforms
void fft3_launch_bluestein2(bool fwd, const FftJob* jobs, unsigned njobs, unsigned nmaps, cudaStream_t st, const Fft3Args& a);
// Bluestein rings: one ring per block; sm_count sizes the look-ahead of the L2 prefetch
void fft3_launch_bluestein(int logq, bool fwd, const FftJob* jobs, unsigned njobs, unsigned nmaps, cudaStream_t st, const Fft3Args& a,
                           int sm_count);

}  // namespace arkcos
