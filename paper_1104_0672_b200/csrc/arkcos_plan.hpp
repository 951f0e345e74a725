// Host-side plan of libarkcos: ring geometry, band / ring-pair tables, FFT length table (step 0 of the hot path,
// PAPER.md:123-125, 162 "we stored the longitudes of all rings ... in constant memory").
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/arkcos.h"
#include "arkcos_band.cuh"
#include "arkcos_fft.cuh"
#include "arkcos_fft3.hpp"
#include "arkcos_direct.cuh"
#include "arkcos_band_cached.cuh"
#include "arkcos_band_tc.hpp"

namespace arkcos {

struct HostGeometry {
    int R = 0;
    int64_t npix = 0, spec_total = 0;
    std::vector<double> theta, phi0, omega;
    std::vector<int> n, shifted, band_lo, band_hi, mprime;
    std::vector<char> direct;        // exact_caps: output ring is recomputed by the direct-space sum (and skipped by the hybrid pass)
    std::vector<int64_t> pix_off, spec_off;
};

struct Stats {
    int64_t ring_pairs = 0, row_samples = 0, workspace_bytes = 0;
    double mac_flops = 0, fft_flops = 0;
    double fft_flops_min = 0;        // ring FFTs of the rings' own lengths (no Bluestein padding), both directions
    double mac_pairs_modes = 0;      // sum over northern ring pairs of (M/2 + 1): products G_ij[m] B_j[m] per hemisphere
    double tc_flops = 0;             // tensor-core flops issued per map by band_mac_tc_kernel (3 x TF32, padded tiles)
    double fft_pixels[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};   // pixels served by each ring-FFT launch, see arkcos_plan_fft_kernels
    double band_flops[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};   // per band kernel, see arkcos_plan_band_kernels
};

}  // namespace arkcos

struct arkcos_plan {
    arkcos_dtype dtype = ARKCOS_F32;
    arkcos_pixelization pix{};
    arkcos_options opt{};
    double theta_max = 0, ell_nyquist = 0;
    int ntab = 0, max_nmaps = 1, device = 0, sm_count = 148;
    bool tables_only = false;
    arkcos::HostGeometry g;
    arkcos::Stats stats;

    int nnorth = 0, npairs = 0, nitems[arkcos::kBandClasses] = {0, 0, 0, 0, 0, 0}, logPT = 0;
    size_t fft_smem = 0;
    int64_t nsamples = 0;

    // device tables
    arkcos::RingRec* d_rings = nullptr;
    arkcos::FftLen* d_lens = nullptr;
    arkcos::PairRec* d_pairs = nullptr;
    arkcos::NorthRec* d_north = nullptr;
    arkcos::EqChunk* d_eqchunks = nullptr;
    int neqchunks = 0, eq_mh = 0, eq_alt = 0;
    uint32_t* d_goff = nullptr;       // cache_kernel_spectra: first float4 of each northern pair's row in d_G
    float* d_G = nullptr;
    arkcos::BandItem* d_direct_items = nullptr;   // exact_caps: {northern ring, first pixel} per block of direct_rings_kernel
    int ndirect = 0;
    arkcos::CapChunk* d_cap_chunks = nullptr;
    arkcos::CapChunkItem* d_cap_chunk_items = nullptr;
    int ncapitems = 0;
    int ncapsingle = 0;               // the first ncapsingle items are single-period runs
    std::vector<std::pair<int64_t, int64_t>> cap_zero;    // output-spectrum ranges cleared before band_mac_capchunk_kernel
    // tensor-core band kernels (arkcos_band_tc.cuh): class-E runs as (run, block of 128 modes) items; the cap runs use
    // d_cap_chunks / d_cap_chunk_items with blocks of 128 modes
    bool use_tc = false;
    int tc_cfg = 0;                   // tile geometry of band_mac_tc_kernel: 0 narrow (TcCfgNarrow), 1 wide (TcCfgWide)
    arkcos::TcChunk* d_tc_chunks = nullptr;
    arkcos::TcTile* d_tc_tiles = nullptr;
    uint32_t* d_tc_cols = nullptr;
    arkcos::TcRing* d_tc_rings = nullptr;
    arkcos::TcItem* d_tc_items[3] = {nullptr, nullptr, nullptr};    // 0 class-E runs, 1 cap runs (single period), 2 cap runs (several)
    int ntc_items[3] = {0, 0, 0};
    int tc_blocks_per_sm = 0;
    int* d_pole = nullptr;
    int* d_nyq = nullptr;             // class-E rings whose Nyquist bin band_nyquist_eq_kernel writes
    int nnyq = 0;
    void* d_pole_scratch = nullptr;   // cx<T>[max_nmaps][npole][2][pole_mh + 1]: unfolded spectra between the two pole launches
    int npole = 0, pole_mh = 0, general_split = 1;
    bool pole_warp_per_mode = false;
    arkcos::BandItem* d_items[arkcos::kBandClasses] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    double* d_table = nullptr;
    int* d_wpair = nullptr;       // ring pair of every group of four stored kernel-row samples
    double* d_table2 = nullptr;   // exact_caps: (K[t], K[t+1] - K[t]) pairs
    void* d_tw = nullptr;        // cx<T>[PT/2]
    void* d_filt = nullptr;      // cx<T>[...] Bluestein filter spectra
    void* d_chirp = nullptr;     // cx<T>[...] Bluestein chirps
    void* d_phase = nullptr;     // cx<T>[...] exp(-i pi k / N) per ring length
    // per direction (0 forward, 1 inverse; the lists differ only for exact_caps plans)
    int* d_fft_order[2] = {nullptr, nullptr};  // rings served by the shared-memory FFT kernels (arkcos_fft.cuh), longest transform first
    int nfft_old[2] = {0, 0};
    // register-resident FFT kernels (arkcos_fft3.cuh): job lists for transform sizes Q = 512, 1024, 2048, 4096
    arkcos::FftJob* d_fft3_jobs[2][4] = {};
    int nfft3[2][4] = {};
    arkcos::FftJob* d_fft3_d2[2] = {};   // power-of-two rings of 8192 complex points (ring_fft3_direct2_kernel)
    int nfft3_d2[2] = {};
    arkcos::FftJob* d_fft3_b2[2] = {};   // Bluestein rings of 4096 < L <= 8192 complex points (ring_fft3_bluestein2_kernel)
    int nfft3_b2[2] = {};
    int nfft3_bluestein[2][4] = {};   // the first jobs of each list are the Bluestein rings, the rest pairs of power-of-two rings
    void* d_tw3 = nullptr;       // cx<float>: pass-3 twiddles of the four transform sizes, see arkcos_fft3.cuh
    int tw3_off[4] = {0, 0, 0, 0};
    void* d_tw16 = nullptr;      // cx<float>[256]: exp(-2 pi i r k / 256) at [16 r + k]
    int fft_bpt = 2;
    void* d_W = nullptr;         // T[nsamples] kernel rows
    void* d_specIn = nullptr;    // cx<T>[max_nmaps][spec_total]
    void* d_specOut = nullptr;
    // arkcos_convolve_multi: the band kernels of this plan read the input-ring spectra another plan made
    mutable void* spec_in_shared = nullptr;
    void* spec_in() const { return spec_in_shared ? spec_in_shared : d_specIn; }
    // lazily allocated staging for arkcos_convolve_host
    mutable void* d_stage_in = nullptr;
    mutable void* d_stage_out = nullptr;
    // arkcos_convolve_host_async: two staging sets, copy / compute streams, events of the last use of each set
    mutable void* d_pipe_in[2] = {nullptr, nullptr};
    mutable void* d_pipe_out[2] = {nullptr, nullptr};
    mutable cudaStream_t s_h2d = nullptr, s_comp = nullptr, s_d2h = nullptr;
    mutable cudaEvent_t ev_h2d[2] = {nullptr, nullptr}, ev_comp[2] = {nullptr, nullptr}, ev_d2h[2] = {nullptr, nullptr};
    mutable uint64_t pipe_calls = 0;
    // CUDA graphs of whole calls, keyed by the call's arguments (most recent first)
    struct GraphEntry { const void* in; void* out; int nmaps; cudaStream_t st; cudaGraphExec_t exec; };
    mutable std::vector<GraphEntry> graphs;
    // optional per-stage timing
    mutable int timing = 0;
    mutable cudaEvent_t ev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    mutable cudaEvent_t ev_band[10] = {};
    mutable cudaEvent_t ev_fft[2][10] = {};      // timing mode 2: before each ring-FFT launch of a direction and after the last
    // fork/join of the band kernels of the different ring classes
    // side streams 0-2: ring-FFT size classes and the big band launches; 0-6: the band kernels of the ring classes
    cudaStream_t side[7] = {}, side_rows = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join[7] = {};
    cudaEvent_t ev_rows_fork = nullptr, ev_rows_done = nullptr;   // kernel-row generator beside the forward FFTs
};
