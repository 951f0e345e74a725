/* arkcos.h -- C ABI of libarkcos.so: hybrid Fourier/direct-space convolution of a ring-pixelized map on
 * the sphere with a compact radial kernel (Elsner & Wandelt, "ARKCoS", arXiv:1104.0672), for NVIDIA B200
 * (sm_100a).  Citations are PAPER.md:<line> of the paper text, plus the section / equation.
 *
 * What one call computes (Eq. 1 / Eq. 6, with the quadrature weight of PAPER.md:99):
 *
 *     out(p) = sum_{q : gamma_pq < theta_max}  K(gamma_pq) * in(q) * Omega_q
 *
 * by the hybrid method of section 4 with the anti-ringing treatment of section 4.3
 * (PAPER.md:219): real FFT along every isolatitude ring, kernel rows K(gamma(theta_i, theta_j, dphi)) sampled
 * on a phi grid (Eq. 9) and Fourier-transformed along phi, multiplied with the input-ring spectra
 * and summed over the input rings j inside the support for every azimuthal mode m, super-Nyquist modes folded
 * onto the ring's own modes, inverse real FFT.  On an ECP grid and in the HEALPix equatorial region the result
 * equals the direct sum up to rounding; where a polar-cap ring is involved it carries the interpolation error
 * of the kernel-row grid (controlled by ell_nyquist / polar_oversample below).
 *
 * Every step runs in CUDA kernels of this library on the caller's stream.  There is no CPU fallback and no
 * cuFFT.  All functions return 0 (ARKCOS_OK) or a negative arkcos_status; nothing throws or aborts across the
 * ABI.  Unless noted, pointers are HOST pointers.
 */
#ifndef ARKCOS_H
#define ARKCOS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct arkcos_plan arkcos_plan;          /* opaque; owns all device tables and the workspace */

typedef enum {
    ARKCOS_OK = 0,
    ARKCOS_INVALID_ARG = -1,       /* NULL pointer, size out of range, in == out, nmaps > max_nmaps, ... */
    ARKCOS_UNSUPPORTED = -2,       /* a valid request this build does not implement (see each function) */
    ARKCOS_CUDA_ERROR = -3,        /* a CUDA runtime call failed (no device, launch failure, ...) */
    ARKCOS_OUT_OF_MEMORY = -4      /* host or device allocation failed */
} arkcos_status;

typedef enum { ARKCOS_ECP = 0, ARKCOS_HEALPIX_RING = 1 } arkcos_pix_kind;
typedef enum { ARKCOS_F32 = 0, ARKCOS_F64 = 1 } arkcos_dtype;

/* Pixelization: pixels grouped into isolatitude rings.
 *  ECP           ntheta rings at theta_i = (i + 1/2) pi / ntheta, nphi pixels each at phi_k = 2 pi k / nphi,
 *                Omega_i = sin(theta_i) (pi/ntheta) (2 pi/nphi); pixel index p = i * nphi + k.
 *                nphi must be a power of two, 4 <= nphi <= 16384 (f32) / 8192 (f64).
 *  HEALPIX_RING  ring scheme, resolution nside: rings 1 .. 4 nside - 1 north to south, cap ring
 *                n has 4 n pixels shifted by pi / (4 n), the 2 nside + 1 equatorial rings have 4 nside pixels, every
 *                other one shifted by pi / (4 nside); Omega = 4 pi / (12 nside^2); pixel index = RING ordering.
 *                nside must be a power of two, 1 <= nside <= 4096 (f32) / 2048 (f64). */
typedef struct {
    arkcos_pix_kind kind;
    int ntheta, nphi;              /* ECP only */
    int nside;                     /* HEALPix only */
} arkcos_pixelization;

/* Radial profile (a precomputed table, interpolated linearly).
 *  table[t] = K(theta_t), theta_t = t * theta_max / (n - 1), t = 0 .. n-1 (both end points included); host memory,
 *  copied by arkcos_plan_create (the caller may free it afterwards).  n >= 2.
 *  The support is gamma < theta_max, strict; 0 < theta_max <= pi, radians, a radius. */
typedef struct {
    const double* table;
    int n;
    double theta_max;
} arkcos_kernel;

/* Options; pass NULL for the defaults (all fields zero).
 *  variant           0: anti-ringing scheme of PAPER.md:219 (periodic extension of the ring spectra, folding of the
 *                       super-Nyquist modes, ring offsets inside the kernel evaluation).  1: the basic scheme of
 *                       PAPER.md:125, 142 (ring spectra zero-padded above their Nyquist frequency, output truncated at
 *                       the output ring's Nyquist frequency); served by the general band kernel only (slow path).
 *  ell_nyquist       length of the phi grid on which a kernel row that touches a polar-cap ring is sampled:
 *                       M'_i = max(8, 2 ceil(ell_nyquist * smax_i)), smax_i = max sin(theta) over output ring i and
 *                       its band, i.e. the row resolves wavenumber ell_nyquist along the ring.  0: chosen from the
 *                       profile at plan time (arkcos_plan_ell_nyquist reports it).  Ignored if polar_oversample > 0.
 *  polar_oversample  > 0: M' = polar_oversample * 4 nside for every such row; 1 is the paper's choice.
 *  max_nmaps         largest nmaps arkcos_convolve will be called with (sizes the workspace); 0 means 1.
 *  cache_kernel_rows 0: the kernel rows are re-evaluated from the profile table inside every arkcos_convolve (the
 *                       paper's timing includes the kernel evaluation, Table 1); 1: they are
 *                       evaluated once in arkcos_plan_create.
 *  cache_kernel_spectra 1 (float plans): the cosine transforms G_ij[m] of the kernel rows (and the rows) are computed
 *                       once in arkcos_plan_create and kept in device memory (4 bytes per ring pair and mode: 1.4 GB at
 *                       nside 2048 for a 15' support); arkcos_convolve then only streams them, two maps per read when
 *                       nmaps > 1.  For many maps with one kernel; rows of any length take the fast path.
 *  exact_caps        1 (HEALPix only): every output ring whose band contains a ring shorter than 4 nside (the polar caps
 *                       and the equatorial rings next to them) is recomputed by the direct-space sum of Eq. 6
 *                        after the hybrid pass, so that hard-edged kernels, for which the Fourier
 *                       scheme only suppresses ringing in the caps, are exact everywhere.  Slow path:
 *                       fp64 distances per pixel pair, weights shared by the maps of a call.
 *  no_tensor_cores   0: float plans run the kernel-row phi-transform of the class-E and cap-ring runs as
 *                       3xTF32 tcgen05 matrix products (FP32-level accuracy); 1: every band kernel
 *                       uses FP32 FMAs only (the round-1 kernels; also what small grids and cached-spectra plans use).
 *  no_cuda_graph     0: arkcos_convolve captures the launches of a call (about 30 kernels on the caller's stream and seven plan-owned
 *                       streams, with their event dependencies) into a CUDA graph the first time it sees a combination of
 *                       (d_in, d_out, nmaps, stream) and replays that graph afterwards (the four most recent combinations are
 *                       kept); not on the NULL / legacy default stream, not while the stream is being captured by the caller
 *                       (then the launches simply join the caller's capture), not in the timing modes.  1: always launch directly. */
typedef struct {
    int variant;
    double ell_nyquist;
    int polar_oversample;
    int max_nmaps;
    int cache_kernel_rows;
    int exact_caps;
    int cache_kernel_spectra;
    int no_tensor_cores;
    int no_cuda_graph;
    int reserved[4];               /* must be zero */
} arkcos_options;

/* Builds the ring-geometry table (theta, N, phi0, offset per ring), the band and ring-pair tables, FFT twiddles,
 * and allocates the workspace on the CURRENT CUDA device.  On failure *out is untouched. */
int arkcos_plan_create(arkcos_plan** out, const arkcos_pixelization* pix, const arkcos_kernel* kernel,
                       arkcos_dtype dtype, const arkcos_options* options /* NULL = defaults */);

/* Same tables, host side only: no CUDA call is made, so it works without a device.  The plan answers the queries
 * below (geometry, bands, M'_i, work model); arkcos_convolve on it returns ARKCOS_INVALID_ARG. */
int arkcos_plan_create_tables_only(arkcos_plan** out, const arkcos_pixelization* pix, const arkcos_kernel* kernel,
                                   arkcos_dtype dtype, const arkcos_options* options);

/* d_in, d_out: DEVICE pointers owned by the caller, element type = the plan's dtype, layout [nmaps][npix]
 * contiguous, pixels in ring order.  d_in is not modified; d_in == d_out (or overlapping) is rejected.
 * cuda_stream: a cudaStream_t (NULL = the default stream).  The call only enqueues kernels on that stream: no
 * synchronisation, no allocation, no host arithmetic.  Two calls on the same plan must not run concurrently
 * (they share the plan's workspace). */
int arkcos_convolve(const arkcos_plan* plan, const void* d_in, void* d_out, int nmaps, void* cuda_stream);

/* One map set, several radial kernels (multi-kernel batching: a bank of wavelet scales, or the O(10) radial
 * terms of an asymmetric-beam expansion, "ASYMFAST"): plans[0 .. nkernels-1] are distinct plans created for the
 * same pixelization, dtype and device (kernels, support radii and options may differ).  The forward ring FFTs and the
 * re-origin of Eq. 8 do not depend on the kernel: they run once, with plans[0]'s tables, and every plan's
 * band step reads those spectra; each plan then runs its own kernel rows, band step and inverse FFTs.
 * d_in: [nmaps][npix] as for arkcos_convolve; d_out: [nkernels][nmaps][npix], kernel-major; both DEVICE pointers.
 * Equal to nkernels arkcos_convolve calls, bit for bit.  Only enqueues work on cuda_stream. */
int arkcos_convolve_multi(const arkcos_plan* const* plans, int nkernels, const void* d_in, void* d_out, int nmaps,
                          void* cuda_stream);

/* arkcos_convolve for callers that cannot allocate device memory inside the call (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): the same launches with the same arguments, except that everything
 * the call writes besides d_out -- the input-ring spectra B_j[m], the output-ring spectra (steps 1 and 3 of the hot path,
 * PAPER.md:123-129) and the unfolded spectra between the two pole-ring launches -- lives in one array that is part of the
 * library image (a file-scope __device__ array of ARKCOS_NO_ALLOC_SCRATCH_BYTES; every GPU that loads the library
 * holds it until exit), not in the plan's workspace, and that no CUDA graph is built: the call makes no cudaMalloc,
 * cudaFree, graph instantiation or other allocating call, it only enqueues memsets and kernels on cuda_stream and on the
 * plan's side streams.  The plan's read-only tables are still the ones arkcos_plan_create allocated.
 * Needs  2 * nmaps * spectrum bytes + pole scratch  <= ARKCOS_NO_ALLOC_SCRATCH_BYTES (fp32: about 8.1 bytes per pixel
 * and map, e.g. HEALPix nside 512 with one map, nside 256 with four); more is refused with ARKCOS_INVALID_ARG and a
 * message that names both numbers, and nothing is enqueued.  Arguments, layout and result as for arkcos_convolve.
 * ALL calls on a device share the array, whatever their plan, and it keeps the last call's contents; the part a call
 * uses is cleared at its start.  Two calls that overlap on the GPU (different streams, no dependency) race on it: order
 * them.  The first call on a device looks up the array's address (cudaGetSymbolAddress): make that one outside stream
 * capture. */
#define ARKCOS_NO_ALLOC_SCRATCH_BYTES (32u << 20)
int arkcos_convolve_no_alloc(const arkcos_plan* plan, const void* d_in, void* d_out, int nmaps, void* cuda_stream);

/* Same result from HOST buffers (pinned memory makes the copies asynchronous): host -> device copy, arkcos_convolve,
 * device -> host copy, all on cuda_stream, then a stream synchronisation.  Uses staging buffers inside the plan. */
int arkcos_convolve_host(const arkcos_plan* plan, const void* h_in, void* h_out, int nmaps, void* cuda_stream);

/* Streaming form of the same for a sequence of maps (the paper's use case: one map per detector): the call
 * returns as soon as its three stages are enqueued on plan-owned streams -- host -> device copy, arkcos_convolve,
 * device -> host copy -- with two sets of staging buffers, so that the upload of call k+1 and the download of call k-1
 * overlap the kernels of call k.  h_in must stay valid and unmodified, and h_out unread, until
 * arkcos_plan_synchronize returns (or two further calls have been made and synchronised).  Pinned host memory is needed
 * for the copies to overlap.  Do not mix with arkcos_convolve / arkcos_convolve_host on the same plan without an
 * arkcos_plan_synchronize in between. */
int arkcos_convolve_host_async(const arkcos_plan* plan, const void* h_in, void* h_out, int nmaps);
int arkcos_plan_synchronize(const arkcos_plan* plan);

int arkcos_plan_destroy(arkcos_plan* plan);      /* NULL is a no-op */

/* ---- queries (host side, no CUDA work) ---- */
int64_t arkcos_plan_npix(const arkcos_plan* plan);
int arkcos_plan_nrings(const arkcos_plan* plan);
/* ring = 0 .. nrings-1 north to south; any output pointer may be NULL.  mprime = M'_i of that OUTPUT ring. */
int arkcos_plan_ring_info(const arkcos_plan* plan, int ring, double* theta, int* n, double* phi0, int64_t* offset,
                          int* band_lo, int* band_hi, int* mprime);
double arkcos_plan_ell_nyquist(const arkcos_plan* plan);

/* Work model of one arkcos_convolve with nmaps = 1; any pointer may be NULL.
 *  ring_pairs        ordered ring pairs (i, j) inside the support
 *  row_samples       kernel-row samples evaluated (after the even and north/south symmetries)
 *  mac_flops         flops of the band kernel: cosine transform of the rows + multiply-accumulate over input rings
 *  fft_flops         flops of the forward + inverse ring FFTs as executed (incl. Bluestein padding)
 *  workspace_bytes   device memory held by the plan */
int arkcos_plan_stats(const arkcos_plan* plan, int64_t* ring_pairs, int64_t* row_samples, double* mac_flops,
                      double* fft_flops, int64_t* workspace_bytes);

/* Optional per-stage timing of arkcos_convolve with CUDA events recorded on the caller's stream between the stages.
 * arkcos_plan_get_timing waits for the last call and returns milliseconds for
 *   ms4[0] kernel-row generator, ms4[1] forward ring FFT, ms4[2] band multiply-accumulate, ms4[3] inverse ring FFT. */
int arkcos_plan_set_timing(const arkcos_plan* plan, int enable /* 0 off, 1 stages, 2 stages + band kernels run serially */);
int arkcos_plan_get_timing(const arkcos_plan* plan, float* ms4);

/* The band step is split over several kernels by ring class; normally they run concurrently on
 * plan-owned side streams.  Returns their number (*n = 9), names (of the launches the plan uses: tensor-core, FP32 or cached-spectra kernels), the work model's flops of each (nmaps = 1) and -- only
 * after a call made in timing mode 2, which runs them one after the other -- their last durations in milliseconds.
 * names / model_flops / last_ms: arrays of 9, any may be NULL. */
int arkcos_plan_band_kernels(const arkcos_plan* plan, int* n, const char** names, double* model_flops, float* last_ms);

/* The ring FFTs of one direction are up to nine launches: per transform size Q = 4096, 2048, 1024, 512 the power-of-two rings
 * (one transform per block) and the Bluestein rings, then the shared-memory kernel for very short or very long rings.
 * Returns their number (*n = 9), names, the pixels each serves (algorithmic bytes of a launch = 8 bytes per pixel and map:
 * every map element is read or written once and so is its half spectrum) and -- only after a call made in timing mode 2,
 * which runs them one after the other -- their last durations in milliseconds per direction.  Arrays of 9; any may be NULL. */
int arkcos_plan_fft_kernels(const arkcos_plan* plan, int* n, const char** names, double* pixels, float* last_ms_forward,
                            float* last_ms_inverse);

/* Further terms of the work model of one arkcos_convolve with nmaps = 1; any pointer may be NULL.
 *  band_pair_modes   sum over northern ring pairs of (M/2 + 1): products G_ij[m] B_j[m] per hemisphere
 *  fft_flops_min     flops of the forward + inverse ring FFTs at the rings' own lengths (no Bluestein padding)
 *  tensor_flops      tensor-core flops issued by band_mac_tc_kernel (3 x TF32 terms, zero-padded tiles; upper bound); 0 if unused
 *  memsets_per_map   cudaMemsetAsync calls per map that clear the output-spectrum ranges the cap fold accumulates into */
int arkcos_plan_work_model(const arkcos_plan* plan, double* band_pair_modes, double* fft_flops_min, double* tensor_flops,
                           int* memsets_per_map);

/* Whether the plan's band step runs on the tensor cores (options.no_tensor_cores = 0, a float plan with computed spectra,
 * band windows that fit): *blocks = blocks of band_mac_tc_kernel launched per arkcos_convolve and map (class-E runs, cap
 * runs single period, cap runs several periods), *resident_per_sm = how many of them one SM holds.  Pointers may be NULL.
 * Returns 1 if the tensor-core kernels are used, 0 if not, negative on error. */
int arkcos_plan_tensor_cores(const arkcos_plan* plan, int blocks[3], int* resident_per_sm);

/* Number of kernels one arkcos_convolve enqueues for this plan (kernel-row generator, ring FFT launches per transform
 * size class and direction, band kernels of the ring classes present); -1 for a NULL plan. */
int arkcos_plan_launches_per_convolve(const arkcos_plan* plan);

/* Measures the FP32 FMA throughput of the current device with a register-resident FFMA chain (the denominator of the
 * "alu" roofline); result in TFLOP/s, best of `repeats` launches.  Synchronises the device. */
int arkcos_probe_fp32_peak(double* tflops, int repeats);

/* ---- truncation-error estimate (host side, no CUDA work, no plan) -----------------------------------------------------
 * Eq. 2: K_l = 2 pi int_{-1}^{1} K(z) P_l(z) dz, z = cos(theta), of the tabulated profile (linear
 * interpolation in theta between the nodes, as the convolution uses it) restricted to theta_lo <= theta < theta_hi,
 * 0 <= theta_lo <= theta_hi <= kernel->theta_max; k_ell: caller's array of lmax + 1 doubles (l = 0 .. lmax), lmax <= 65536. */
int arkcos_kernel_legendre(const arkcos_kernel* kernel, double theta_lo, double theta_hi, int lmax, double* k_ell);

/* Eq. 7: mean quadratic error  sigma^2 = sum_{l=0}^{lmax} (2l+1)/(4 pi) dK_l^2 C_l  made by cutting the
 * profile at theta_cut when the map is isotropic with power spectrum c_ell[0 .. lmax]; dK_l is the Legendre transform of
 * "the difference of the exact and the truncated kernel" = the profile on [theta_cut, theta_max).  *signal2 = the same sum
 * with the whole profile's K_l (variance of the exactly smoothed map).  theta_cut >= theta_max gives sigma2 = 0.
 * sigma2 / signal2 may be NULL. */
int arkcos_kernel_truncation_error(const arkcos_kernel* kernel, double theta_cut, const double* c_ell, int lmax,
                                   double* sigma2, double* signal2);

/* Support-radius chooser built on Eq. 7 ("it can be truncated at that radius without introducing significant
 * errors"): among the candidate cuts g * theta_max / ngrid, moving inwards from theta_max, the smallest one up to which
 * sigma(cut) <= rel_tol * sqrt(signal2) holds throughout.  *theta_cut = theta_max when even the outermost cell fails.
 * A plan made from the table's first nodes up to *theta_cut then carries that relative truncation error. */
int arkcos_kernel_choose_cut(const arkcos_kernel* kernel, const double* c_ell, int lmax, double rel_tol, int ngrid,
                             double* theta_cut, double* sigma2, double* signal2);

/* Companion for options.ell_nyquist (the phi grid of kernel rows that touch a polar-cap ring): the smallest wavenumber L
 * such that the smoothed map's power beyond it, sum_{l > L} (2l+1)/(4 pi) K_l^2 C_l, is at most rel_tol^2 of the whole sum. */
int arkcos_kernel_choose_ell_nyquist(const arkcos_kernel* kernel, const double* c_ell, int lmax, double rel_tol,
                                     double* ell_nyquist);

const char* arkcos_strerror(int status);
const char* arkcos_last_error(void);             /* detail of the last failure on this thread ("" if none) */

#ifdef __cplusplus
}
#endif
#endif /* ARKCOS_H */
