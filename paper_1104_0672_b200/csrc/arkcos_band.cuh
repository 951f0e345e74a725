// Kernel-row generator and banded per-mode multiply-accumulate (steps 3-6 of the hot path).
//
// For output ring i and input ring j inside the support, the kernel row kappa_ij(psi) = K(gamma(theta_i,theta_j,psi))
// (Eq. 9) is even in psi, so its transform along phi is a cosine series over half a row:
//     G_ij[m] = (Omega_j / M) sum_d kappa(psi_d) cos(m psi_d) = sum_t W_ij[t] cos(m (2t + par) pi / M)
// with W the non-zero half-row samples (weight 2 for a sample that has a mirror image, "only on the first
// 2 nside + 1 pixels of a ring").  The output ring's folded spectrum is
//     Dp_i[m'] = sum_j sum_{m = m' + w N_i or w N_i - m', 0 <= m <= M/2} (+-) G_ij[m] Bp_j[m]  (conjugated for the second family)
// ("multiplied ... summation over n_support elements in the theta-direction", PAPER.md:219 duplicate + fold).
// DESIGN.md "Band kernel" derives the signs; the same G serves ring i and its mirror image in the south
// ("only for the northern hemisphere", "northern and southern hemisphere simultaneously").
#pragma once
#include "arkcos_device.cuh"
#include "arkcos_fft.cuh"

namespace arkcos {

struct PairRec {
    double A, B;       // x = A + B sin^2(psi/2): A = 4 sin^2((theta_i - theta_j)/2), B = 4 sin(theta_i) sin(theta_j)
    double scale;      // Omega_j / M
    int64_t woff;      // first sample of the row in W
    int M;             // length of the phi grid of this row (even)
    int par;           // sample positions psi_t = (2t + par) pi / M ; par = 1: half-step offset
    int cnt;           // evaluated samples t = 0 .. cnt-1; the row is stored zero-padded to a multiple of 4 (woff % 4 == 0)
    int j;             // input ring (northern image)
};

struct NorthRec { int pair_lo, pair_hi; };     // pairs of northern output ring i
struct BandItem { int ring, m0; };             // one block of the band kernel: output ring, first folded mode

// Step 3: evaluate the tabulated profile on the half-row of every ring pair.  The distance is
// computed in double precision for both dtypes.  One thread per stored sample (rows are zero-padded to
// multiples of four samples: wpair[g / 4] is the ring pair of the four samples from g on).
template <class T> __global__ void __launch_bounds__(128) kernel_rows_kernel(const PairRec* __restrict__ pairs, const int* __restrict__ wpair,
                                                      int64_t nsamples, const double* __restrict__ table, int ntab,
                                                      double theta_max, T* __restrict__ W)
{
    const int64_t g = (int64_t)blockIdx.x * 128 + (int64_t)threadIdx.x;
    if (g >= nsamples) return;
    const PairRec pr = pairs[wpair[g >> 2]];
    const int t = (int)(g - pr.woff);
    if (t >= pr.cnt) { W[g] = (T)0; return; }
    const double inv2M = 1.0 / (2.0 * (double)pr.M);
    const double tscale = (double)(ntab - 1) / theta_max;
    const int u = 2 * t + pr.par;
    const double sh = sinpi((double)u * inv2M);                        // sin(psi/2), psi = u pi / M
    const double x = pr.A + pr.B * sh * sh;
    const double gamma = gamma_of_chord2(x);
    double val = 0.0;
    if (gamma < theta_max) {
        const double uu = gamma * tscale;
        int tt = (int)floor(uu);
        tt = max(0, min(tt, ntab - 2));
        const double f = uu - (double)tt;
        const double k0 = table[tt], k1 = table[tt + 1];
        const double mult = (u == 0 || u == pr.M) ? 1.0 : 2.0;
        val = (k0 + f * (k1 - k0)) * pr.scale * mult;
    }
    W[g] = (T)val;
}

// Bp_j extended to any mode m >= 0 from the stored half spectrum b[0 .. N/2] (periodic extension).
template <class T> __device__ __forceinline__ cx<T> ext_mode(const cx<T>* __restrict__ b, int m, int N, int shifted)
{
    const int wj = m / N, r = m - wj * N;
    cx<T> v;
    if (2 * r <= N) v = b[r];
    else {
        v = cconj(b[N - r]);
        if (shifted) v = mk<T>(-v.x, -v.y);
    }
    if (shifted && (wj & 1)) v = mk<T>(-v.x, -v.y);
    return v;
}

// Reference band kernel: kGeneralSplit threads per folded output mode m', each taking every kGeneralSplit-th ring pair of
// the band (the sums meet by warp shuffles), cosines by rotation re-seeded every RESEED samples.  grid = (items, nmaps);
// an item is a ring and a first mode, kBandThreads / kGeneralSplit modes per block.  The plan picks kGeneralSplit = 4 when
// the kernel has too few blocks to fill the device (it is latency-bound then), 1 otherwise (coalesced coefficient loads).
constexpr int kBandThreads = 128;
constexpr int kGeneralPack = 6;              // items per block of the four-threads-per-mode form
template <class T, int RESEED, int kGeneralSplit>
__global__ void __launch_bounds__(kBandThreads * kGeneralPack) band_mac_general_kernel(const BandItem* __restrict__ items, int nitems, const NorthRec* __restrict__ north,
                                        const PairRec* __restrict__ pairs, const T* __restrict__ W,
                                        const RingRec* __restrict__ rings, int R, const cx<T>* __restrict__ specIn,
                                        cx<T>* __restrict__ specOut, int64_t spec_stride, int variant_a)
{
    // blockDim.y items per block (whole warps each: the shuffles stay inside an item): few large blocks keep this
    // latency-bound kernel on few SMs instead of a small block on every SM
    const int item = (int)blockIdx.x * (int)blockDim.y + (int)threadIdx.y;
    if (item >= nitems) return;
    const BandItem it = items[item];
    const int i = it.ring, iS = R - 1 - i;
    const RingRec ri = rings[i];
    const int slice = (int)threadIdx.x % kGeneralSplit;
    const int Ni = ri.n, mp_raw = it.m0 + (int)threadIdx.x / kGeneralSplit;
    const bool live = 2 * mp_raw <= Ni;
    const int mp = live ? mp_raw : 0;                           // idle threads follow along (the shuffles need whole warps)
    const cx<T>* __restrict__ in = specIn + (int64_t)blockIdx.y * spec_stride;
    cx<T> accN = mk<T>(0, 0), accS = mk<T>(0, 0);
    int memo_M[2] = {-1, -1}, memo_par[2] = {-1, -1};
    cx<T> memo_rot[2], memo_seed[2];
    memo_rot[0] = memo_rot[1] = memo_seed[0] = memo_seed[1] = mk<T>(0, 0);
    const NorthRec nr = north[i];
    // the records of the next pair travel while this one is worked on (pair record -> ring records -> coefficients is a
    // chain of dependent loads; the kernel is latency-bound)
    int pnx = min(nr.pair_lo + slice, nr.pair_hi - 1);
    PairRec prn = pairs[pnx];
    RingRec rjn = rings[prn.j], rjSn = rings[R - 1 - prn.j];
    for (int p = nr.pair_lo + slice; p < nr.pair_hi; p += kGeneralSplit) {
        const PairRec pr = prn;
        const RingRec rj = rjn, rjS = rjSn;
        pnx = min(p + kGeneralSplit, nr.pair_hi - 1);
        prn = pairs[pnx];
        rjn = rings[prn.j];
        rjSn = rings[R - 1 - prn.j];
        const cx<T>* __restrict__ bN = in + rj.spec_off;
        const cx<T>* __restrict__ bS = in + rjS.spec_off;
        const T* __restrict__ w = W + pr.woff;
        const int M = pr.M, Mh = M >> 1;
#pragma unroll
        for (int fam = 0; fam < 2; ++fam) {
            int wi = fam;
            for (int m = fam ? Ni - mp : mp; m <= Mh; m += Ni, ++wi) {
                // G_ij[m] = sum_t w[t] cos(m (2t + par) pi / M)
                // the step exp(2 pi i m / M) and the first seed exp(i pi m par / M) depend on (m, M, par) only and the pairs of a
                // ring share one or two grids M: kept from the previous pair when they repeat (first term of each family)
                const bool first = wi == fam;
                cx<T> rot;
                if (first && memo_M[fam] == M) rot = memo_rot[fam];
                else {
                    rot = cispi_ratio<T>((uint32_t)((2u * (uint32_t)m) % (2u * (uint32_t)M)), (uint32_t)M);
                    if (first) { memo_M[fam] = M; memo_rot[fam] = rot; memo_par[fam] = -1; }
                }
                T G = 0;
                for (int t0 = 0; t0 < pr.cnt; t0 += RESEED) {
                    // m <= M/2 < 2^15 and 2 t0 + par < 2 M <= 2^17: the product fits 32 bits
                    cx<T> c;
                    if (t0 == 0 && pr.par == 0) c = mk<T>((T)1, (T)0);
                    else if (t0 == 0 && first && memo_par[fam] == 1) c = memo_seed[fam];
                    else {
                        const uint32_t q = ((uint32_t)m * (uint32_t)(2 * t0 + pr.par)) % (2u * (uint32_t)M);
                        c = cispi_ratio<T>((uint32_t)q, (uint32_t)M);
                        if (t0 == 0 && first) { memo_par[fam] = 1; memo_seed[fam] = c; }
                    }
                    const int t1 = min(pr.cnt, t0 + RESEED);
                    for (int t = t0; t < t1; ++t) {
                        G += w[t] * c.x;
                        c = cmul(c, rot);
                    }
                }
                if (2 * m == M) G *= (T)0.5;                         // the +-M/2 bins carry half the Nyquist term each
                if (variant_a) {
                    // basic variant: Bp_j zero-padded above ring j's Nyquist frequency (its own bin
                    // split half/half when the grid extends past it), output truncated at ring i's Nyquist frequency
                    if (2 * m > Ni || 2 * m > rj.n) continue;
                    if (2 * m == rj.n && M > rj.n) G *= (T)0.5;
                }
                if (ri.shifted && (wi & 1)) G = -G;                   // exp(i m phi0_i) = (-1)^w exp(+-i m' phi0_i)
                cx<T> vN = ext_mode(bN, m, rj.n, rj.shifted);
                cx<T> vS = ext_mode(bS, m, rjS.n, rjS.shifted);
                if (fam) { vN.y = -vN.y; vS.y = -vS.y; }
                accN.x += G * vN.x; accN.y += G * vN.y;
                accS.x += G * vS.x; accS.y += G * vS.y;
            }
        }
    }
#pragma unroll
    for (int d = 1; d < kGeneralSplit; d <<= 1) {
        accN.x += __shfl_xor_sync(0xffffffffu, accN.x, d); accN.y += __shfl_xor_sync(0xffffffffu, accN.y, d);
        accS.x += __shfl_xor_sync(0xffffffffu, accS.x, d); accS.y += __shfl_xor_sync(0xffffffffu, accS.y, d);
    }
    if (!live || slice != 0) return;
    cx<T>* __restrict__ out = specOut + (int64_t)blockIdx.y * spec_stride;
    out[ri.spec_off + mp] = accN;
    if (iS != i) out[rings[iS].spec_off + mp] = accS;
}

}  // namespace arkcos

namespace arkcos {

// ---- fast band kernel for "uniform" output rings: every ring pair of the ring is sampled on the same grid length M ----
// One thread per folded output mode m'.  For each unfolded mode m that folds onto m' the thread builds the cosines
// cos(m u pi / M) of the row-sample positions ONCE in registers (rotation, re-seeded every 8 steps from an exact
// sincospi) and reuses them for all input rings of the band; the rows and the per-pair records sit in shared memory.
constexpr int kMaxPairs = 64;
constexpr int kBandClasses = 6;   // 0: general kernel; 1..4: band_mac_uniform_kernel<12,odd>, <12>, <20>, <32,odd>; 5: band_mac_capchunk_kernel (cap rings in the single-period regime)

struct __align__(16) PairMeta {
    int offN, offS;       // first coefficient of input ring j (north image) and of its mirror image (element offsets)
    uint32_t magic;       // ceil(2^32 / Nj): m / Nj = umulhi(m, magic) for m < 2^15
    uint32_t info;        // bits 0-14: Nj - 1 ... see pack_info()
};
// info word: Nj (bits 0-15), ring j shifted (bit 16), par (bit 17), row length / 4 (bits 18-23)
__host__ __device__ inline uint32_t pack_info(int Nj, int shifted, int par, int c4)
{
    return (uint32_t)Nj | ((uint32_t)shifted << 16) | ((uint32_t)par << 17) | ((uint32_t)c4 << 18);
}

template <int TMAX, bool HAS_ODD>
__global__ void __launch_bounds__(kBandThreads)
band_mac_uniform_kernel(const BandItem* __restrict__ items, const NorthRec* __restrict__ north,
                        const PairRec* __restrict__ pairs, const float* __restrict__ W,
                        const RingRec* __restrict__ rings, int R, const cx<float>* __restrict__ specIn,
                        cx<float>* __restrict__ specOut, int64_t spec_stride)
{
    __shared__ __align__(16) float sW[kMaxPairs * TMAX];
    __shared__ PairMeta sP[kMaxPairs];
    __shared__ int sTneed;
    const BandItem it = items[blockIdx.x];
    const int i = it.ring, iS = R - 1 - i;
    const RingRec ri = rings[i];
    const NorthRec nr = north[i];
    const int np = nr.pair_hi - nr.pair_lo;
    if (threadIdx.x == 0) sTneed = 0;
    __syncthreads();
    for (int p = threadIdx.x; p < np; p += kBandThreads) {
        const PairRec pr = pairs[nr.pair_lo + p];
        const RingRec rj = rings[pr.j], rjS = rings[R - 1 - pr.j];
        PairMeta pm;
        pm.offN = (int)rj.spec_off;
        pm.offS = (int)rjS.spec_off;
        pm.magic = (uint32_t)((0x100000000ull + (uint64_t)rj.n - 1ull) / (uint64_t)rj.n);
        pm.info = pack_info(rj.n, rj.shifted, pr.par, (pr.cnt + 3) >> 2);
        sP[p] = pm;
        atomicMax(&sTneed, pr.cnt);
    }
    for (int idx = threadIdx.x; idx < np * (TMAX / 4); idx += kBandThreads) {
        const int p = idx / (TMAX / 4), t4 = idx - p * (TMAX / 4);
        const PairRec& pr = pairs[nr.pair_lo + p];
        if (4 * t4 < pr.cnt) reinterpret_cast<float4*>(sW + p * TMAX)[t4] = reinterpret_cast<const float4*>(W + pr.woff)[t4];
    }
    __syncthreads();
    const int Ni = ri.n, mp = it.m0 + (int)threadIdx.x;
    if (2 * mp > Ni) return;
    const int M = pairs[nr.pair_lo].M, Mh = M >> 1, tneed = sTneed;
    const uint32_t twoM = 2u * (uint32_t)M;
    const cx<float>* __restrict__ in = specIn + (int64_t)blockIdx.y * spec_stride;
    cx<float> accN = mk<float>(0, 0), accS = mk<float>(0, 0);

    for (int fam = 0; fam < 2; ++fam) {
        int wi = fam;
        for (int m = fam ? Ni - mp : mp; m <= Mh; m += Ni, ++wi) {
            float ce[TMAX], co[HAS_ODD ? TMAX : 1];
            {
                const cx<float> rot = cispi_ratio<float>((2u * (uint32_t)m) % twoM, (uint32_t)M);
                cx<float> c = mk<float>(1.f, 0.f), d = mk<float>(1.f, 0.f);
#pragma unroll
                for (int t = 0; t < TMAX; ++t) {
                    if ((t & 7) == 0) {
                        if (t < tneed) {
                            c = cispi_ratio<float>((2u * (uint32_t)m * (uint32_t)t) % twoM, (uint32_t)M);
                            if (HAS_ODD) d = cispi_ratio<float>(((uint32_t)m * (uint32_t)(2 * t + 1)) % twoM, (uint32_t)M);
                        }
                    } else {
                        c = cmul(c, rot);
                        if (HAS_ODD) d = cmul(d, rot);
                    }
                    ce[t] = c.x;
                    if (HAS_ODD) co[t] = d.x;
                }
            }
            // sign bits: half weight at the +-M/2 bins; exp(i m phi0_i) = (-1)^w exp(+-i m' phi0_i); conjugate family
            const float gs = (2 * m == M) ? 0.5f : 1.f;
            const uint32_t sgn_i = (ri.shifted && (wi & 1)) ? 0x80000000u : 0u;
            const uint32_t sgn_fam = fam ? 0x80000000u : 0u;
#pragma unroll 2
            for (int p = 0; p < np; ++p) {
                const PairMeta pm = sP[p];
                const int Nj = (int)(pm.info & 0xffffu), c4 = (int)(pm.info >> 18);
                // periodic extension of the stored half spectra (same index for ring j and its mirror image)
                const int wj = (int)__umulhi((uint32_t)m, pm.magic), r = m - wj * Nj;
                const bool refl = 2 * r > Nj;
                const int idx = refl ? Nj - r : r;
                const cx<float> vN = in[pm.offN + idx], vS = in[pm.offS + idx];
                const float4* __restrict__ w4 = reinterpret_cast<const float4*>(sW + p * TMAX);
                float G = 0.f;
                if (HAS_ODD && (pm.info & (1u << 17))) {
#pragma unroll
                    for (int t4 = 0; t4 < TMAX / 4; ++t4) {
                        if (t4 < c4) {
                            const float4 w = w4[t4];
                            G = fmaf(w.x, co[4 * t4], G); G = fmaf(w.y, co[4 * t4 + 1], G);
                            G = fmaf(w.z, co[4 * t4 + 2], G); G = fmaf(w.w, co[4 * t4 + 3], G);
                        }
                    }
                } else {
#pragma unroll
                    for (int t4 = 0; t4 < TMAX / 4; ++t4) {
                        if (t4 < c4) {
                            const float4 w = w4[t4];
                            G = fmaf(w.x, ce[4 * t4], G); G = fmaf(w.y, ce[4 * t4 + 1], G);
                            G = fmaf(w.z, ce[4 * t4 + 2], G); G = fmaf(w.w, ce[4 * t4 + 3], G);
                        }
                    }
                }
                G *= gs;
                // value used = (+-re, +-im) of the stored coefficient: reflection conjugates, a shifted ring flips the sign
                // on reflection and on every odd period, the second family conjugates again
                const uint32_t shj = (pm.info >> 16) & 1u;
                const uint32_t flip = (shj & ((refl ? 1u : 0u) ^ ((uint32_t)wj & 1u))) << 31;
                const uint32_t sre = sgn_i ^ flip, sim = sre ^ (refl ? 0x80000000u : 0u) ^ sgn_fam;
                const float gr = __uint_as_float(__float_as_uint(G) ^ sre), gi = __uint_as_float(__float_as_uint(G) ^ sim);
                accN.x = fmaf(gr, vN.x, accN.x); accN.y = fmaf(gi, vN.y, accN.y);
                accS.x = fmaf(gr, vS.x, accS.x); accS.y = fmaf(gi, vS.y, accS.y);
            }
        }
    }
    cx<float>* __restrict__ out = specOut + (int64_t)blockIdx.y * spec_stride;
    out[ri.spec_off + mp] = accN;
    if (iS != i) out[rings[iS].spec_off + mp] = accS;
}

// Nyquist bin m' = N_i / 2 of the class-E rings (N_i = N_j = M for the whole band; the run kernels stop at M/2 - 1).
// Both families of the fold meet there at m = M/2 with half the weight each, the second one conjugated (and negated on a
// shifted output ring), and G_ij[M/2] = sum_t w[t] cos((2t + par) pi / 2) = sum_t (-1)^t w[t] on the integer grid, 0 on
// the half-step grid.  So  D_i[M/2] = sum_j G_ij Re B_j[M/2]  (shifted ring: i sum_j G_ij Im B_j[M/2]).
// One warp per output ring, the lanes take the ring pairs; grid = (ceil(nrings / WARPS), nmaps).
template <int WARPS>
__global__ void __launch_bounds__(32 * WARPS)
band_nyquist_eq_kernel(const int* __restrict__ ring_list, int nrings, const NorthRec* __restrict__ north,
                       const PairRec* __restrict__ pairs, const float* __restrict__ W, const RingRec* __restrict__ rings, int R,
                       const cx<float>* __restrict__ specIn, cx<float>* __restrict__ specOut, int64_t spec_stride)
{
    const int k = (int)blockIdx.x * WARPS + ((int)threadIdx.x >> 5), lane = (int)threadIdx.x & 31;
    if (k >= nrings) return;
    const int i = ring_list[k], iS = R - 1 - i;
    const RingRec ri = rings[i];
    const NorthRec nr = north[i];
    const int Mh = ri.n >> 1;
    const cx<float>* __restrict__ in = specIn + (int64_t)blockIdx.y * spec_stride;
    float aN = 0.f, aS = 0.f;
    for (int p = nr.pair_lo + lane; p < nr.pair_hi; p += 32) {
        const PairRec pr = pairs[p];
        if (pr.par) continue;
        const cx<float> vN = in[rings[pr.j].spec_off + Mh], vS = in[rings[R - 1 - pr.j].spec_off + Mh];
        const float4* __restrict__ w4 = reinterpret_cast<const float4*>(W + pr.woff);
        float G = 0.f;
        for (int t4 = 0; 4 * t4 < pr.cnt; ++t4) {                    // rows are stored zero-padded to a multiple of four
            const float4 w = w4[t4];
            G += (w.x - w.y) + (w.z - w.w);
        }
        aN = fmaf(G, ri.shifted ? vN.y : vN.x, aN);
        aS = fmaf(G, ri.shifted ? vS.y : vS.x, aS);
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        aN += __shfl_xor_sync(0xffffffffu, aN, d);
        aS += __shfl_xor_sync(0xffffffffu, aS, d);
    }
    if (lane != 0) return;
    cx<float>* __restrict__ out = specOut + (int64_t)blockIdx.y * spec_stride;
    out[ri.spec_off + Mh] = ri.shifted ? mk<float>(0.f, aN) : mk<float>(aN, 0.f);
    if (iS != i) out[rings[iS].spec_off + Mh] = ri.shifted ? mk<float>(0.f, aS) : mk<float>(aS, 0.f);
}

}  // namespace arkcos

namespace arkcos {

// ---- band kernel for runs of output rings whose pairs all live on one common grid (class E: N_i = N_j = M) -------------
// HEALPix equatorial region and ECP (exact there).  A thread owns MT modes m < M/2 for a whole chunk of
// consecutive output rings: the cosines cos(m u pi / M) are built once per thread (exact sincospi each), every input-ring
// coefficient Bp_j[m] is loaded once per tile of TI output rings and reused from registers, the rows of the tile sit
// in shared memory in a dense [ring of the tile][input ring] layout.  No index arithmetic on the mode axis: m < M/2 = N_j/2
// needs no periodic extension.  (The Nyquist bin m = M/2 of these rings is left to band_mac_uniform_kernel.)
// ALT = 1: the half-step parity of pair (i, j) is (i ^ j) & 1 (HEALPix: every other equatorial ring is shifted,
// PAPER.md:125); ALT = 0: all rows sit on the integer grid (ECP).
struct EqChunk { int i0, n; };
constexpr int kEqJMax = kMaxPairs + 8;

template <int TI, int MT, int TMAX, int ALT, int PAR, int C4>
__device__ __forceinline__ void eq_accumulate(const float* __restrict__ sWj, const float (&ce)[MT][TMAX],
                                              const float (&co)[MT][TMAX], const cx<float> (&v)[2][MT],
                                              cx<float> (&acc)[TI][2][MT])
{
#pragma unroll
    for (int ii = 0; ii < TI; ++ii) {
        const float4* __restrict__ w4 = reinterpret_cast<const float4*>(sWj + ii * (kEqJMax * TMAX));
        const bool odd = ALT && ((PAR ^ ii) & 1) != 0;          // compile-time after unrolling
        float2 sG[MT];                                          // (even-sample sum, odd-sample sum): packed FMAs (FFMA2)
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) sG[mt] = make_float2(0.f, 0.f);
#pragma unroll
        for (int t4 = 0; t4 < C4; ++t4) {
            const float4 w = w4[t4];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                const float* c = odd ? co[mt] : ce[mt];
                sG[mt] = ffma2(make_float2(w.x, w.y), make_float2(c[4 * t4], c[4 * t4 + 1]), sG[mt]);
                sG[mt] = ffma2(make_float2(w.z, w.w), make_float2(c[4 * t4 + 2], c[4 * t4 + 3]), sG[mt]);
            }
        }
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) {
            const float G = sG[mt].x + sG[mt].y;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const float2 a = ffma2(make_float2(G, G), make_float2(v[h][mt].x, v[h][mt].y),
                                       make_float2(acc[ii][h][mt].x, acc[ii][h][mt].y));
                acc[ii][h][mt] = mk<float>(a.x, a.y);
            }
        }
    }
}

// one input ring of the tile: rows of the TI output rings, all taken with the longest row length of this input ring
// (shorter and missing rows are zero-filled)
template <int TI, int MT, int TMAX, int ALT>
__device__ __forceinline__ void eq_input_ring(const float* __restrict__ sWj, int c4, bool par, const float (&ce)[MT][TMAX],
                                              const float (&co)[MT][TMAX], const cx<float> (&v)[2][MT],
                                              cx<float> (&acc)[TI][2][MT])
{
    static_assert(TMAX == 12, "row length classes 1..3");
    if (ALT && par) {
        if (c4 == 3) eq_accumulate<TI, MT, TMAX, ALT, 1, 3>(sWj, ce, co, v, acc);
        else if (c4 == 2) eq_accumulate<TI, MT, TMAX, ALT, 1, 2>(sWj, ce, co, v, acc);
        else eq_accumulate<TI, MT, TMAX, ALT, 1, 1>(sWj, ce, co, v, acc);
    } else {
        if (c4 == 3) eq_accumulate<TI, MT, TMAX, ALT, 0, 3>(sWj, ce, co, v, acc);
        else if (c4 == 2) eq_accumulate<TI, MT, TMAX, ALT, 0, 2>(sWj, ce, co, v, acc);
        else eq_accumulate<TI, MT, TMAX, ALT, 0, 1>(sWj, ce, co, v, acc);
    }
}

template <int TI, int MT, int TMAX, int ALT>
__global__ void __launch_bounds__(kBandThreads)
band_mac_eq_kernel(const EqChunk* __restrict__ chunks, const NorthRec* __restrict__ north,
                   const PairRec* __restrict__ pairs, const float* __restrict__ W, const RingRec* __restrict__ rings,
                   int R, const cx<float>* __restrict__ specIn, cx<float>* __restrict__ specOut, int64_t spec_stride)
{
    __shared__ __align__(16) float sW[TI * kEqJMax * TMAX];       // [ii][jj][t]
    __shared__ int sC[kEqJMax];                                    // [jj]: longest row length / 4 over the tile's rings
    __shared__ int2 sJ[kEqJMax];                                   // spectrum offsets of input ring jlo + jj (N, S)
    static_assert(MT == 2, "a thread owns two adjacent modes: one 16-byte access per ring");
    __shared__ float4 sB[4][2][kBandThreads];                      // in-flight input-ring coefficients, [stage][N/S][thread]
    const EqChunk ch = chunks[blockIdx.y];
    const int M = rings[ch.i0].n, Mh = M >> 1;
    int m[MT];
    float ce[MT][TMAX], co[MT][TMAX];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
        m[mt] = (int)blockIdx.x * (kBandThreads * MT) + MT * (int)threadIdx.x + mt;
        const uint32_t mm = (uint32_t)min(m[mt], Mh - 1), twoM = 2u * (uint32_t)M;
#pragma unroll
        for (int t = 0; t < TMAX; ++t) {
            ce[mt][t] = cispi_ratio<float>((mm * (uint32_t)(2 * t)) % twoM, (uint32_t)M).x;
            co[mt][t] = ALT ? cispi_ratio<float>((mm * (uint32_t)(2 * t + 1)) % twoM, (uint32_t)M).x : 0.f;
        }
    }
    // ring rows start on even coefficient indices (plan), so the thread's mode pair is one aligned 16-byte word
    const cx<float>* __restrict__ in0 = specIn + (int64_t)blockIdx.z * spec_stride + min(m[0], Mh - 2);
    cx<float>* __restrict__ out = specOut + (int64_t)blockIdx.z * spec_stride;

    for (int tile = 0; tile < ch.n; tile += TI) {
        const int nti = min(TI, ch.n - tile), i0 = ch.i0 + tile;
        const int p_first = north[i0].pair_lo, p_last = north[i0 + nti - 1].pair_hi;
        const int jlo = pairs[p_first].j, jw = pairs[p_last - 1].j - jlo + 1;
        __syncthreads();
        for (int k = threadIdx.x; k < jw; k += kBandThreads) sC[k] = 0;
        for (int k = threadIdx.x; k < TI * jw * (TMAX / 4); k += kBandThreads) {
            const int ii = k / (jw * (TMAX / 4)), r = k - ii * (jw * (TMAX / 4));
            reinterpret_cast<float4*>(sW + ii * (kEqJMax * TMAX))[r] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        for (int jj = threadIdx.x; jj < jw; jj += kBandThreads)
            sJ[jj] = make_int2((int)rings[jlo + jj].spec_off, (int)rings[R - 1 - jlo - jj].spec_off);
        __syncthreads();
        for (int k = threadIdx.x; k < (p_last - p_first) * (TMAX / 4); k += kBandThreads) {
            const int p = p_first + k / (TMAX / 4), t4 = k % (TMAX / 4);
            const PairRec& pr = pairs[p];
            int ii = 0;                                                     // ring of the tile this pair belongs to
#pragma unroll
            for (int q = 1; q < TI; ++q) ii += (q < nti && p >= north[i0 + q].pair_lo) ? 1 : 0;
            const int slot = ii * kEqJMax + (pr.j - jlo), c4 = (pr.cnt + 3) >> 2;
            if (t4 < c4)
                reinterpret_cast<float4*>(sW + slot * TMAX)[t4] = reinterpret_cast<const float4*>(W + pr.woff)[t4];
            if (t4 == 0) atomicMax(&sC[pr.j - jlo], c4);
        }
        __syncthreads();
        cx<float> acc[TI][2][MT];
#pragma unroll
        for (int ii = 0; ii < TI; ++ii)
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) acc[ii][h][mt] = mk<float>(0.f, 0.f);

        // Bp_j[m] of the window's input rings: cp.async into a four-deep ring of thread-private shared-memory slots
        // (three input rings in flight while one is accumulated; no barrier, a thread only reads what it copied itself)
        auto fetch = [&](int jj) {
            if (jj < jw) {
                const int2 off = sJ[jj];
                cp_async16(&sB[jj & 3][0][threadIdx.x], in0 + off.x);
                cp_async16(&sB[jj & 3][1][threadIdx.x], in0 + off.y);
            }
            cp_async_commit();
        };
        fetch(0); fetch(1); fetch(2);
        const bool par0 = ALT && ((i0 ^ jlo) & 1);
        for (int jj = 0; jj < jw; ++jj) {
            fetch(jj + 3);
            cp_async_wait<3>();
            cx<float> v[2][MT];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const float4 q = sB[jj & 3][h][threadIdx.x];
                v[h][0] = mk<float>(q.x, q.y);
                v[h][1] = mk<float>(q.z, q.w);
            }
            eq_input_ring<TI, MT, TMAX, ALT>(sW + jj * TMAX, sC[jj], par0 != ((jj & 1) != 0), ce, co, v, acc);
        }
#pragma unroll
        for (int ii = 0; ii < TI; ++ii) {
            if (ii < nti) {
                const int i = i0 + ii, iS = R - 1 - i;
                const int64_t offN = rings[i].spec_off, offS = rings[iS].spec_off;
                if (m[0] < Mh) {
                    *reinterpret_cast<float4*>(out + offN + m[0]) =
                        make_float4(acc[ii][0][0].x, acc[ii][0][0].y, acc[ii][0][1].x, acc[ii][0][1].y);
                    if (iS != i)
                        *reinterpret_cast<float4*>(out + offS + m[0]) =
                            make_float4(acc[ii][1][0].x, acc[ii][1][0].y, acc[ii][1][1].x, acc[ii][1][1].y);
                }
            }
        }
    }
}

}  // namespace arkcos

namespace arkcos {

// ---- band kernel for short rings with long rows (the rings next to the poles) ----------------------------------------------
// There a row covers the whole circle (cnt ~ M/2) and many unfolded modes fold onto each of the few output modes, so the
// work is spread over the UNFOLDED modes: phase 1, one warp per m in [0, M/2]: T(m) = sum_j G_ij[m] Bp_j[m] into a
// scratch array; phase 2 (a second, small launch), one thread per folded mode m': the signed sum of T over
// m = m' + w N_i and w N_i - m'.  Every pair of the ring has the same M.
constexpr int kPoleThreads = 256;
constexpr int kPoleWarps = kPoleThreads / 32;

// Many such rings (a hard-edged kernel with a fine grid: > 100 rings per cap): one block per output ring, a thread per
// unfolded mode walks the samples of a row itself; T through shared memory, both phases in one launch.
template <class T, int RESEED>
__global__ void __launch_bounds__(kPoleThreads)
band_mac_pole1_kernel(const int* __restrict__ ring_list, const NorthRec* __restrict__ north,
                     const PairRec* __restrict__ pairs, const T* __restrict__ W, const RingRec* __restrict__ rings,
                     int R, const cx<T>* __restrict__ specIn, cx<T>* __restrict__ specOut, int64_t spec_stride)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* sT = reinterpret_cast<cx<T>*>(smem_raw);             // [2][Mh + 1]
    const int i = ring_list[blockIdx.x], iS = R - 1 - i;
    const RingRec ri = rings[i];
    const NorthRec nr = north[i];
    const int M = pairs[nr.pair_lo].M, Mh = M >> 1, Ni = ri.n;
    const cx<T>* __restrict__ in = specIn + (int64_t)blockIdx.y * spec_stride;
    for (int m = threadIdx.x; m <= Mh; m += kPoleThreads) {
        const cx<T> rot = cispi_ratio<T>((2u * (uint32_t)m) % (2u * (uint32_t)M), (uint32_t)M);
        cx<T> tN = mk<T>(0, 0), tS = mk<T>(0, 0);
        for (int p = nr.pair_lo; p < nr.pair_hi; ++p) {
            const PairRec pr = pairs[p];
            const T* __restrict__ w = W + pr.woff;
            T G = 0;
            for (int t0 = 0; t0 < pr.cnt; t0 += RESEED) {
                const uint64_t q = ((uint64_t)m * (uint64_t)(2 * t0 + pr.par)) % (uint64_t)(2 * M);
                cx<T> c = cispi_ratio<T>((uint32_t)q, (uint32_t)M);
                const int t1 = min(pr.cnt, t0 + RESEED);
                for (int t = t0; t < t1; ++t) {
                    G += w[t] * c.x;
                    c = cmul(c, rot);
                }
            }
            const RingRec rj = rings[pr.j], rjS = rings[R - 1 - pr.j];
            const cx<T> vN = ext_mode(in + rj.spec_off, m, rj.n, rj.shifted);
            const cx<T> vS = ext_mode(in + rjS.spec_off, m, rjS.n, rjS.shifted);
            tN.x += G * vN.x; tN.y += G * vN.y;
            tS.x += G * vS.x; tS.y += G * vS.y;
        }
        if (2 * m == M) { tN = cscale(tN, (T)0.5); tS = cscale(tS, (T)0.5); }   // +-M/2 bins: half the Nyquist term each
        sT[m] = tN;
        sT[Mh + 1 + m] = tS;
    }
    __syncthreads();
    cx<T>* __restrict__ out = specOut + (int64_t)blockIdx.y * spec_stride;
    for (int mp = threadIdx.x; 2 * mp <= Ni; mp += kPoleThreads) {
        cx<T> aN = mk<T>(0, 0), aS = mk<T>(0, 0);
        for (int fam = 0; fam < 2; ++fam) {
            int wi = fam;
            for (int m = fam ? Ni - mp : mp; m <= Mh; m += Ni, ++wi) {
                const T sg = (ri.shifted && (wi & 1)) ? (T)-1 : (T)1;        // exp(i m phi0_i) = (-1)^w exp(+-i m' phi0_i)
                const cx<T> tN = sT[m], tS = sT[Mh + 1 + m];
                aN.x += sg * tN.x; aN.y += (fam ? -sg : sg) * tN.y;
                aS.x += sg * tS.x; aS.y += (fam ? -sg : sg) * tS.y;
            }
        }
        out[ri.spec_off + mp] = aN;
        if (iS != i) out[rings[iS].spec_off + mp] = aS;
    }
}


// Few such rings (a smooth kernel: ~10 per cap, too few blocks to fill the device): two launches.
// Phase 1.  grid = (rings of the list x blocks_per_ring, nmaps); a warp owns one unfolded mode m, its lanes share the
// samples of a row (stride 32, cosines by rotation with exp(i 64 pi m / M): at most 32 steps) and meet by shuffles.
// T[m] of the ring and of its mirror image go to scratch[((map * nlist + k) * 2 + hemisphere) * tstride + m].
template <class T>
__global__ void __launch_bounds__(kPoleThreads)
band_mac_pole_kernel(const int* __restrict__ ring_list, int blocks_per_ring, const NorthRec* __restrict__ north,
                     const PairRec* __restrict__ pairs, const T* __restrict__ W, const RingRec* __restrict__ rings,
                     int R, const cx<T>* __restrict__ specIn, int64_t spec_stride, cx<T>* __restrict__ scratch, int tstride)
{
    const int k = (int)blockIdx.x / blocks_per_ring, lane = (int)threadIdx.x & 31;
    const int m = ((int)blockIdx.x % blocks_per_ring) * kPoleWarps + ((int)threadIdx.x >> 5);
    const int i = ring_list[k];
    const NorthRec nr = north[i];
    const int M = pairs[nr.pair_lo].M, Mh = M >> 1;
    if (m > Mh) return;
    const cx<T>* __restrict__ in = specIn + (int64_t)blockIdx.y * spec_stride;
    const cx<T> rot = cispi_ratio<T>((64u * (uint32_t)m) % (2u * (uint32_t)M), (uint32_t)M);
    cx<T> tN = mk<T>(0, 0), tS = mk<T>(0, 0);
    // lane l keeps the records of pair pair_lo + l and its two coefficients (all pairs' loads in flight at once: the chain
    // pair record -> ring records -> coefficients is what the warp would otherwise wait for, pair after pair)
    const int npairs = nr.pair_hi - nr.pair_lo;
    PairRec prl = pairs[nr.pair_lo + min(lane, npairs - 1)];
    cx<T> vNl, vSl;
    {
        const RingRec rj = rings[prl.j], rjS = rings[R - 1 - prl.j];
        vNl = ext_mode(in + rj.spec_off, m, rj.n, rj.shifted);
        vSl = ext_mode(in + rjS.spec_off, m, rjS.n, rjS.shifted);
    }
    for (int p = nr.pair_lo; p < nr.pair_hi; ++p) {
        const int src = (p - nr.pair_lo) & 31;
        if (p > nr.pair_lo && src == 0) {                       // more than 32 pairs: the next batch
            prl = pairs[min(p + lane, nr.pair_hi - 1)];
            const RingRec rj = rings[prl.j], rjS = rings[R - 1 - prl.j];
            vNl = ext_mode(in + rj.spec_off, m, rj.n, rj.shifted);
            vSl = ext_mode(in + rjS.spec_off, m, rjS.n, rjS.shifted);
        }
        PairRec pr;
        pr.woff = __shfl_sync(0xffffffffu, prl.woff, src);
        pr.cnt = __shfl_sync(0xffffffffu, prl.cnt, src);
        pr.par = __shfl_sync(0xffffffffu, prl.par, src);
        const cx<T> vN = mk<T>(__shfl_sync(0xffffffffu, vNl.x, src), __shfl_sync(0xffffffffu, vNl.y, src));
        const cx<T> vS = mk<T>(__shfl_sync(0xffffffffu, vSl.x, src), __shfl_sync(0xffffffffu, vSl.y, src));
        const T* __restrict__ w = W + pr.woff;
        // G_ij[m] = sum_t w[t] cos(m (2t + par) pi / M)
        cx<T> c = cispi_ratio<T>(((uint32_t)m * (uint32_t)(2 * lane + pr.par)) % (2u * (uint32_t)M), (uint32_t)M);
        T G = 0;
        for (int t = lane; t < pr.cnt; t += 32) {
            G += w[t] * c.x;
            c = cmul(c, rot);
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) G += __shfl_xor_sync(0xffffffffu, G, d);
        tN.x += G * vN.x; tN.y += G * vN.y;
        tS.x += G * vS.x; tS.y += G * vS.y;
    }
    if (2 * m == M) { tN = cscale(tN, (T)0.5); tS = cscale(tS, (T)0.5); }   // +-M/2 bins: half the Nyquist term each
    if (lane == 0) {
        cx<T>* __restrict__ dst = scratch + ((int64_t)blockIdx.y * (gridDim.x / blocks_per_ring) + k) * 2 * tstride;
        dst[m] = tN;
        dst[tstride + m] = tS;
    }
}

// Phase 2.  grid = (rings of the list, nmaps): one thread per folded mode m', the signed sum of T over m = m' + w N_i and
// w N_i - m' in a fixed order.
template <class T>
__global__ void __launch_bounds__(kPoleThreads)
band_mac_pole_fold_kernel(const int* __restrict__ ring_list, const NorthRec* __restrict__ north, const PairRec* __restrict__ pairs,
                          const RingRec* __restrict__ rings, int R, const cx<T>* __restrict__ scratch, int tstride,
                          cx<T>* __restrict__ specOut, int64_t spec_stride)
{
    const int i = ring_list[blockIdx.x], iS = R - 1 - i;
    const RingRec ri = rings[i];
    const int M = pairs[north[i].pair_lo].M, Mh = M >> 1, Ni = ri.n;
    const cx<T>* __restrict__ sT = scratch + ((int64_t)blockIdx.y * gridDim.x + blockIdx.x) * 2 * tstride;
    cx<T>* __restrict__ out = specOut + (int64_t)blockIdx.y * spec_stride;
    for (int mp = threadIdx.x; 2 * mp <= Ni; mp += kPoleThreads) {
        cx<T> aN = mk<T>(0, 0), aS = mk<T>(0, 0);
        for (int fam = 0; fam < 2; ++fam) {
            int wi = fam;
            for (int m = fam ? Ni - mp : mp; m <= Mh; m += Ni, ++wi) {
                const T sg = (ri.shifted && (wi & 1)) ? (T)-1 : (T)1;        // exp(i m phi0_i) = (-1)^w exp(+-i m' phi0_i)
                const cx<T> tN = sT[m], tS = sT[tstride + m];
                aN.x += sg * tN.x; aN.y += (fam ? -sg : sg) * tN.y;
                aS.x += sg * tS.x; aS.y += (fam ? -sg : sg) * tS.y;
            }
        }
        out[ri.spec_off + mp] = aN;
        if (iS != i) out[rings[iS].spec_off + mp] = aS;
    }
}

}  // namespace arkcos

namespace arkcos {

// ---- cap kernel, chunked: runs of consecutive cap rings that share one grid length M' --------------------------------------
// The plan rounds M'_i up to a multiple of 128 (reading R10), so ~18 consecutive cap rings share M'.  Such a run is
// processed like a run of equatorial rings (band_mac_eq_kernel): a thread owns two adjacent UNFOLDED modes m <= M'/2 for
// the whole chunk, its cosine table is built once, the (periodically extended) coefficient Bp_j[m] of an input ring is
// loaded once per tile of TI output rings and reused from registers, rows are staged per tile with one row length per
// input ring.  What differs from the equatorial case: the extension of Bp_j (reflection above N_j/2: conjugate, sign on
// a shifted ring and on its odd periods) and the fold: T_i[m], m = w N_i + r, belongs to the folded mode r (r <= N_i/2) or
// N_i - r (conjugated; sign on the odd periods of a shifted ring i), so the block adds it into the zero-initialised
// output spectrum with a vector reduction.  With M'/2 < N_i (Gaussian-like kernels: M' ~ 1.7 N_i) every output
// coefficient receives at most two such terms and the sum does not depend on their order; hard-edged kernels (M' up to
// 3 N_i) fold three or four terms, whose order of addition is then not fixed (last-bit differences between runs).
constexpr int kCapChunkRings = 8;          // longest run handed to one block (two tiles): enough blocks to balance the device
struct CapChunk { int i0, n, M, multi; };    // multi = 1: M/2 reaches past a ring length (several periods)
struct CapChunkItem { int chunk, bx; };

template <int TI, int TMAX, bool MULTI>
__global__ void __launch_bounds__(kBandThreads)
band_mac_capchunk_kernel(const CapChunkItem* __restrict__ items, const CapChunk* __restrict__ chunks,
                         const NorthRec* __restrict__ north, const PairRec* __restrict__ pairs,
                         const float* __restrict__ W, const RingRec* __restrict__ rings, int R,
                         const cx<float>* __restrict__ specIn, cx<float>* __restrict__ specOut, int64_t spec_stride)
{
    constexpr int MT = 2, G4 = TMAX / 4;
    __shared__ __align__(16) float sW[TI * kEqJMax * TMAX];       // [ii][jj][t]
    __shared__ int sC[kEqJMax];                                    // [jj]: longest row length / 4 over the tile's rings
    __shared__ int4 sJ[kEqJMax];                                   // input ring jlo + jj: spectrum offsets (N, S), N_j, shifted
    const CapChunkItem it = items[blockIdx.x];
    const CapChunk ch = chunks[it.chunk];
    const int M = ch.M, Mh = M >> 1;
    const int m0 = it.bx * (kBandThreads * MT) + MT * (int)threadIdx.x;      // modes m0, m0 + 1
    float ce[MT][TMAX];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
        const uint32_t mm = (uint32_t)min(m0 + mt, Mh), twoM = 2u * (uint32_t)M;
        const cx<float> rot = cispi_ratio<float>((2u * mm) % twoM, (uint32_t)M);
        cx<float> a = mk<float>(1.f, 0.f);
#pragma unroll
        for (int t = 0; t < TMAX; ++t) {
            if ((t & 7) == 0) { if (t > 0) a = cispi_ratio<float>((2u * mm * (uint32_t)t) % twoM, (uint32_t)M); }
            else a = cmul(a, rot);
            ce[mt][t] = a.x;
        }
    }
    const cx<float>* __restrict__ in = specIn + (int64_t)blockIdx.y * spec_stride;
    cx<float>* __restrict__ out = specOut + (int64_t)blockIdx.y * spec_stride;
    const int mA = min(m0, Mh), mB = min(m0 + 1, Mh);

    // extended coefficient of input ring (Nj, shj) at mode m from the stored half spectrum (single period: m < Nj)
    // periodic extension of the stored half spectrum of a ring (N_j, shifted flag in bit 31, magic = ceil(2^32 / N_j)):
    // m = w N_j + r; above N_j/2 the coefficient is the conjugate of the one at N_j - r; a shifted ring changes sign on
    // reflection and on every odd period (reading R8)
    // (MULTI = false: the plan guarantees M'/2 < N_j and M'/2 < N_i for every ring involved, period 0 only)
    auto ext_index = [](int m, int nj_sh, uint32_t magic) {
        const int Nj = nj_sh & 0x7fffffff, w = MULTI ? (int)__umulhi((uint32_t)m, magic) : 0, r = m - w * Nj;
        return 2 * r > Nj ? Nj - r : r;
    };
    auto ext_value = [](cx<float> b, int m, int nj_sh, uint32_t magic) {
        const int Nj = nj_sh & 0x7fffffff, w = MULTI ? (int)__umulhi((uint32_t)m, magic) : 0, r = m - w * Nj;
        const bool refl = 2 * r > Nj;
        if (refl) b.y = -b.y;
        if (nj_sh < 0 && (refl != ((w & 1) != 0))) { b.x = -b.x; b.y = -b.y; }
        return b;
    };

    for (int tile = 0; tile < ch.n; tile += TI) {
        const int nti = min(TI, ch.n - tile), i0 = ch.i0 + tile;
        const int p_first = north[i0].pair_lo, p_last = north[i0 + nti - 1].pair_hi;
        const int jlo = pairs[p_first].j, jw = pairs[p_last - 1].j - jlo + 1;
        __syncthreads();
        for (int k = threadIdx.x; k < jw; k += kBandThreads) sC[k] = 0;
        for (int k = threadIdx.x; k < TI * jw * G4; k += kBandThreads) {
            const int ii = k / (jw * G4), r = k - ii * (jw * G4);
            reinterpret_cast<float4*>(sW + ii * (kEqJMax * TMAX))[r] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        for (int jj = threadIdx.x; jj < jw; jj += kBandThreads) {
            const RingRec rj = rings[jlo + jj];
            sJ[jj] = make_int4((int)rj.spec_off, (int)rings[R - 1 - jlo - jj].spec_off, rj.n | (rj.shifted ? (int)0x80000000 : 0),
                               MULTI ? (int)(uint32_t)((0x100000000ull + (uint64_t)rj.n - 1ull) / (uint64_t)rj.n) : 0);
        }
        __syncthreads();
        for (int k = threadIdx.x; k < (p_last - p_first) * G4; k += kBandThreads) {
            const int p = p_first + k / G4, t4 = k % G4;
            const PairRec& pr = pairs[p];
            int ii = 0;                                                     // ring of the tile this pair belongs to
#pragma unroll
            for (int q = 1; q < TI; ++q) ii += (q < nti && p >= north[i0 + q].pair_lo) ? 1 : 0;
            const int slot = ii * kEqJMax + (pr.j - jlo), c4 = (pr.cnt + 3) >> 2;
            if (t4 < c4)
                reinterpret_cast<float4*>(sW + slot * TMAX)[t4] = reinterpret_cast<const float4*>(W + pr.woff)[t4];
            if (t4 == 0) atomicMax(&sC[pr.j - jlo], c4);
        }
        __syncthreads();
        cx<float> acc[TI][2][MT];
#pragma unroll
        for (int ii = 0; ii < TI; ++ii)
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) acc[ii][h][mt] = mk<float>(0.f, 0.f);

        cx<float> nx[2][MT];                                                // coefficients of the next input ring (raw)
        auto fetch = [&](int jj) {
            const int4 rj = sJ[min(jj, jw - 1)];
            const int ia = ext_index(mA, rj.z, (uint32_t)rj.w), ib = ext_index(mB, rj.z, (uint32_t)rj.w);
            nx[0][0] = in[rj.x + ia]; nx[0][1] = in[rj.x + ib];
            nx[1][0] = in[rj.y + ia]; nx[1][1] = in[rj.y + ib];
        };
        fetch(0);
        for (int jj = 0; jj < jw; ++jj) {
            const int4 rj = sJ[jj];
            cx<float> v[2][MT];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                v[h][0] = ext_value(nx[h][0], mA, rj.z, (uint32_t)rj.w);
                v[h][1] = ext_value(nx[h][1], mB, rj.z, (uint32_t)rj.w);
            }
            fetch(jj + 1);
            const float* sWj = sW + jj * TMAX;
            const int c4 = sC[jj];
            if (c4 >= 5) eq_accumulate<TI, MT, TMAX, 0, 0, (G4 >= 5 ? 5 : 1)>(sWj, ce, ce, v, acc);
            else if (c4 == 4) eq_accumulate<TI, MT, TMAX, 0, 0, (G4 >= 4 ? 4 : 1)>(sWj, ce, ce, v, acc);
            else if (c4 == 3) eq_accumulate<TI, MT, TMAX, 0, 0, 3>(sWj, ce, ce, v, acc);
            else if (c4 == 2) eq_accumulate<TI, MT, TMAX, 0, 0, 2>(sWj, ce, ce, v, acc);
            else eq_accumulate<TI, MT, TMAX, 0, 0, 1>(sWj, ce, ce, v, acc);
        }
        // fold: mode m adds to m (m <= N_i/2) and / or to N_i - m (conjugated; sign if ring i is shifted)
#pragma unroll
        for (int ii = 0; ii < TI; ++ii) {
            if (ii < nti) {
                const int i = i0 + ii, iS = R - 1 - i;
                const RingRec ri = rings[i];
                const int64_t offS = rings[iS].spec_off;
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    const int m = m0 + mt;
                    if (m > Mh) continue;
                    const float hw = (2 * m == M) ? 0.5f : 1.f;          // the +-M/2 bins carry half the Nyquist term each
                    // m = w N_i + r: folded mode r in period w (r <= N_i/2) and / or N_i - r in period w + 1 (conjugated);
                    // a shifted ring changes sign on every odd period
                    const int w = MULTI ? m / ri.n : 0, r = m - w * ri.n;
                    const float s0 = (ri.shifted && (w & 1)) ? -1.f : 1.f, s1 = ri.shifted ? -s0 : s0;
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        if (h == 1 && iS == i) continue;
                        float2* dst = reinterpret_cast<float2*>(out + (h ? offS : ri.spec_off));
                        const float tx = hw * acc[ii][h][mt].x, ty = hw * acc[ii][h][mt].y;
                        if (2 * r <= ri.n) atomicAdd(dst + r, make_float2(s0 * tx, s0 * ty));
                        if (2 * r >= ri.n) atomicAdd(dst + (ri.n - r), make_float2(s1 * tx, -s1 * ty));
                        if (MULTI && r == 0 && w > 0) atomicAdd(dst, make_float2(s0 * tx, -s0 * ty));     // m = -w N_i folds onto 0 as well
                    }
                }
            }
        }
    }
}

}  // namespace arkcos
