// libarkcos: plan construction (host) and the C ABI of include/arkcos.h.
#include <math.h>
#include <stdio.h>
#include <string.h>
#include <stdlib.h>

#include <algorithm>
#include <map>
#include <mutex>
#include <new>
#include <type_traits>

#include "arkcos_plan.hpp"

using namespace arkcos;

namespace {

thread_local std::string g_last_error;

int fail(int code, const std::string& msg)
{
    g_last_error = msg;
    return code;
}

}  // namespace

namespace arkcos {
int set_last_error(int code, const std::string& msg) { return fail(code, msg); }      // for the other translation units
}

namespace {

#define CUDA_TRY(expr)                                                                                        \
    do {                                                                                                      \
        cudaError_t e_ = (expr);                                                                              \
        if (e_ != cudaSuccess) {                                                                              \
            cudaGetLastError();                                                                               \
            return fail(e_ == cudaErrorMemoryAllocation ? ARKCOS_OUT_OF_MEMORY : ARKCOS_CUDA_ERROR,           \
                        std::string(#expr) + ": " + cudaGetErrorString(e_));                                  \
        }                                                                                                     \
    } while (0)

bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }
int ilog2(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }
const double kPi = 3.14159265358979323846264338327950288;

// ---- step 0: ring geometry (HEALPix ring centres: Gorski et al. 2005, cited PAPER.md:125) ----
int build_geometry(const arkcos_pixelization& pix, HostGeometry& g)
{
    if (pix.kind == ARKCOS_ECP) {
        const int R = pix.ntheta, N = pix.nphi;
        g.R = R;
        for (int i = 0; i < R; ++i) {
            const double th = (i + 0.5) * kPi / R;
            g.theta.push_back(th);
            g.n.push_back(N);
            g.phi0.push_back(0.0);
            g.shifted.push_back(0);
            g.omega.push_back(sin(th) * (kPi / R) * (2.0 * kPi / N));
        }
    } else {
        const int ns = pix.nside, R = 4 * ns - 1;
        g.R = R;
        const double om = 4.0 * kPi / (12.0 * (double)ns * (double)ns);
        for (int idx = 0; idx < R; ++idx) {
            const int i = idx + 1;
            double th;
            int n, sh;
            if (i < ns) {                    // north cap: z = 1 - i^2/(3 ns^2), theta = 2 asin(sqrt((1-z)/2))
                th = 2.0 * asin(i / (sqrt(6.0) * ns));
                n = 4 * i;
                sh = 1;
            } else if (i <= 3 * ns) {        // equatorial belt: z = 4/3 - 2i/(3 ns)
                th = acos(4.0 / 3.0 - 2.0 * i / (3.0 * ns));
                n = 4 * ns;
                sh = ((i - ns) % 2 == 0) ? 1 : 0;
            } else {                         // south cap: mirror image
                const int ii = 4 * ns - i;
                th = kPi - 2.0 * asin(ii / (sqrt(6.0) * ns));
                n = 4 * ii;
                sh = 1;
            }
            g.theta.push_back(th);
            g.n.push_back(n);
            g.shifted.push_back(sh);
            g.phi0.push_back(sh ? kPi / n : 0.0);
            g.omega.push_back(om);
        }
    }
    g.pix_off.assign(g.R + 1, 0);
    g.spec_off.assign(g.R + 1, 0);
    for (int i = 0; i < g.R; ++i) {
        g.pix_off[i + 1] = g.pix_off[i] + g.n[i];
        g.spec_off[i + 1] = g.spec_off[i] + ((g.n[i] / 2 + 2) & ~1);     // N/2 + 1 coefficients, rows start 16-byte aligned
    }
    g.npix = g.pix_off[g.R];
    g.spec_total = g.spec_off[g.R];
    return 0;
}

// band of ring i: rings j with |theta_i - theta_j| < theta_max (contiguous, theta is monotonic)
void build_bands(HostGeometry& g, double theta_max)
{
    g.band_lo.resize(g.R);
    g.band_hi.resize(g.R);
    int lo = 0, hi = 0;
    for (int i = 0; i < g.R; ++i) {
        while (!(fabs(g.theta[i] - g.theta[lo]) < theta_max)) ++lo;
        if (hi < i) hi = i;
        while (hi + 1 < g.R && fabs(g.theta[i] - g.theta[hi + 1]) < theta_max) ++hi;
        g.band_lo[i] = lo;
        g.band_hi[i] = hi;
    }
}

// Automatic ell_nyquist (reading R10): smallest wavenumber beyond which the 1-D spectra of straight cuts
// through the profile hold less than `tol` of their L1 mass, capped at ell_cap.  Cuts at offsets 0 and theta_max/2.
double auto_ell_nyquist(const double* table, int ntab, double theta_max, double ell_cap)
{
    const int NL = 1024;
    const int NS = (int)std::min(65536.0, std::max(2048.0, ceil(2.0 * ell_cap * theta_max)));
    const double tol = 1e-7;
    double best = 0.0;
    std::vector<double> f(NS + 1), spec(NL + 1);
    for (int cut = 0; cut < 2; ++cut) {
        const double off = cut * 0.5 * theta_max;
        const double amax = sqrt(theta_max * theta_max - off * off);
        for (int s = 0; s <= NS; ++s) {
            const double a = amax * s / NS, gam = sqrt(a * a + off * off);
            double u = gam * (ntab - 1) / theta_max;
            int t = std::min(std::max((int)floor(u), 0), ntab - 2);
            f[s] = gam < theta_max ? table[t] + (u - t) * (table[t + 1] - table[t]) : 0.0;
        }
        double total = 0.0;
        for (int l = 0; l <= NL; ++l) {
            const double ell = ell_cap * l / NL;
            double acc = 0.0;
            for (int s = 0; s <= NS; ++s) acc += ((s == 0 || s == NS) ? 0.5 : 1.0) * f[s] * cos(ell * amax * s / NS);
            spec[l] = fabs(acc);
            total += spec[l];
        }
        if (!(total > 0.0)) continue;
        double tail = 0.0;
        int l = NL;
        for (; l > 0; --l) {
            tail += spec[l];
            if (tail > tol * total) break;
        }
        best = std::max(best, ell_cap * std::min(l + 1, NL) / NL);
    }
    return best > 0.0 ? best : ell_cap;
}

constexpr int kPoleMaxModes = 1024;   // longest unfolded spectrum (M/2 + 1) the pole kernel keeps in shared memory

struct HostTables {
    std::vector<RingRec> rings;
    std::vector<FftLen> lens;
    std::vector<int> bluestein_ids;     // lens that need a filter spectrum
    std::vector<PairRec> pairs;
    std::vector<NorthRec> north;
    std::vector<BandItem> items[kBandClasses];
    std::vector<CapChunkItem> cap_chunk_items_multi;   // items of runs that need more than one period of the ring spectra
    int cap_nsingle = 0;
    std::vector<CapChunk> cap_chunks;            // runs of cap rings with one grid length for band_mac_capchunk_kernel
    std::vector<CapChunkItem> cap_chunk_items;
    std::vector<std::pair<int64_t, int64_t>> cap_zero;   // (first coefficient, count) ranges of the output spectrum to clear
    std::vector<int> pole_rings;                 // rings for band_mac_pole_kernel
    std::vector<int> nyq_rings;                  // class-E rings: their Nyquist bin goes to band_nyquist_eq_kernel
    int pole_mh = 0;
    int general_split = 1;                       // threads per mode of band_mac_general_kernel
    bool pole_warp_per_mode = false;             // long rows: band_mac_pole_kernel + fold; short rows: band_mac_pole1_kernel
    std::vector<EqChunk> eq_chunks;              // runs of consecutive class-E rings for band_mac_eq_kernel   // per band-kernel class (see band_class)
    int eq_alt = 0;
    bool use_tc = false;                         // tensor-core band kernels (arkcos_band_tc.cuh) serve the class-E and cap runs
    int tc_cfg = 0;                              // their tile geometry: 0 narrow windows, 1 wide windows / long rows
    std::vector<TcChunk> tc_chunks;              // runs of rings served by band_mac_tc_kernel, their tiles and column words
    std::vector<TcTile> tc_tiles;
    std::vector<uint32_t> tc_cols;
    std::vector<TcItem> tc_items[3];             // thread blocks: 0 class-E runs, 1 cap runs (single period), 2 cap runs (several)
    std::vector<TcRing> tc_rings;                // per ring: spectrum offsets (ring, mirror image), length | shifted, magic divisor
    // per direction (0 forward, 1 inverse): exact_caps plans transform only the rings the hybrid pass needs
    std::vector<int> fft_order[2];       // rings of the shared-memory FFT kernels, sorted by decreasing transform size
    std::vector<FftJob> fft3_jobs[2][4]; // jobs of the register-resident FFT kernels, Q = 512 << k
    std::vector<FftJob> fft3_d2[2];      // power-of-two rings of 8192 complex points (ring_fft3_direct2_kernel), one ring per job
    std::vector<FftJob> fft3_b2[2];      // Bluestein rings of 4096 < L <= 8192 complex points (ring_fft3_bluestein2_kernel), mirror rings adjacent
    int64_t filt_total = 0, chirp_total = 0, ph_total = 0, nsamples = 0;
    int logPT = 1;
};

// FFT length table: one entry per distinct ring length
// need[d][i]: ring i is transformed in direction d (0 forward, 1 inverse)
void build_fft_lens(const HostGeometry& g, HostTables& t, Stats& st, bool use_fft3, const std::vector<char> (&need)[2])
{
    std::map<int, int> id_of;
    t.rings.resize(g.R);
    for (int i = 0; i < g.R; ++i) {
        const int N = g.n[i], L = N / 2;
        auto it = id_of.find(N);
        if (it == id_of.end()) {
            FftLen f{};
            f.L = L;
            f.pow2 = is_pow2(L) ? 1 : 0;
            f.logP = f.pow2 ? ilog2(L) : ilog2(2 * L - 1);
            f.filt_off = 0;
            f.chirp_off = 0;
            f.ph_off = t.ph_total;
            t.ph_total += L + 1;
            if (!f.pow2) {
                f.filt_off = t.filt_total;
                t.filt_total += (int64_t)1 << f.logP;
                f.chirp_off = t.chirp_total;
                t.chirp_total += L;
                t.bluestein_ids.push_back((int)t.lens.size());
            }
            t.logPT = std::max(t.logPT, f.logP);
            it = id_of.emplace(N, (int)t.lens.size()).first;
            t.lens.push_back(f);
        }
        RingRec r{};
        r.pix_off = g.pix_off[i];
        r.spec_off = g.spec_off[i];
        r.n = N;
        r.shifted = g.shifted[i];
        r.len_id = it->second;
        t.rings[i] = r;
        const FftLen& f = t.lens[r.len_id];
        const double P = (double)(1 << f.logP);
        // forward + inverse: complex FFT(s) + O(N) split / chirps
        const double ndir = (need[0][i] ? 1.0 : 0.0) + (need[1][i] ? 1.0 : 0.0);
        st.fft_flops += ndir * (f.pow2 ? 5.0 * P * f.logP + 20.0 * L : 2.0 * 5.0 * P * f.logP + 6.0 * P + 32.0 * L);
        st.fft_flops_min += ndir * (5.0 * L * log2((double)std::max(L, 2)) + 20.0 * L);
    }
    // Rings whose transform size Q (L for a power of two, half the Bluestein convolution length otherwise) is 512 .. 4096
    // go to the register-resident kernels: Bluestein rings first, a ring next to its mirror image (same tables), then
    // the power-of-two rings two per block.  Everything else stays with the shared-memory kernels.
    auto cls_of = [&](int i) {
        const FftLen& f = t.lens[t.rings[i].len_id];
        const int logq = f.pow2 ? f.logP : f.logP - 1;
        return (use_fft3 && logq >= 9 && logq <= 12) ? logq - 9 : -1;
    };
    for (int d = 0; d < 2; ++d) {
        std::vector<int> direct[4];
        std::vector<char> taken(g.R, 0);
        for (int i = g.R / 2; i >= 0; --i) {                 // longest rings first
            const int twin[2] = {i, g.R - 1 - i};
            for (int h = 0; h < 2; ++h) {
                const int r = twin[h];
                const int c = cls_of(r);
                if (c < 0 || taken[r]) continue;
                taken[r] = 1;
                if (!need[d][r]) continue;
                if (t.lens[t.rings[r].len_id].pow2) direct[c].push_back(r);
                else {
                    FftJob j{};
                    j.r0 = t.rings[r];
                    j.f = t.lens[t.rings[r].len_id];
                    t.fft3_jobs[d][c].push_back(j);
                }
            }
        }
        for (int c = 0; c < 4; ++c)
            for (size_t k = 0; k < direct[c].size(); k += 2)
            {
                FftJob j{};
                j.r0 = t.rings[direct[c][k]];
                j.f = t.lens[j.r0.len_id];
                j.has1 = k + 1 < direct[c].size() ? 1 : 0;
                if (j.has1) j.r1 = t.rings[direct[c][k + 1]];
                t.fft3_jobs[d][c].push_back(j);
            }
        for (int i = 0; i < g.R; ++i) {                       // twice the largest register-resident size, power of two
            const FftLen& f = t.lens[t.rings[i].len_id];
            if (taken[i] || !use_fft3 || !f.pow2 || f.L != 8192) continue;
            taken[i] = 1;
            if (!need[d][i]) continue;
            FftJob j{};
            j.r0 = t.rings[i];
            j.f = f;
            t.fft3_d2[d].push_back(j);
        }
        for (int i = g.R / 2; i >= 0; --i) {                 // Bluestein rings with a convolution of 16384 points, longest first
            const int twin[2] = {i, g.R - 1 - i};
            for (int h = 0; h < 2; ++h) {
                const int r = twin[h];
                const FftLen& f = t.lens[t.rings[r].len_id];
                if (taken[r] || !use_fft3 || f.pow2 || f.logP != 14) continue;
                taken[r] = 1;
                if (!need[d][r]) continue;
                FftJob j{};
                j.r0 = t.rings[r];
                j.f = f;
                t.fft3_b2[d].push_back(j);
            }
        }
        for (int i = 0; i < g.R; ++i)
            if (!taken[i] && need[d][i]) t.fft_order[d].push_back(i);
        std::stable_sort(t.fft_order[d].begin(), t.fft_order[d].end(), [&](int a, int b) {
            const FftLen &fa = t.lens[t.rings[a].len_id], &fb = t.lens[t.rings[b].len_id];
            const int wa = (fa.pow2 ? 1 : 2) << fa.logP, wb = (fb.pow2 ? 1 : 2) << fb.logP;
            return wa > wb;
        });
    }
    // launch order of one direction: Q = 4096 power-of-two, Bluestein, then 2048, 1024, 512 alike, then the shared-memory
    // kernel (pixel counts of the forward direction; the inverse differs only for exact_caps plans)
    for (int c = 0; c < 4; ++c)
        for (const FftJob& j : t.fft3_jobs[0][c]) {
            const int slot = 2 * (3 - c) + (j.f.pow2 ? 0 : 1);
            st.fft_pixels[slot] += j.r0.n + (j.has1 ? j.r1.n : 0);
        }
    for (int i : t.fft_order[0]) st.fft_pixels[8] += g.n[i];
    for (const FftJob& j : t.fft3_d2[0]) st.fft_pixels[8] += j.r0.n;      // launched beside the shared-memory kernel
    for (const FftJob& j : t.fft3_b2[0]) st.fft_pixels[8] += j.r0.n;
}

// Ring-pair table for the northern output rings (the southern ones reuse the rows of their mirror images).
void build_pairs(HostGeometry& g, double theta_max, double ell_nyq, int fixed_mprime, int band_threads, bool allow_fast, bool allow_pole, bool cached,
                 bool allow_tc, int sm_count, HostTables& t, Stats& st)
{
    const int R = g.R, nnorth = (R + 1) / 2;
    // tensor-core band kernels: float plans with computed spectra; the window of a tile of kTcTI consecutive output rings
    // must fit the kernel's slots for every tile the plan could form: the narrow geometry if it does, else the wide one
    bool use_tc = allow_tc && allow_fast && !cached;
    int tc_cfg = 0;
    if (use_tc) {
        int wmax = 0;
        for (int i = 0; i < nnorth; ++i) wmax = std::max(wmax, g.band_hi[std::min(i + kTcTI - 1, nnorth - 1)] - g.band_lo[i] + 1);
        tc_cfg = wmax <= tc_geom(0).jw ? 0 : 1;
        use_tc = wmax <= tc_geom(tc_cfg).jw;
    }
    const TcGeom tg = tc_geom(tc_cfg);
    t.tc_cfg = tc_cfg;
    t.use_tc = use_tc;
    std::vector<int> eq_rings, general_rings;
    bool any_odd = false;
    const double shm = sin(0.5 * theta_max), xmax = 4.0 * shm * shm;
    g.mprime.assign(R, 0);
    const int nmax = *std::max_element(g.n.begin(), g.n.end());
    for (int i = 0; i < R; ++i) {
        double smax = 0.0;
        for (int j = g.band_lo[i]; j <= g.band_hi[i]; ++j) smax = std::max(smax, sin(g.theta[j]));
        g.mprime[i] = fixed_mprime > 0 ? fixed_mprime : std::max(8, 2 * (int)ceil(ell_nyq * smax));
        // grids of 512 points and more are rounded up to a multiple of 128 so that runs of consecutive cap rings share one
        // grid length (reading R10; band_mac_capchunk_kernel)
        // (multiples of 256 from 2048 on when the tensor-core kernel serves the runs: twice as many rings per block)
        const int step = use_tc && g.mprime[i] >= 2048 ? 256 : 128;
        if (fixed_mprime <= 0 && g.mprime[i] >= 512) g.mprime[i] = (g.mprime[i] + step - 1) / step * step;
    }
    for (int i = 0; i < R; ++i) any_odd = any_odd || (g.n[i] == nmax && g.shifted[i] != g.shifted[std::min(i + 1, R - 1)] && g.n[std::min(i + 1, R - 1)] == nmax);
    const int eq_alt = any_odd ? 1 : 0;
    int ncap_long = 0, ncap_multi = 0;                     // cap rings of 512+ pixels, and those whose grid spans several periods
    for (int i = 0; i < nnorth; ++i)
        if (g.n[i] >= 512 && g.n[i] < nmax) { ++ncap_long; ncap_multi += g.mprime[i] / 2 >= g.n[i] ? 1 : 0; }
    const bool multi_is_rule = 4 * ncap_multi > ncap_long;
    t.eq_alt = eq_alt;
    t.north.resize(nnorth);
    for (int i = 0; i < nnorth; ++i) {
        t.north[i].pair_lo = (int)t.pairs.size();
        double ring_flops = 0.0;
        const bool has_mirror = (R - 1 - i) != i;
        for (int j = g.band_lo[i]; j <= g.band_hi[i]; ++j) {
            PairRec p{};
            const double sd = sin(0.5 * (g.theta[i] - g.theta[j]));
            p.A = 4.0 * sd * sd;
            p.B = 4.0 * sin(g.theta[i]) * sin(g.theta[j]);
            if (g.n[i] == nmax && g.n[j] == nmax) {   // class E: common grid, ring offset inside the kernel evaluation
                p.M = g.n[i];
                p.par = g.shifted[i] != g.shifted[j] ? 1 : 0;
            } else {                         // class C: a cap ring is involved, Eq. 8 on both rings
                p.M = g.mprime[i];
                p.par = 0;
            }
            p.scale = g.omega[j] / (double)p.M;
            int umax = p.M;
            if (p.B > 0.0) {
                const double ratio = (xmax - p.A) / p.B;
                if (ratio < 1.0) {
                    const double psimax = 2.0 * asin(sqrt(std::max(ratio, 0.0)));
                    umax = std::min((double)p.M, floor(psimax * p.M / kPi) + 2.0);
                }
            }
            p.cnt = umax >= p.par ? (umax - p.par) / 2 + 1 : 0;
            p.j = j;
            p.woff = t.nsamples;
            t.nsamples += (p.cnt + 3) & ~3;          // rows are stored zero-padded to a multiple of four samples
            t.pairs.push_back(p);
            st.ring_pairs += has_mirror ? 2 : 1;
            if (g.direct[i]) continue;               // (the direct-space sum uses the pair record, the hybrid pass skips the ring)
            const double modes = p.M / 2 + 1;
            ring_flops += modes * (2.0 * p.cnt + (has_mirror ? 8.0 : 4.0));
            st.mac_flops += modes * (2.0 * p.cnt + (has_mirror ? 8.0 : 4.0));
            st.mac_pairs_modes += modes;
        }
        t.north[i].pair_hi = (int)t.pairs.size();
        if (g.direct[i]) continue;
        // which band kernel serves this ring: the fast ones need one grid length M for the whole ring, short rows
        // and few pairs (rows and pair records live in shared memory)
        int cls = 0;
        if (allow_fast) {
            const int lo = t.north[i].pair_lo, hi = t.north[i].pair_hi;
            bool same = hi - lo <= kMaxPairs, odd = false;
            int maxcnt = 0;
            for (int p = lo; p < hi; ++p) {
                same = same && t.pairs[p].M == t.pairs[lo].M;
                odd = odd || t.pairs[p].par;
                maxcnt = std::max(maxcnt, t.pairs[p].cnt);
            }
            bool all_e = same, alt_ok = true;
            for (int p = lo; p < hi && all_e; ++p) {
                all_e = t.pairs[p].M == g.n[i] && g.n[t.pairs[p].j] == g.n[i];
                alt_ok = alt_ok && t.pairs[p].par == (eq_alt ? ((i ^ t.pairs[p].j) & 1) : 0);
            }
            // rows of the tensor-core kernel hold K sample positions: K/2 samples with half-step positions, K without
            const bool tc_eq = use_tc && (g.n[i] / 2) % 128 == 0;
            if (all_e && alt_ok && hi > lo && (maxcnt <= (tc_eq ? (eq_alt ? tg.k / 2 : tg.k) : 12) || cached) && g.n[i] >= 8 && g.spec_total < (int64_t)INT32_MAX) {
                eq_rings.push_back(i);
                st.band_flops[2] += ring_flops;
                // the Nyquist bin m = M/2 goes to a kernel of its own (a warp per ring, rows of any length)
                t.nyq_rings.push_back(i);
                continue;
            }
            if (same && hi > lo) {
                if (maxcnt <= 12) cls = odd ? 1 : 2;
                else if (maxcnt <= 20 && !odd) cls = 3;
                else if (maxcnt <= 32) cls = 4;
                // runs of band_mac_capchunk_kernel: one grid length, integer grid, rings long enough for 256-mode blocks
                if (use_tc) {
                    // tensor-core run kernel: integer grid, rows of at most K samples, any number of periods
                    if (!odd && maxcnt <= tg.k && g.n[i] >= 256 && g.n[i] < nmax && t.pairs[lo].M / 2 < (1 << 15)) cls = 5;
                } else if ((cls == 2 || cls == 3 || (cached && !odd))) {
                    bool single_period = t.pairs[lo].M / 2 < g.n[i] && g.n[i] <= t.pairs[lo].M;
                    for (int p = lo; p < hi; ++p) single_period = single_period && t.pairs[lo].M / 2 < g.n[t.pairs[p].j];
                    // multi-period rings join the run kernel when they are the rule (hard-edged kernels: M' up to 3 N_i) or when
                    // the spectra are cached; a few stragglers of a Gaussian plan stay with the uniform kernels
                    if (g.n[i] >= 512 && t.pairs[lo].M / 2 < (1 << 15) && (single_period || cached || multi_is_rule)) cls = 5;
                }
            }
        }
        if (cls == 0 && allow_pole && t.north[i].pair_hi > t.north[i].pair_lo) {
            bool same = true;
            const int M0 = t.pairs[t.north[i].pair_lo].M;
            for (int p = t.north[i].pair_lo; p < t.north[i].pair_hi; ++p) same = same && t.pairs[p].M == M0;
            if (same && M0 / 2 + 1 <= kPoleMaxModes) {
                t.pole_rings.push_back(i);
                st.band_flops[1] += ring_flops;
                t.pole_mh = std::max(t.pole_mh, M0 / 2);
                continue;
            }
        }
        // band-kernel slots: 0 general, 1 pole, 2 eq, 3 uniform<12>, 4 uniform<20>, 5 uniform<32,odd>, 6 uniform<12,odd>
        static const int slot_of_cls[kBandClasses] = {0, 6, 3, 4, 5, 7};
        if (cls != 5) st.band_flops[slot_of_cls[cls]] += ring_flops;
        if (cls == 5) {
            const int M = t.pairs[t.north[i].pair_lo].M;
            // single-period ring: M/2 below the length of ring i and of every ring of its band (a run is homogeneous)
            bool single = M / 2 < g.n[i] && g.n[i] <= M;
            for (int p = t.north[i].pair_lo; p < t.north[i].pair_hi; ++p) single = single && M / 2 < g.n[t.pairs[p].j];
            const int multi = single ? 0 : 1;
            st.band_flops[7 + multi] += ring_flops;          // slot 7: runs of a single period, 8: of several
            if (!t.cap_chunks.empty() && t.cap_chunks.back().i0 + t.cap_chunks.back().n == i && t.cap_chunks.back().M == M &&
                t.cap_chunks.back().multi == multi && t.cap_chunks.back().n < (use_tc ? kTcChunkRings : kCapChunkRings))
                ++t.cap_chunks.back().n;
            else
                t.cap_chunks.push_back(CapChunk{i, 1, M, multi});
            continue;
        }
        if (cls == 0) { general_rings.push_back(i); continue; }      // items once the split is known
        for (int m0 = 0; m0 <= g.n[i] / 2; m0 += band_threads) t.items[cls].push_back(BandItem{i, m0});
    }
    // general kernel: four threads per mode when it would have too few blocks to fill the device
    {
        int64_t blocks1 = 0;
        for (int i : general_rings) blocks1 += (g.n[i] / 2 + band_threads) / band_threads;
        t.general_split = blocks1 < 8 * (int64_t)sm_count ? 4 : 1;
        for (int i : general_rings)
            for (int m0 = 0; m0 <= g.n[i] / 2; m0 += band_threads / t.general_split) t.items[0].push_back(BandItem{i, m0});
        // pole kernel: one block per ring leaves the device idle when the rings are few; then a warp per mode, two launches
        t.pole_warp_per_mode = !t.pole_rings.empty() && 4 * (int)t.pole_rings.size() <= sm_count;
    }
    // chunks of consecutive class-E rings: about one block per resident slot of the device (4 blocks per SM)
    {
        const int mh = eq_rings.empty() ? 0 : g.n[eq_rings[0]] / 2;
        const int gx = std::max(1, (mh + kBandThreads * 2 - 1) / (kBandThreads * 2));
        const int target = std::max(1, (4 * sm_count) / gx);
        int chn = std::max(8, ((int)eq_rings.size() + target - 1) / target);
        if (use_tc) chn = std::min(chn, kTcMaxTiles * kTcTI);       // the tile records of a run live in shared memory
        for (size_t k = 0; k < eq_rings.size(); ++k) {
            const int i = eq_rings[k];
            if (!t.eq_chunks.empty() && t.eq_chunks.back().i0 + t.eq_chunks.back().n == i && t.eq_chunks.back().n < chn &&
                g.n[t.eq_chunks.back().i0] == g.n[i])
                ++t.eq_chunks.back().n;
            else
                t.eq_chunks.push_back(EqChunk{i, 1});
        }
    }
    if (use_tc) {
        // tables of band_mac_tc_kernel: per run its tiles of kTcTI output rings (window of input rings) and, per tile, one
        // word per accumulator column = 4 * (input ring - window start) + output ring of the tile
        auto add_run = [&](int i0, int n, int M, int multi, int cls, bool with_nyquist) {
            TcChunk c{i0, n, M, multi, (int)t.tc_tiles.size()};
            for (int tile = 0; tile < n; tile += kTcTI) {
                const int nti = std::min(kTcTI, n - tile), ia = i0 + tile;
                const int jlo = t.pairs[t.north[ia].pair_lo].j, jhi = t.pairs[t.north[ia + nti - 1].pair_hi - 1].j;
                TcTile tile_rec{jlo, jhi, ia, nti, {0, 0, 0, 0}, {0, 0, 0, 0}, {0, 0, 0, 0}};
                for (int ii = 0; ii < nti; ++ii) {
                    tile_rec.offN[ii] = (int)g.spec_off[ia + ii];
                    tile_rec.offS[ii] = (int)g.spec_off[R - 1 - ia - ii];
                    tile_rec.n_sh[ii] = g.n[ia + ii] | (g.shifted[ia + ii] ? (int)0x80000000 : 0);
                }
                t.tc_tiles.push_back(tile_rec);
                for (int col = 0; col < tg.n; ++col) {
                    const int jj = col / kTcTI, ii = col % kTcTI;
                    uint32_t word = kTcNoPair;
                    if (ii < nti) {
                        const NorthRec& nr = t.north[ia + ii];
                        const int pj = jlo + jj - t.pairs[nr.pair_lo].j;
                        if (pj >= 0 && pj < nr.pair_hi - nr.pair_lo) {
                            const PairRec& pr = t.pairs[nr.pair_lo + pj];
                            word = (uint32_t)(pr.woff / 4) | ((uint32_t)pr.cnt << 25) | ((uint32_t)pr.par << 31);
                        }
                    }
                    t.tc_cols.push_back(word);
                }
            }
            t.tc_chunks.push_back(c);
            const int nmodes = with_nyquist ? M / 2 + 1 : M / 2;
            for (int bx = 0; bx * 128 * tg.mt < nmodes; ++bx) {
                t.tc_items[cls].push_back(TcItem{(int)t.tc_chunks.size() - 1, bx});
                // upper bound: the kernel issues fewer K steps for tiles whose rows are short
                st.tc_flops += (double)((n + kTcTI - 1) / kTcTI) * tg.mt * 3.0 * (tg.k / 8) * 2.0 * 128.0 * tg.n * 8.0;
            }
        };
        for (int j = 0; j < R; ++j)
            t.tc_rings.push_back(TcRing{(int)g.spec_off[j], (int)g.spec_off[R - 1 - j], g.n[j] | (g.shifted[j] ? (int)0x80000000 : 0),
                                        (uint32_t)((0x100000000ull + (uint64_t)g.n[j] - 1ull) / (uint64_t)g.n[j])});
        for (const EqChunk& e : t.eq_chunks)
            if ((g.n[e.i0] / 2) % 128 == 0) add_run(e.i0, e.n, g.n[e.i0], 0, 0, false);
        // cap runs from the pole towards the equator: the longest (last) first
        for (size_t c = t.cap_chunks.size(); c-- > 0;)
            add_run(t.cap_chunks[c].i0, t.cap_chunks[c].n, t.cap_chunks[c].M, t.cap_chunks[c].multi, t.cap_chunks[c].multi ? 2 : 1, true);
    }
    for (size_t c = 0; c < t.cap_chunks.size(); ++c) {
        const CapChunk& ch = t.cap_chunks[c];
        const int modes_per_block = use_tc ? 128 : kBandThreads * 2;
        for (int bx = 0; bx * modes_per_block <= ch.M / 2; ++bx)
            (ch.multi ? t.cap_chunk_items_multi : t.cap_chunk_items).push_back(CapChunkItem{(int)c, bx});
        // output coefficients of the chunk's rings (north and mirror image) are accumulated: they start from zero
        const int iA = ch.i0, iB = ch.i0 + ch.n - 1;
        auto add_range = [&](int ra, int rb) {
            const int64_t a = g.spec_off[ra], n = g.spec_off[rb + 1] - a;
            if (!t.cap_zero.empty() && t.cap_zero.back().first + t.cap_zero.back().second == a) t.cap_zero.back().second += n;
            else t.cap_zero.push_back({a, n});
        };
        add_range(iA, iB);
        // mirror images of the run's rings, without the rings of the run itself (a run may end on the self-mirror middle ring)
        const int lo = std::max(R - 1 - iB, iB + 1);
        if (lo <= R - 1 - iA) add_range(lo, R - 1 - iA);
    }
    // longest blocks first (the chunks run from the pole towards the equator, M' grows)
    std::reverse(t.cap_chunk_items.begin(), t.cap_chunk_items.end());
    std::reverse(t.cap_chunk_items_multi.begin(), t.cap_chunk_items_multi.end());
    t.cap_nsingle = (int)t.cap_chunk_items.size();                               // single-period items first, then the others
    t.cap_chunk_items.insert(t.cap_chunk_items.end(), t.cap_chunk_items_multi.begin(), t.cap_chunk_items_multi.end());
    std::sort(t.cap_zero.begin(), t.cap_zero.end());
    for (size_t k = 1; k < t.cap_zero.size();) {                             // merge adjacent ranges
        if (t.cap_zero[k - 1].first + t.cap_zero[k - 1].second == t.cap_zero[k].first) {
            t.cap_zero[k - 1].second += t.cap_zero[k].second;
            t.cap_zero.erase(t.cap_zero.begin() + k);
        } else ++k;
    }
    st.row_samples = 0;
    for (const PairRec& p : t.pairs) st.row_samples += p.cnt;
}

template <class V> int upload(V** dst, const std::vector<V>& src, int64_t* bytes)
{
    const size_t nb = std::max<size_t>(src.size(), 1) * sizeof(V);
    CUDA_TRY(cudaMalloc((void**)dst, nb));
    if (!src.empty()) CUDA_TRY(cudaMemcpy(*dst, src.data(), src.size() * sizeof(V), cudaMemcpyHostToDevice));
    *bytes += (int64_t)nb;
    return 0;
}

// twiddles exp(-2 pi i k / PT) from double precision, Bluestein filters by a plan-time kernel, workspace
template <class T, int BPT> int set_fft_smem(size_t bytes)
{
    CUDA_TRY(cudaFuncSetAttribute(ring_fft_forward_kernel<T, BPT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    CUDA_TRY(cudaFuncSetAttribute(ring_fft_inverse_kernel<T, BPT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    CUDA_TRY(cudaFuncSetAttribute(bluestein_filter_kernel<T, BPT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return 0;
}

// job lists and the 16 x 16 twiddle table of the register-resident FFT kernels (float plans only)
template <class T> int setup_fft3(arkcos_plan* pl, const HostTables& t)
{
    if constexpr (sizeof(T) == 4) {
    for (int d = 0; d < 2; ++d)
        for (int c = 0; c < 4; ++c) {
            pl->nfft3[d][c] = (int)t.fft3_jobs[d][c].size();
            if (int rc = upload(&pl->d_fft3_jobs[d][c], t.fft3_jobs[d][c], &pl->stats.workspace_bytes)) return rc;
        }
    for (int d = 0; d < 2; ++d) {
        pl->nfft3_d2[d] = (int)t.fft3_d2[d].size();
        if (int rc = upload(&pl->d_fft3_d2[d], t.fft3_d2[d], &pl->stats.workspace_bytes)) return rc;
        pl->nfft3_b2[d] = (int)t.fft3_b2[d].size();
        if (int rc = upload(&pl->d_fft3_b2[d], t.fft3_b2[d], &pl->stats.workspace_bytes)) return rc;
    }
    std::vector<cx<float>> tw16(256);
    for (int k = 0; k < 16; ++k)
        for (int r = 0; r < 16; ++r)
            tw16[16 * r + k] = mk<float>((float)cos(2.0 * kPi * r * k / 256.0), (float)(-sin(2.0 * kPi * r * k / 256.0)));
    cx<float>* d = nullptr;
    if (int rc = upload(&d, tw16, &pl->stats.workspace_bytes)) return rc;
    pl->d_tw16 = d;
    // pass-3 twiddles of the four transform sizes: exp(-2 pi i r i / Q) at [256 (r - 1) + i], Q = 512 << c, r < Q / 256
    std::vector<cx<float>> tw3;
    for (int c = 0; c < 4; ++c) {
        const int Q = 512 << c, RL = Q / 256;
        pl->tw3_off[c] = (int)tw3.size();
        for (int r = 1; r < RL; ++r)
            for (int i = 0; i < 256; ++i)
                tw3.push_back(mk<float>((float)cos(2.0 * kPi * r * i / Q), (float)(-sin(2.0 * kPi * r * i / Q))));
    }
    cx<float>* d3 = nullptr;
    if (int rc = upload(&d3, tw3, &pl->stats.workspace_bytes)) return rc;
    pl->d_tw3 = d3;
    CUDA_TRY((cudaError_t)fft3_setup());
    }
    return 0;
}

// twiddles, chirps and phases from double precision, Bluestein filters by a plan-time kernel, workspace
template <class T> int build_device_numeric(arkcos_plan* pl, const HostTables& t)
{
    const int PT = 1 << t.logPT;
    std::vector<cx<T>> tw(PT);
    for (int k = 0; k < PT; ++k) tw[k] = mk<T>((T)cos(2.0 * kPi * k / PT), (T)(-sin(2.0 * kPi * k / PT)));
    cx<T>* d_tw = nullptr;
    if (int rc = upload(&d_tw, tw, &pl->stats.workspace_bytes)) return rc;
    pl->d_tw = d_tw;
    std::vector<cx<T>> chirp((size_t)t.chirp_total), phase((size_t)t.ph_total);
    for (const FftLen& f : t.lens) {
        const int L = f.L, N = 2 * L;
        for (int k = 0; k <= L; ++k)                       // exp(-i pi k / N)
            phase[f.ph_off + k] = mk<T>((T)cos(kPi * k / N), (T)(-sin(kPi * k / N)));
        if (f.pow2) continue;
        for (int n = 0; n < L; ++n) {                      // exp(-i pi n^2 / L), phase reduced exactly
            const long long r = ((long long)n * n) % (2LL * L);
            chirp[f.chirp_off + n] = mk<T>((T)cos(kPi * (double)r / L), (T)(-sin(kPi * (double)r / L)));
        }
    }
    cx<T>*d_chirp = nullptr, *d_phase = nullptr;
    if (int rc = upload(&d_chirp, chirp, &pl->stats.workspace_bytes)) return rc;
    pl->d_chirp = d_chirp;
    if (int rc = upload(&d_phase, phase, &pl->stats.workspace_bytes)) return rc;
    pl->d_phase = d_phase;
    for (int d = 0; d < 2; ++d) {
        if (int rc = upload(&pl->d_fft_order[d], t.fft_order[d], &pl->stats.workspace_bytes)) return rc;
        pl->nfft_old[d] = (int)t.fft_order[d].size();
    }
    if (int rc = setup_fft3<T>(pl, t)) return rc;
    pl->fft_smem = fft_smem_elems(PT) * sizeof(cx<T>);
    pl->fft_bpt = PT <= 8 * kFftThreads * 2 ? 2 : 4;
    if (pl->fft_smem > 227 * 1024 || PT > 8 * kFftThreads * 4) return fail(ARKCOS_UNSUPPORTED, "ring too long for the shared-memory FFT");
    if (int rc = pl->fft_bpt == 2 ? set_fft_smem<T, 2>(pl->fft_smem) : set_fft_smem<T, 4>(pl->fft_smem)) return rc;

    const size_t fb = (size_t)std::max<int64_t>(t.filt_total, 1) * sizeof(cx<T>);
    CUDA_TRY(cudaMalloc(&pl->d_filt, fb));
    pl->stats.workspace_bytes += (int64_t)fb;
    if (!t.bluestein_ids.empty()) {
        int* d_which = nullptr;
        int64_t dummy = 0;
        if (int rc = upload(&d_which, t.bluestein_ids, &dummy)) return rc;
        if (pl->fft_bpt == 2)
            bluestein_filter_kernel<T, 2><<<(unsigned)t.bluestein_ids.size(), kFftThreads, pl->fft_smem>>>(
                pl->d_lens, d_which, d_tw, pl->logPT, d_chirp, (cx<T>*)pl->d_filt);
        else
            bluestein_filter_kernel<T, 4><<<(unsigned)t.bluestein_ids.size(), kFftThreads, pl->fft_smem>>>(
                pl->d_lens, d_which, d_tw, pl->logPT, d_chirp, (cx<T>*)pl->d_filt);
        cudaError_t e = cudaDeviceSynchronize();
        cudaFree(d_which);
        CUDA_TRY(e);
    }
    const size_t wb = (size_t)std::max<int64_t>(t.nsamples, 1) * sizeof(T);
    CUDA_TRY(cudaMalloc(&pl->d_W, wb));
    const size_t sb = (size_t)pl->max_nmaps * (size_t)pl->g.spec_total * sizeof(cx<T>);
    CUDA_TRY(cudaMalloc(&pl->d_specIn, sb));
    CUDA_TRY(cudaMalloc(&pl->d_specOut, sb));
    pl->stats.workspace_bytes += (int64_t)(wb + 2 * sb);
    return 0;
}
}  // namespace

namespace {

template <class T> int enqueue_rows(const arkcos_plan* pl, cudaStream_t st)
{
    if (pl->npairs > 0 && pl->nsamples > 0)
        kernel_rows_kernel<T><<<(unsigned)((pl->nsamples + 127) / 128), 128, 0, st>>>(pl->d_pairs, pl->d_wpair, pl->nsamples, pl->d_table, pl->ntab,
                                                                                      pl->theta_max, (T*)pl->d_W);
    return 0;
}

template <int TMAX, bool HAS_ODD> void launch_uniform_class(const arkcos_plan* pl, int cls, int nmaps, cudaStream_t st)
{
    if (pl->nitems[cls] == 0) return;
    band_mac_uniform_kernel<TMAX, HAS_ODD><<<dim3((unsigned)pl->nitems[cls], (unsigned)nmaps), kBandThreads, 0, st>>>(
        pl->d_items[cls], pl->d_north, pl->d_pairs, (const float*)pl->d_W, pl->d_rings, pl->g.R,
        (const cx<float>*)pl->spec_in(), (cx<float>*)pl->d_specOut, pl->g.spec_total);
}

// which: 1 = the big launches (class-E runs on st, cap runs on side stream 0), 2 = the small uniform classes (side stream 2),
// 3 = both in the order of the timing slots (serial timing mode).
void launch_uniform(const arkcos_plan* pl, int nmaps, cudaStream_t st, bool serial, int which)
{
    // every small class on a stream of its own: they are latency-bound, tiny grids
    cudaStream_t s1 = serial ? st : pl->side[2], s2 = serial ? st : pl->side[3], s3 = serial ? st : pl->side[4], sc = serial ? st : pl->side[0];
    auto launch_cap = [&](auto multi_tag, int first, int count, cudaStream_t sc) {
        constexpr bool MULTI = decltype(multi_tag)::value;
        if (count <= 0) return;
        const unsigned n = (unsigned)count;
        const CapChunkItem* items = pl->d_cap_chunk_items + first;
        if (pl->d_G && nmaps >= 4)
            band_mac_capchunk_cached_kernel<4, 4, MULTI, 1><<<dim3(n, (unsigned)((nmaps + 3) / 4)), 256, 0, sc>>>(
                items, pl->d_cap_chunks, pl->d_north, pl->d_pairs, pl->d_goff, pl->d_G, pl->d_rings, pl->g.R,
                (const cx<float>*)pl->spec_in(), (cx<float>*)pl->d_specOut, pl->g.spec_total, nmaps);
        else if (pl->d_G && nmaps > 1)
            band_mac_capchunk_cached_kernel<4, 2, MULTI, 2><<<dim3(n, (unsigned)((nmaps + 1) / 2)), kBandThreads, 0, sc>>>(
                items, pl->d_cap_chunks, pl->d_north, pl->d_pairs, pl->d_goff, pl->d_G, pl->d_rings, pl->g.R,
                (const cx<float>*)pl->spec_in(), (cx<float>*)pl->d_specOut, pl->g.spec_total, nmaps);
        else if (pl->d_G)
            band_mac_capchunk_cached_kernel<4, 1, MULTI, 2><<<dim3(n, 1), kBandThreads, 0, sc>>>(
                items, pl->d_cap_chunks, pl->d_north, pl->d_pairs, pl->d_goff, pl->d_G, pl->d_rings, pl->g.R,
                (const cx<float>*)pl->spec_in(), (cx<float>*)pl->d_specOut, pl->g.spec_total, nmaps);
        else if (pl->use_tc) {
            if (pl->ntc_items[MULTI ? 2 : 1] > 0)
                tc_launch(pl->tc_cfg, MULTI ? 3 : 2, (unsigned)pl->ntc_items[MULTI ? 2 : 1], (unsigned)nmaps, sc, pl->d_tc_items[MULTI ? 2 : 1],
                          pl->d_tc_chunks, pl->d_tc_tiles, pl->d_tc_cols, pl->d_tc_rings, (const float*)pl->d_W, pl->g.R,
                          (const cx<float>*)pl->spec_in(), (cx<float>*)pl->d_specOut, pl->g.spec_total);
        } else
            band_mac_capchunk_kernel<4, 20, MULTI><<<dim3(n, (unsigned)nmaps), kBandThreads, 0, sc>>>(
                items, pl->d_cap_chunks, pl->d_north, pl->d_pairs, (const float*)pl->d_W, pl->d_rings, pl->g.R,
                (const cx<float>*)pl->spec_in(), (cx<float>*)pl->d_specOut, pl->g.spec_total);
    };
    // the runs whose grids span several periods are few blocks (fewer than SMs): on a stream of their own and ahead of the
    // launches that fill the device; behind the single-period runs on one stream they ran alone on a quarter of the SMs
    if (!serial && (which & 1) && pl->ncapitems > 0) launch_cap(std::true_type{}, pl->ncapsingle, pl->ncapitems - pl->ncapsingle, pl->side[6]);
    if (!(which & 1)) {
    } else if (pl->neqchunks > 0 && pl->d_G) {
        const unsigned gx = (unsigned)((pl->eq_mh + 255) / 256);
        auto launch_eq = [&](auto nm_tag, auto mt_tag) {
            constexpr int NM = decltype(nm_tag)::value, MT = decltype(mt_tag)::value;
            band_mac_eq_cached_kernel<4, NM, MT><<<dim3(gx, (unsigned)pl->neqchunks, (unsigned)((nmaps + NM - 1) / NM)), 256 / MT,
                                                   cached_smem_bytes<NM>(), st>>>(
                pl->d_eqchunks, pl->d_north, pl->d_pairs, pl->d_goff, pl->d_G, pl->d_rings, pl->g.R,
                (const cx<float>*)pl->spec_in(), (cx<float>*)pl->d_specOut, pl->g.spec_total, nmaps);
        };
        // G is read once per group of maps: four maps per read (one mode per thread) from four maps on
        if (nmaps >= 4) launch_eq(std::integral_constant<int, 4>{}, std::integral_constant<int, 1>{});
        else if (nmaps > 1) launch_eq(std::integral_constant<int, 2>{}, std::integral_constant<int, 2>{});
        else launch_eq(std::integral_constant<int, 1>{}, std::integral_constant<int, 2>{});
    } else if (pl->neqchunks > 0 && pl->use_tc && pl->ntc_items[0] > 0) {
        tc_launch(pl->tc_cfg, pl->eq_alt ? 0 : 1, (unsigned)pl->ntc_items[0], (unsigned)nmaps, st, pl->d_tc_items[0], pl->d_tc_chunks, pl->d_tc_tiles,
                  pl->d_tc_cols, pl->d_tc_rings, (const float*)pl->d_W, pl->g.R, (const cx<float>*)pl->spec_in(), (cx<float>*)pl->d_specOut,
                  pl->g.spec_total);
    } else if (pl->neqchunks > 0) {
        constexpr int TI = 4, MT = 2;
        const dim3 grid((unsigned)((pl->eq_mh + kBandThreads * MT - 1) / (kBandThreads * MT)), (unsigned)pl->neqchunks, (unsigned)nmaps);
        if (pl->eq_alt)
            band_mac_eq_kernel<TI, MT, 12, 1><<<grid, kBandThreads, 0, st>>>(
                pl->d_eqchunks, pl->d_north, pl->d_pairs, (const float*)pl->d_W, pl->d_rings, pl->g.R,
                (const cx<float>*)pl->spec_in(), (cx<float>*)pl->d_specOut, pl->g.spec_total);
        else
            band_mac_eq_kernel<TI, MT, 12, 0><<<grid, kBandThreads, 0, st>>>(
                pl->d_eqchunks, pl->d_north, pl->d_pairs, (const float*)pl->d_W, pl->d_rings, pl->g.R,
                (const cx<float>*)pl->spec_in(), (cx<float>*)pl->d_specOut, pl->g.spec_total);
    }
    if (serial) cudaEventRecord(pl->ev_band[3], st);
    if (which & 2) launch_uniform_class<12, false>(pl, 2, nmaps, s1);
    if (serial) cudaEventRecord(pl->ev_band[4], st);
    if (which & 2) launch_uniform_class<20, false>(pl, 3, nmaps, s1);
    if (serial) cudaEventRecord(pl->ev_band[5], st);
    if (which & 2) launch_uniform_class<32, true>(pl, 4, nmaps, s2);
    if (serial) cudaEventRecord(pl->ev_band[6], st);
    if (which & 2) launch_uniform_class<12, true>(pl, 1, nmaps, s3);
    if ((which & 2) && pl->nnyq > 0)
        band_nyquist_eq_kernel<4><<<dim3((unsigned)((pl->nnyq + 3) / 4), (unsigned)nmaps), 128, 0, s3>>>(
            pl->d_nyq, pl->nnyq, pl->d_north, pl->d_pairs, (const float*)pl->d_W, pl->d_rings, pl->g.R,
            (const cx<float>*)pl->spec_in(), (cx<float>*)pl->d_specOut, pl->g.spec_total);
    if (serial) cudaEventRecord(pl->ev_band[7], st);
    if (pl->ncapitems > 0 && (which & 1)) {
        launch_cap(std::false_type{}, 0, pl->ncapsingle, sc);
        if (serial) {
            cudaEventRecord(pl->ev_band[8], st);
            launch_cap(std::true_type{}, pl->ncapsingle, pl->ncapitems - pl->ncapsingle, sc);
        }
    } else if (serial) cudaEventRecord(pl->ev_band[8], st);
    if (serial) cudaEventRecord(pl->ev_band[9], st);
}

// Ring FFTs of one direction (FWD: map -> specIn, else specOut -> map).  Float plans: one launch per transform size of the
// register-resident kernels (the largest on the caller's stream, the others forked onto the plan's side streams, they
// touch disjoint rings) plus the shared-memory kernel for whatever is left (very short or very long rings).
template <int LOGQ, bool FWD>
void launch_fft3(const arkcos_plan* pl, const void* d_in, void* d_out, int nmaps, cudaStream_t st)
{
    const int c = LOGQ - 9, dir = FWD ? 0 : 1, slot = 2 * (3 - c);
    if (pl->nfft3[dir][c] == 0) {
        if (pl->timing == 2) { cudaEventRecord(pl->ev_fft[dir][slot], st); cudaEventRecord(pl->ev_fft[dir][slot + 1], st); }
        return;
    }
    const HostGeometry& g = pl->g;
    Fft3Args a{};
    a.in = (const float*)d_in;
    a.outmap = (float*)d_out;
    a.npix = g.npix;
    a.spec = (cx<float>*)(FWD ? pl->spec_in() : pl->d_specOut);
    a.spec_stride = g.spec_total;
    a.tw = (const cx<float>*)pl->d_tw;
    a.tw16 = (const cx<float>*)pl->d_tw16;
    a.tw3 = (const cx<float>*)pl->d_tw3 + pl->tw3_off[c];
    a.filt = (const cx<float>*)pl->d_filt;
    a.chirp = (const cx<float>*)pl->d_chirp;
    a.phase = (const cx<float>*)pl->d_phase;
    a.logPT = pl->logPT;
    const int nb = pl->nfft3_bluestein[dir][c], nd = pl->nfft3[dir][c] - nb;
    if (pl->timing == 2) cudaEventRecord(pl->ev_fft[dir][slot], st);
    if (nd > 0)                                       // power-of-two rings: one transform per block
        fft3_launch_direct(LOGQ, FWD, pl->d_fft3_jobs[dir][c] + nb, (unsigned)nd, (unsigned)nmaps, st, a);
    if (pl->timing == 2) cudaEventRecord(pl->ev_fft[dir][slot + 1], st);
    if (nb > 0)
        fft3_launch_bluestein(LOGQ, FWD, pl->d_fft3_jobs[dir][c], (unsigned)nb, (unsigned)nmaps, st, a, pl->sm_count);
}

template <class T, bool FWD>
void launch_ring_ffts(const arkcos_plan* pl, const void* d_in, void* d_out, int nmaps, cudaStream_t st)
{
    const HostGeometry& g = pl->g;
    bool forked = false;
    auto launch_old = [&](cudaStream_t so) {            // the shared-memory kernel: very short or very long rings, fp64 plans
        if constexpr (sizeof(T) == 4) {
            if (pl->nfft3_d2[FWD ? 0 : 1] + pl->nfft3_b2[FWD ? 0 : 1] > 0) {   // rings of 8194 .. 16384 pixels on size-4096 transforms
                Fft3Args a{};
                a.in = (const float*)d_in;
                a.outmap = (float*)d_out;
                a.npix = g.npix;
                a.spec = (cx<float>*)(FWD ? pl->spec_in() : pl->d_specOut);
                a.spec_stride = g.spec_total;
                a.tw = (const cx<float>*)pl->d_tw;
                a.tw16 = (const cx<float>*)pl->d_tw16;
                a.tw3 = (const cx<float>*)pl->d_tw3 + pl->tw3_off[3];
                a.phase = (const cx<float>*)pl->d_phase;
                a.logPT = pl->logPT;
                a.filt = (const cx<float>*)pl->d_filt;
                a.chirp = (const cx<float>*)pl->d_chirp;
                if (pl->nfft3_b2[FWD ? 0 : 1] > 0)
                    fft3_launch_bluestein2(FWD, pl->d_fft3_b2[FWD ? 0 : 1], (unsigned)pl->nfft3_b2[FWD ? 0 : 1], (unsigned)nmaps, so, a);
                if (pl->nfft3_d2[FWD ? 0 : 1] > 0)
                    fft3_launch_direct2(FWD, pl->d_fft3_d2[FWD ? 0 : 1], (unsigned)pl->nfft3_d2[FWD ? 0 : 1], (unsigned)nmaps, so, a);
            }
        }
        if (pl->nfft_old[FWD ? 0 : 1] == 0) return;
        const dim3 gfft((unsigned)pl->nfft_old[FWD ? 0 : 1], (unsigned)nmaps);
        if (FWD) {
            if (pl->fft_bpt == 2)
                ring_fft_forward_kernel<T, 2><<<gfft, kFftThreads, pl->fft_smem, so>>>(
                    (const T*)d_in, g.npix, (cx<T>*)pl->spec_in(), g.spec_total, pl->d_rings, pl->d_fft_order[FWD ? 0 : 1], pl->d_lens,
                    (const cx<T>*)pl->d_tw, pl->logPT, (const cx<T>*)pl->d_filt, (const cx<T>*)pl->d_chirp, (const cx<T>*)pl->d_phase);
            else
                ring_fft_forward_kernel<T, 4><<<gfft, kFftThreads, pl->fft_smem, so>>>(
                    (const T*)d_in, g.npix, (cx<T>*)pl->spec_in(), g.spec_total, pl->d_rings, pl->d_fft_order[FWD ? 0 : 1], pl->d_lens,
                    (const cx<T>*)pl->d_tw, pl->logPT, (const cx<T>*)pl->d_filt, (const cx<T>*)pl->d_chirp, (const cx<T>*)pl->d_phase);
        } else {
            if (pl->fft_bpt == 2)
                ring_fft_inverse_kernel<T, 2><<<gfft, kFftThreads, pl->fft_smem, so>>>(
                    (const cx<T>*)pl->d_specOut, g.spec_total, (T*)d_out, g.npix, pl->d_rings, pl->d_fft_order[FWD ? 0 : 1], pl->d_lens,
                    (const cx<T>*)pl->d_tw, pl->logPT, (const cx<T>*)pl->d_filt, (const cx<T>*)pl->d_chirp, (const cx<T>*)pl->d_phase);
            else
                ring_fft_inverse_kernel<T, 4><<<gfft, kFftThreads, pl->fft_smem, so>>>(
                    (const cx<T>*)pl->d_specOut, g.spec_total, (T*)d_out, g.npix, pl->d_rings, pl->d_fft_order[FWD ? 0 : 1], pl->d_lens,
                    (const cx<T>*)pl->d_tw, pl->logPT, (const cx<T>*)pl->d_filt, (const cx<T>*)pl->d_chirp, (const cx<T>*)pl->d_phase);
        }
    };
    if constexpr (sizeof(T) == 4) {
        const int dir = FWD ? 0 : 1;
        const int nside_launches = (pl->nfft3[dir][2] > 0) + (pl->nfft3[dir][1] + pl->nfft3[dir][0] > 0) + (pl->nfft_old[dir] + pl->nfft3_d2[dir] + pl->nfft3_b2[dir] > 0);
        forked = pl->nfft3[dir][3] > 0 && nside_launches > 0 && pl->timing != 2;
        if (forked) {
            cudaEventRecord(pl->ev_fork, st);
            for (int k = 0; k < 3; ++k) cudaStreamWaitEvent(pl->side[k], pl->ev_fork, 0);
        }
        if (forked) {
            // the small size classes first (single-wave, latency-bound launches): the blocks of the big launches then fill the
            // SMs around them; issued behind the big launches they would only start in their last wave (-10 us per call)
            launch_fft3<9, FWD>(pl, d_in, d_out, nmaps, pl->side[1]);
            launch_fft3<10, FWD>(pl, d_in, d_out, nmaps, pl->side[1]);
            launch_fft3<11, FWD>(pl, d_in, d_out, nmaps, pl->side[0]);
            launch_fft3<12, FWD>(pl, d_in, d_out, nmaps, st);
        } else {                                      // one stream (timing mode 2: in the order of the event slots)
            launch_fft3<12, FWD>(pl, d_in, d_out, nmaps, st);
            launch_fft3<11, FWD>(pl, d_in, d_out, nmaps, st);
            launch_fft3<10, FWD>(pl, d_in, d_out, nmaps, st);
            launch_fft3<9, FWD>(pl, d_in, d_out, nmaps, st);
        }
    } else if (pl->timing == 2)
        for (int k = 0; k < 8; ++k) cudaEventRecord(pl->ev_fft[FWD ? 0 : 1][k], st);
    if (pl->timing == 2) cudaEventRecord(pl->ev_fft[FWD ? 0 : 1][8], st);
    launch_old(forked ? pl->side[2] : st);
    if (pl->timing == 2) cudaEventRecord(pl->ev_fft[FWD ? 0 : 1][9], st);
    if (forked)
        for (int k = 0; k < 3; ++k) {
            cudaEventRecord(pl->ev_join[k], pl->side[k]);
            cudaStreamWaitEvent(st, pl->ev_join[k], 0);
        }
}

// skip_forward: the input-ring spectra pl->spec_in() are already there (arkcos_convolve_multi: another plan of the same
// pixelization made them on this stream); d_in is then only read by the exact_caps direct sum.
template <class T> int enqueue_convolve(const arkcos_plan* pl, const void* d_in, void* d_out, int nmaps, cudaStream_t st, bool skip_forward = false)
{
    const HostGeometry& g = pl->g;
    const bool tm = pl->timing != 0;
    if (tm) cudaEventRecord(pl->ev[0], st);
    // the kernel rows do not depend on the map: outside the timing modes they are generated on a side stream of their own
    // while the forward FFTs run
    const bool rows_aside = !tm && !pl->opt.cache_kernel_rows && pl->npairs > 0;
    // the cap fold accumulates into the output spectrum: clear those ranges early, beside the forward FFTs as well
    auto clear_cap_ranges = [&](cudaStream_t q) {
        if (pl->ncapitems > 0)
            for (const auto& z : pl->cap_zero)
                for (int k = 0; k < nmaps; ++k)
                    cudaMemsetAsync((cx<float>*)pl->d_specOut + (int64_t)k * g.spec_total + z.first, 0,
                                    (size_t)z.second * sizeof(cx<float>), q);
    };
    const bool aside = !tm && pl->ncapitems > 0 && !rows_aside;
    if (rows_aside || aside) {
        cudaEventRecord(pl->ev_rows_fork, st);
        cudaStreamWaitEvent(pl->side_rows, pl->ev_rows_fork, 0);
        clear_cap_ranges(pl->side_rows);
        if (rows_aside) enqueue_rows<T>(pl, pl->side_rows);
        cudaEventRecord(pl->ev_rows_done, pl->side_rows);
    } else {
        clear_cap_ranges(st);
        if (!pl->opt.cache_kernel_rows) enqueue_rows<T>(pl, st);
    }
    if (tm) cudaEventRecord(pl->ev[1], st);
    if (!skip_forward) launch_ring_ffts<T, true>(pl, d_in, d_out, nmaps, st);
    if (rows_aside || aside) cudaStreamWaitEvent(st, pl->ev_rows_done, 0);
    if (tm) cudaEventRecord(pl->ev[2], st);
    // the band kernels of the different ring classes write disjoint rings: fork them onto the plan's side streams
    // (timing mode 2: one after the other on the caller's stream with an event between them)
    const bool serial = pl->timing == 2;
    // The small latency-bound kernels (general, pole, uniform classes: 25-45 us each whatever the device gives them) are issued
    // first, the big launches (tensor-core / run kernels, a whole SM per block) behind them: the big blocks take the SMs the
    // small kernels leave free and the others as they drain.  (Issued last, the small kernels only start in the big launches'
    // last wave and the stage ends 15 us later; measured both ways, profiles/r2_final.md.)
    cudaStream_t s0 = serial ? st : pl->side[1], sp = serial ? st : pl->side[5];
    if (!serial) {
        cudaEventRecord(pl->ev_fork, st);
        for (int k = 0; k < 7; ++k) cudaStreamWaitEvent(pl->side[k], pl->ev_fork, 0);
    }
    if (serial) cudaEventRecord(pl->ev_band[0], st);
    if (pl->nitems[0] > 0) {
        // the four-threads-per-mode form is latency-bound: six items per block (fewer, larger blocks)
        const int pk = pl->general_split == 4 ? kGeneralPack : 1;
        const dim3 gg((unsigned)((pl->nitems[0] + pk - 1) / pk), (unsigned)nmaps), bb((unsigned)kBandThreads, (unsigned)pk);
        if (pl->general_split == 4)
            band_mac_general_kernel<T, 16, 4><<<gg, bb, 0, s0>>>(
                pl->d_items[0], pl->nitems[0], pl->d_north, pl->d_pairs, (const T*)pl->d_W, pl->d_rings, g.R, (const cx<T>*)pl->spec_in(),
                (cx<T>*)pl->d_specOut, g.spec_total, pl->opt.variant == 1 ? 1 : 0);
        else
            band_mac_general_kernel<T, 16, 1><<<gg, bb, 0, s0>>>(
                pl->d_items[0], pl->nitems[0], pl->d_north, pl->d_pairs, (const T*)pl->d_W, pl->d_rings, g.R, (const cx<T>*)pl->spec_in(),
                (cx<T>*)pl->d_specOut, g.spec_total, pl->opt.variant == 1 ? 1 : 0);
    }
    if (serial) cudaEventRecord(pl->ev_band[1], st);
    if (pl->npole > 0 && !pl->pole_warp_per_mode)
        band_mac_pole1_kernel<T, 16><<<dim3((unsigned)pl->npole, (unsigned)nmaps), kPoleThreads,
                                        2 * (size_t)(pl->pole_mh + 1) * sizeof(cx<T>), sp>>>(
            pl->d_pole, pl->d_north, pl->d_pairs, (const T*)pl->d_W, pl->d_rings, g.R, (const cx<T>*)pl->spec_in(),
            (cx<T>*)pl->d_specOut, g.spec_total);
    else if (pl->npole > 0) {
        const int tstride = pl->pole_mh + 1, bpr = (tstride + kPoleWarps - 1) / kPoleWarps;
        band_mac_pole_kernel<T><<<dim3((unsigned)(pl->npole * bpr), (unsigned)nmaps), kPoleThreads, 0, sp>>>(
            pl->d_pole, bpr, pl->d_north, pl->d_pairs, (const T*)pl->d_W, pl->d_rings, g.R, (const cx<T>*)pl->spec_in(), g.spec_total,
            (cx<T>*)pl->d_pole_scratch, tstride);
        band_mac_pole_fold_kernel<T><<<dim3((unsigned)pl->npole, (unsigned)nmaps), kPoleThreads, 0, sp>>>(
            pl->d_pole, pl->d_north, pl->d_pairs, pl->d_rings, g.R, (const cx<T>*)pl->d_pole_scratch, tstride, (cx<T>*)pl->d_specOut,
            g.spec_total);
    }
    if (serial) cudaEventRecord(pl->ev_band[2], st);
    launch_uniform(pl, nmaps, st, serial, serial ? 3 : 2);
    if (!serial) launch_uniform(pl, nmaps, st, false, 1);
    if (!serial)
        for (int k = 0; k < 7; ++k) {
            cudaEventRecord(pl->ev_join[k], pl->side[k]);
            cudaStreamWaitEvent(st, pl->ev_join[k], 0);
        }
    if (tm) cudaEventRecord(pl->ev[3], st);
    launch_ring_ffts<T, false>(pl, d_in, d_out, nmaps, st);
    if (pl->ndirect > 0) {                      // exact_caps: overwrite the cap-zone rings with the direct-space sum
        const double sh = sin(0.5 * pl->theta_max), xmax = 4.0 * sh * sh;
        auto launch = [&](auto nm_tag) {
            constexpr int NM = decltype(nm_tag)::value;
            direct_rings_kernel<T, NM, 4><<<dim3((unsigned)pl->ndirect, (unsigned)((nmaps + NM - 1) / NM)), kDirectThreads, DirectCfg<T, NM>::smem, st>>>(
                pl->d_direct_items, pl->d_north, pl->d_pairs, pl->d_rings, g.R, (const double2*)pl->d_table2, pl->ntab, pl->theta_max, xmax,
                (const T*)d_in, (T*)d_out, g.npix, nmaps);
        };
        // a thread holds 8 accumulators per map (four quadrants, two hemispheres)
        constexpr int kMaxNM = sizeof(T) == 4 ? 8 : 4;
        if (nmaps >= 5 && kMaxNM >= 8) launch(std::integral_constant<int, kMaxNM>{});
        else if (nmaps >= 3) launch(std::integral_constant<int, 4>{});
        else if (nmaps == 2) launch(std::integral_constant<int, 2>{});
        else launch(std::integral_constant<int, 1>{});
    }
    if (tm) cudaEventRecord(pl->ev[4], st);
    CUDA_TRY(cudaGetLastError());
    return 0;
}

__global__ void fma_chain_kernel(float* out, int iters, float a, float b)
{
    float x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; ++i) {
        x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
        x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
}

size_t elem_size(arkcos_dtype d) { return d == ARKCOS_F64 ? 8 : 4; }

}  // namespace

// arkcos_convolve_no_alloc: the spectra and the pole scratch of a call, in the library image instead of the plan's workspace.
// In host code the name below is a host-side stand-in, not a device address: g_no_alloc_ptr[device] is the address
// cudaGetSymbolAddress gave on that device, looked up once per device with that device current.
static __device__ __align__(256) unsigned char g_no_alloc_scratch[ARKCOS_NO_ALLOC_SCRATCH_BYTES];
static const int kNoAllocMaxDevices = 64;
static void* g_no_alloc_ptr[kNoAllocMaxDevices] = {};
static std::mutex g_no_alloc_mutex;

extern "C" {

static int plan_create_impl(arkcos_plan** out, const arkcos_pixelization* pix, const arkcos_kernel* kernel, arkcos_dtype dtype,
                            const arkcos_options* options, bool tables_only)
{
    if (!out || !pix || !kernel || !kernel->table) return fail(ARKCOS_INVALID_ARG, "NULL argument");
    if (dtype != ARKCOS_F32 && dtype != ARKCOS_F64) return fail(ARKCOS_INVALID_ARG, "bad dtype");
    if (kernel->n < 2 || !(kernel->theta_max > 0.0) || !(kernel->theta_max <= kPi + 1e-12))
        return fail(ARKCOS_INVALID_ARG, "kernel: need n >= 2 and 0 < theta_max <= pi");
    arkcos_options opt{};
    if (options) opt = *options;
    for (int r : opt.reserved) if (r != 0) return fail(ARKCOS_INVALID_ARG, "options.reserved must be zero");
    if (opt.variant != 0 && opt.variant != 1) return fail(ARKCOS_INVALID_ARG, "options.variant must be 0 or 1");
    if (opt.exact_caps != 0 && opt.exact_caps != 1) return fail(ARKCOS_INVALID_ARG, "options.exact_caps must be 0 or 1");
    if (opt.cache_kernel_spectra != 0 && opt.cache_kernel_spectra != 1)
        return fail(ARKCOS_INVALID_ARG, "options.cache_kernel_spectra must be 0 or 1");
    if (opt.no_tensor_cores != 0 && opt.no_tensor_cores != 1) return fail(ARKCOS_INVALID_ARG, "options.no_tensor_cores must be 0 or 1");
    if (opt.no_cuda_graph != 0 && opt.no_cuda_graph != 1) return fail(ARKCOS_INVALID_ARG, "options.no_cuda_graph must be 0 or 1");
    if (opt.cache_kernel_spectra && (dtype != ARKCOS_F32 || opt.variant != 0))
        return fail(ARKCOS_UNSUPPORTED, "cache_kernel_spectra needs a float plan of variant 0");
    if (opt.cache_kernel_spectra) opt.cache_kernel_rows = 1;     // the spectra are made from the rows, once
    if (opt.max_nmaps < 0 || opt.polar_oversample < 0 || opt.ell_nyquist < 0.0 || opt.max_nmaps > 65535)
        return fail(ARKCOS_INVALID_ARG, "negative option");
    const int maxlen = dtype == ARKCOS_F32 ? 16384 : 8192;
    if (pix->kind == ARKCOS_ECP) {
        if (pix->ntheta < 1 || pix->ntheta > (1 << 20) || !is_pow2(pix->nphi) || pix->nphi < 4 || pix->nphi > maxlen)
            return fail(ARKCOS_INVALID_ARG, "ECP: need ntheta >= 1 and nphi a power of two in [4, 16384 (f32) / 8192 (f64)]");
    } else if (pix->kind == ARKCOS_HEALPIX_RING) {
        if (!is_pow2(pix->nside) || 4 * pix->nside > maxlen)
            return fail(ARKCOS_INVALID_ARG, "HEALPix: nside must be a power of two <= 4096 (f32) / 2048 (f64)");
    } else return fail(ARKCOS_INVALID_ARG, "bad pixelization kind");

    arkcos_plan* pl = new (std::nothrow) arkcos_plan();
    if (!pl) return fail(ARKCOS_OUT_OF_MEMORY, "host allocation");
    struct Guard { arkcos_plan* p; ~Guard() { if (p) arkcos_plan_destroy(p); } } guard{pl};
    pl->dtype = dtype;
    pl->pix = *pix;
    pl->opt = opt;
    pl->theta_max = kernel->theta_max;
    pl->ntab = kernel->n;
    pl->max_nmaps = opt.max_nmaps > 0 ? opt.max_nmaps : 1;
    pl->tables_only = tables_only;
    if (!tables_only) CUDA_TRY(cudaGetDevice(&pl->device));

    build_geometry(*pix, pl->g);
    // the band kernels index the ring spectra of one map with 32-bit offsets
    if (pl->g.spec_total >= (int64_t)INT32_MAX) return fail(ARKCOS_UNSUPPORTED, "pixelization too large: ring spectra of one map exceed 2^31 coefficients");
    build_bands(pl->g, pl->theta_max);
    int fixed_mprime = 0;
    if (pix->kind == ARKCOS_HEALPIX_RING) {
        if (opt.polar_oversample > 0) fixed_mprime = opt.polar_oversample * 4 * pix->nside;
        else pl->ell_nyquist = opt.ell_nyquist > 0.0 ? opt.ell_nyquist
                                                     : auto_ell_nyquist(kernel->table, kernel->n, kernel->theta_max, 8.0 * pix->nside);
    }
    int sm_count = 148;
    if (!tables_only) CUDA_TRY(cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, pl->device));
    pl->sm_count = sm_count;
    HostTables t;
    // exact_caps: every output ring whose band contains a ring shorter than the longest one (the caps and the equatorial
    // rings next to them) comes from the direct-space sum; the hybrid pass then needs forward transforms of the full-length
    // rings only (the bands of the rings it still serves hold nothing else) and inverse transforms of those rings alone
    std::vector<char> need[2] = {std::vector<char>(pl->g.R, 1), std::vector<char>(pl->g.R, 1)};
    pl->g.direct.assign(pl->g.R, 0);
    if (opt.exact_caps && pix->kind == ARKCOS_HEALPIX_RING) {
        HostGeometry& g = pl->g;
        const int nmax = *std::max_element(g.n.begin(), g.n.end());
        for (int i = 0; i < g.R; ++i) {
            bool all_full = true;
            for (int j = g.band_lo[i]; j <= g.band_hi[i]; ++j) all_full = all_full && g.n[j] == nmax;
            g.direct[i] = all_full ? 0 : 1;
            need[0][i] = g.n[i] == nmax;
            need[1][i] = all_full;
        }
    }
    build_fft_lens(pl->g, t, pl->stats, dtype == ARKCOS_F32, need);
    build_pairs(pl->g, pl->theta_max, pl->ell_nyquist, fixed_mprime, kBandThreads, dtype == ARKCOS_F32 && opt.variant == 0, opt.variant == 0, opt.cache_kernel_spectra != 0, opt.no_tensor_cores == 0, sm_count, t, pl->stats);
    if (t.pairs.size() > (size_t)INT32_MAX) return fail(ARKCOS_UNSUPPORTED, "too many ring pairs");
    pl->nnorth = (int)t.north.size();
    pl->npairs = (int)t.pairs.size();
    for (int c = 0; c < kBandClasses; ++c) pl->nitems[c] = (int)t.items[c].size();
    pl->neqchunks = (int)t.eq_chunks.size();
    pl->use_tc = t.use_tc;
    pl->tc_cfg = t.tc_cfg;
    for (int c = 0; c < 3; ++c) pl->ntc_items[c] = (int)t.tc_items[c].size();
    if (t.nsamples / 4 >= (1 << 25)) return fail(ARKCOS_UNSUPPORTED, "too many kernel-row samples");
    pl->npole = (int)t.pole_rings.size();
    pl->nnyq = (int)t.nyq_rings.size();
    pl->pole_mh = t.pole_mh;
    pl->general_split = t.general_split;
    pl->pole_warp_per_mode = t.pole_warp_per_mode;
    pl->eq_alt = t.eq_alt;
    pl->eq_mh = t.eq_chunks.empty() ? 0 : pl->g.n[t.eq_chunks[0].i0] / 2;
    for (const EqChunk& c : t.eq_chunks) pl->eq_mh = std::max(pl->eq_mh, pl->g.n[c.i0] / 2);
    pl->nsamples = t.nsamples;
    pl->logPT = t.logPT;
    for (int d = 0; d < 2; ++d) {
        pl->nfft_old[d] = (int)t.fft_order[d].size();
        for (int c = 0; c < 4; ++c) {
            pl->nfft3[d][c] = (int)t.fft3_jobs[d][c].size();
            pl->nfft3_bluestein[d][c] = 0;
            for (const FftJob& j : t.fft3_jobs[d][c]) pl->nfft3_bluestein[d][c] += j.f.pow2 ? 0 : 1;
        }
    }

    if (tables_only) {
        guard.p = nullptr;
        *out = pl;
        return ARKCOS_OK;
    }
    int64_t* wsb = &pl->stats.workspace_bytes;
    if (int rc = upload(&pl->d_rings, t.rings, wsb)) return rc;
    if (int rc = upload(&pl->d_lens, t.lens, wsb)) return rc;
    if (int rc = upload(&pl->d_pairs, t.pairs, wsb)) return rc;
    {
        // ring pair of every group of four stored row samples (kernel_rows_kernel: one thread per sample)
        std::vector<int> wpair((size_t)(t.nsamples / 4), 0);
        for (size_t p = 0; p < t.pairs.size(); ++p)
            for (int64_t q = t.pairs[p].woff / 4, e = q + (t.pairs[p].cnt + 3) / 4; q < e; ++q) wpair[(size_t)q] = (int)p;
        if (int rc = upload(&pl->d_wpair, wpair, wsb)) return rc;
    }
    if (int rc = upload(&pl->d_north, t.north, wsb)) return rc;
    for (int c = 0; c < kBandClasses; ++c)
        if (int rc = upload(&pl->d_items[c], t.items[c], wsb)) return rc;
    if (int rc = upload(&pl->d_eqchunks, t.eq_chunks, wsb)) return rc;
    if (int rc = upload(&pl->d_pole, t.pole_rings, wsb)) return rc;
    if (int rc = upload(&pl->d_nyq, t.nyq_rings, wsb)) return rc;
    if (!t.pole_rings.empty()) {                // unfolded spectra T[m] of the pole kernel, ring and mirror image, per map
        const size_t nb = (size_t)pl->max_nmaps * t.pole_rings.size() * 2 * (size_t)(t.pole_mh + 1) * 2 * elem_size(dtype);
        CUDA_TRY(cudaMalloc(&pl->d_pole_scratch, nb));
        *wsb += (int64_t)nb;
    }
    if (opt.exact_caps && pix->kind == ARKCOS_HEALPIX_RING) {
        const HostGeometry& g = pl->g;
        std::vector<BandItem> items;
        for (int i = 0; i < (g.R + 1) / 2; ++i) {
            if (!g.direct[i]) continue;
            if (g.n[i] % 4 != 0) return fail(ARKCOS_UNSUPPORTED, "exact_caps needs rings of a multiple of four pixels");
            for (int k0 = 0; k0 < g.n[i] / 4; k0 += kDirectThreads) items.push_back(BandItem{i, k0});     // first quadrant
        }
        pl->ndirect = (int)items.size();
        if (int rc = upload(&pl->d_direct_items, items, wsb)) return rc;
        // profile table as (K[t], K[t+1] - K[t]): one 16-byte load per interpolation
        std::vector<double> tab2(2 * (size_t)(kernel->n - 1));
        for (int tt = 0; tt + 1 < kernel->n; ++tt) {
            tab2[2 * (size_t)tt] = kernel->table[tt];
            tab2[2 * (size_t)tt + 1] = kernel->table[tt + 1] - kernel->table[tt];
        }
        if (int rc = upload(&pl->d_table2, tab2, wsb)) return rc;
        // the instantiations that stage input windows use more than 48 KB of dynamic shared memory
        if (dtype == ARKCOS_F32) {
            CUDA_TRY(cudaFuncSetAttribute(direct_rings_kernel<float, 8, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)DirectCfg<float, 8>::smem));
            CUDA_TRY(cudaFuncSetAttribute(direct_rings_kernel<float, 4, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)DirectCfg<float, 4>::smem));
        } else
            CUDA_TRY(cudaFuncSetAttribute(direct_rings_kernel<double, 4, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)DirectCfg<double, 4>::smem));
    }
    if (pl->use_tc) {
        if (int rc = upload(&pl->d_tc_chunks, t.tc_chunks, wsb)) return rc;
        if (int rc = upload(&pl->d_tc_tiles, t.tc_tiles, wsb)) return rc;
        if (int rc = upload(&pl->d_tc_cols, t.tc_cols, wsb)) return rc;
        if (int rc = upload(&pl->d_tc_rings, t.tc_rings, wsb)) return rc;
        for (int c = 0; c < 3; ++c)
            if (int rc = upload(&pl->d_tc_items[c], t.tc_items[c], wsb)) return rc;
        CUDA_TRY((cudaError_t)tc_setup(pl->tc_cfg, &pl->tc_blocks_per_sm));
    }
    if (int rc = upload(&pl->d_cap_chunks, t.cap_chunks, wsb)) return rc;
    if (int rc = upload(&pl->d_cap_chunk_items, t.cap_chunk_items, wsb)) return rc;
    pl->ncapitems = (int)t.cap_chunk_items.size();
    pl->ncapsingle = t.cap_nsingle;
    pl->cap_zero = t.cap_zero;
    std::vector<double> tab(kernel->table, kernel->table + kernel->n);
    if (int rc = upload(&pl->d_table, tab, wsb)) return rc;
    if (int rc = dtype == ARKCOS_F32 ? build_device_numeric<float>(pl, t) : build_device_numeric<double>(pl, t)) return rc;
    for (auto& e : pl->ev) CUDA_TRY(cudaEventCreate(&e));
    for (auto& e : pl->ev_band) CUDA_TRY(cudaEventCreate(&e));
    for (auto& d : pl->ev_fft) for (auto& e : d) CUDA_TRY(cudaEventCreate(&e));
    CUDA_TRY(cudaEventCreateWithFlags(&pl->ev_fork, cudaEventDisableTiming));
    for (auto& e : pl->ev_join) CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    for (auto& q : pl->side) CUDA_TRY(cudaStreamCreateWithFlags(&q, cudaStreamNonBlocking));
    CUDA_TRY(cudaStreamCreateWithFlags(&pl->side_rows, cudaStreamNonBlocking));
    CUDA_TRY(cudaEventCreateWithFlags(&pl->ev_rows_fork, cudaEventDisableTiming));
    CUDA_TRY(cudaEventCreateWithFlags(&pl->ev_rows_done, cudaEventDisableTiming));
    if (opt.cache_kernel_rows) {
        dtype == ARKCOS_F32 ? enqueue_rows<float>(pl, 0) : enqueue_rows<double>(pl, 0);
        CUDA_TRY(cudaDeviceSynchronize());
    }
    if (opt.cache_kernel_spectra && pl->npairs > 0) {
        CUDA_TRY(cudaFuncSetAttribute(band_mac_eq_cached_kernel<4, 4, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cached_smem_bytes<4>()));
        // one row of M/2 + 1 floats per northern ring pair, padded to a multiple of four
        std::vector<uint32_t> goff(t.pairs.size());
        uint64_t n4 = 0;
        int mh_max = 0;
        for (size_t p = 0; p < t.pairs.size(); ++p) {
            goff[p] = (uint32_t)n4;
            n4 += (uint64_t)(t.pairs[p].M / 2 + 1 + 3) / 4;
            mh_max = std::max(mh_max, t.pairs[p].M / 2);
        }
        if (n4 >= 0xffffffffull) return fail(ARKCOS_UNSUPPORTED, "kernel spectra too large to cache");
        if (int rc = upload(&pl->d_goff, goff, wsb)) return rc;
        CUDA_TRY(cudaMalloc(&pl->d_G, (size_t)n4 * 16));
        pl->stats.workspace_bytes += (int64_t)n4 * 16;
        CUDA_TRY(cudaMemset(pl->d_G, 0, (size_t)n4 * 16));
        kernel_spectra_kernel<<<dim3((unsigned)pl->npairs, (unsigned)(mh_max / 256 + 1)), 256>>>(
            pl->d_pairs, (const float*)pl->d_W, pl->d_goff, pl->d_G);
        CUDA_TRY(cudaDeviceSynchronize());
    }
    CUDA_TRY(cudaGetLastError());
    guard.p = nullptr;
    *out = pl;
    g_last_error.clear();
    return ARKCOS_OK;
}

int arkcos_plan_create(arkcos_plan** out, const arkcos_pixelization* pix, const arkcos_kernel* kernel, arkcos_dtype dtype,
                       const arkcos_options* options)
{
    return plan_create_impl(out, pix, kernel, dtype, options, false);
}

int arkcos_plan_create_tables_only(arkcos_plan** out, const arkcos_pixelization* pix, const arkcos_kernel* kernel,
                                   arkcos_dtype dtype, const arkcos_options* options)
{
    return plan_create_impl(out, pix, kernel, dtype, options, true);
}

int arkcos_convolve(const arkcos_plan* pl, const void* d_in, void* d_out, int nmaps, void* cuda_stream)
{
    if (!pl || !d_in || !d_out) return fail(ARKCOS_INVALID_ARG, "NULL argument");
    if (pl->tables_only) return fail(ARKCOS_INVALID_ARG, "plan was created with arkcos_plan_create_tables_only");
    if (nmaps < 1 || nmaps > pl->max_nmaps) return fail(ARKCOS_INVALID_ARG, "nmaps must be in [1, max_nmaps]");
    const size_t bytes = (size_t)nmaps * (size_t)pl->g.npix * elem_size(pl->dtype);
    const char *a = (const char*)d_in, *b = (const char*)d_out;
    if (a < b + bytes && b < a + bytes) return fail(ARKCOS_INVALID_ARG, "d_in and d_out overlap");
    if (((uintptr_t)d_in | (uintptr_t)d_out) & 15) return fail(ARKCOS_INVALID_ARG, "d_in / d_out must be 16-byte aligned");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev != pl->device) return fail(ARKCOS_INVALID_ARG, "the current device is not the device the plan was created on");
    auto enqueue = [&]() {
        return pl->dtype == ARKCOS_F32 ? enqueue_convolve<float>(pl, d_in, d_out, nmaps, st)
                                       : enqueue_convolve<double>(pl, d_in, d_out, nmaps, st);
    };
    // One graph launch instead of ~30 kernel launches and their cross-stream events (options.no_cuda_graph).
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    const bool graph_ok = !pl->opt.no_cuda_graph && pl->timing == 0 && st != nullptr && st != cudaStreamLegacy &&
                          st != cudaStreamPerThread && cudaStreamIsCapturing(st, &cap) == cudaSuccess && cap == cudaStreamCaptureStatusNone;
    if (!graph_ok) return enqueue();
    for (size_t k = 0; k < pl->graphs.size(); ++k) {
        const arkcos_plan::GraphEntry e = pl->graphs[k];
        if (e.in == d_in && e.out == d_out && e.nmaps == nmaps && e.st == st) {
            if (k > 0) { pl->graphs.erase(pl->graphs.begin() + k); pl->graphs.insert(pl->graphs.begin(), e); }
            CUDA_TRY(cudaGraphLaunch(e.exec, st));
            return ARKCOS_OK;
        }
    }
    if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
        cudaGetLastError();
        return enqueue();
    }
    const int rc = enqueue();
    cudaGraph_t graph = nullptr;
    const cudaError_t ce = cudaStreamEndCapture(st, &graph);
    cudaGraphExec_t exec = nullptr;
    if (rc != ARKCOS_OK || ce != cudaSuccess || !graph || cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) {
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        return rc != ARKCOS_OK ? rc : enqueue();                // capture refused: launch directly
    }
    cudaGraphDestroy(graph);
    if (pl->graphs.size() >= 4) { cudaGraphExecDestroy(pl->graphs.back().exec); pl->graphs.pop_back(); }
    pl->graphs.insert(pl->graphs.begin(), arkcos_plan::GraphEntry{d_in, d_out, nmaps, st, exec});
    CUDA_TRY(cudaGraphLaunch(exec, st));
    return ARKCOS_OK;
}

int arkcos_convolve_no_alloc(const arkcos_plan* pl, const void* d_in, void* d_out, int nmaps, void* cuda_stream)
{
    if (!pl || !d_in || !d_out) return fail(ARKCOS_INVALID_ARG, "NULL argument");
    if (pl->tables_only) return fail(ARKCOS_INVALID_ARG, "plan was created with arkcos_plan_create_tables_only");
    if (nmaps < 1 || nmaps > pl->max_nmaps) return fail(ARKCOS_INVALID_ARG, "nmaps must be in [1, max_nmaps]");
    const size_t bytes = (size_t)nmaps * (size_t)pl->g.npix * elem_size(pl->dtype);
    const char *a = (const char*)d_in, *b = (const char*)d_out;
    if (a < b + bytes && b < a + bytes) return fail(ARKCOS_INVALID_ARG, "d_in and d_out overlap");
    if (((uintptr_t)d_in | (uintptr_t)d_out) & 15) return fail(ARKCOS_INVALID_ARG, "d_in / d_out must be 16-byte aligned");
    // layout of the shared array: [input-ring spectra | output-ring spectra | unfolded pole spectra], each 256-byte aligned,
    // per-map strides as in the plan's own workspace (build_device_numeric, plan_create_impl)
    auto up = [](size_t x) { return (x + 255) & ~(size_t)255; };
    const size_t sb = up((size_t)nmaps * (size_t)pl->g.spec_total * 2 * elem_size(pl->dtype));
    const size_t pb = pl->d_pole_scratch ? up((size_t)nmaps * (size_t)pl->npole * 2 * (size_t)(pl->pole_mh + 1) * 2 * elem_size(pl->dtype)) : 0;
    const size_t need = 2 * sb + pb;
    if (need > (size_t)ARKCOS_NO_ALLOC_SCRATCH_BYTES)
        return fail(ARKCOS_INVALID_ARG, "arkcos_convolve_no_alloc: this plan with " + std::to_string(nmaps) + " map(s) needs " +
                                            std::to_string(need) + " bytes of scratch, the library holds ARKCOS_NO_ALLOC_SCRATCH_BYTES = " +
                                            std::to_string((size_t)ARKCOS_NO_ALLOC_SCRATCH_BYTES) + "; use arkcos_convolve");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev != pl->device) return fail(ARKCOS_INVALID_ARG, "the current device is not the device the plan was created on");
    if (dev < 0 || dev >= kNoAllocMaxDevices) return fail(ARKCOS_INVALID_ARG, "device ordinal beyond the table of scratch addresses");
    unsigned char* base = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_no_alloc_mutex);
        if (!g_no_alloc_ptr[dev]) {
            void* p = nullptr;
            CUDA_TRY(cudaGetSymbolAddress(&p, g_no_alloc_scratch));
            g_no_alloc_ptr[dev] = p;
        }
        base = (unsigned char*)g_no_alloc_ptr[dev];
    }
    // the array keeps the last call's contents (any plan's): start from zeros in the part this call uses
    CUDA_TRY(cudaMemsetAsync(base, 0, need, st));
    // the launches read the three addresses from the plan: point them at the array for the time of the enqueue
    arkcos_plan* mpl = const_cast<arkcos_plan*>(pl);
    void* const keep_in = pl->spec_in_shared;
    void* const keep_out = pl->d_specOut;
    void* const keep_pole = pl->d_pole_scratch;
    mpl->spec_in_shared = base;
    mpl->d_specOut = base + sb;
    if (pb) mpl->d_pole_scratch = base + 2 * sb;
    const int rc = pl->dtype == ARKCOS_F32 ? enqueue_convolve<float>(pl, d_in, d_out, nmaps, st)
                                           : enqueue_convolve<double>(pl, d_in, d_out, nmaps, st);
    mpl->spec_in_shared = keep_in;
    mpl->d_specOut = keep_out;
    mpl->d_pole_scratch = keep_pole;
    return rc;
}

int arkcos_convolve_multi(const arkcos_plan* const* plans, int nkernels, const void* d_in, void* d_out, int nmaps, void* cuda_stream)
{
    if (!plans || nkernels < 1 || !d_in || !d_out) return fail(ARKCOS_INVALID_ARG, "NULL argument or nkernels < 1");
    const arkcos_plan* p0 = plans[0];
    if (!p0) return fail(ARKCOS_INVALID_ARG, "NULL plan");
    for (int k = 0; k < nkernels; ++k) {
        const arkcos_plan* pk = plans[k];
        if (!pk || pk->tables_only) return fail(ARKCOS_INVALID_ARG, "NULL or tables-only plan");
        // one forward transform serves every kernel only if the ring spectra have one layout and one meaning
        if (pk->pix.kind != p0->pix.kind || pk->pix.ntheta != p0->pix.ntheta || pk->pix.nphi != p0->pix.nphi ||
            pk->pix.nside != p0->pix.nside || pk->dtype != p0->dtype || pk->device != p0->device)
            return fail(ARKCOS_INVALID_ARG, "arkcos_convolve_multi: the plans must share pixelization, dtype and device");
        if (nmaps < 1 || nmaps > pk->max_nmaps) return fail(ARKCOS_INVALID_ARG, "nmaps must be in [1, max_nmaps] of every plan");
        for (int q = 0; q < k; ++q)
            if (plans[q] == pk) return fail(ARKCOS_INVALID_ARG, "arkcos_convolve_multi: a plan appears twice (one workspace per plan)");
    }
    const size_t bytes = (size_t)nmaps * (size_t)p0->g.npix * elem_size(p0->dtype);
    const char *a = (const char*)d_in, *b = (const char*)d_out;
    if (a < b + bytes * (size_t)nkernels && b < a + bytes) return fail(ARKCOS_INVALID_ARG, "d_in and d_out overlap");
    if (((uintptr_t)d_in | (uintptr_t)d_out | (uintptr_t)bytes) & 15) return fail(ARKCOS_INVALID_ARG, "d_in / d_out / nmaps * npix * element size must be multiples of 16 bytes");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev != p0->device) return fail(ARKCOS_INVALID_ARG, "the current device is not the device the plans were created on");
    for (int k = 0; k < nkernels; ++k) {
        const arkcos_plan* pk = plans[k];
        void* out_k = (char*)d_out + (size_t)k * bytes;
        pk->spec_in_shared = k > 0 ? p0->d_specIn : nullptr;
        const int rc = pk->dtype == ARKCOS_F32 ? enqueue_convolve<float>(pk, d_in, out_k, nmaps, st, k > 0)
                                               : enqueue_convolve<double>(pk, d_in, out_k, nmaps, st, k > 0);
        pk->spec_in_shared = nullptr;
        if (rc) return rc;
    }
    return ARKCOS_OK;
}

int arkcos_convolve_host(const arkcos_plan* pl, const void* h_in, void* h_out, int nmaps, void* cuda_stream)
{
    if (!pl || !h_in || !h_out) return fail(ARKCOS_INVALID_ARG, "NULL argument");
    if (pl->tables_only) return fail(ARKCOS_INVALID_ARG, "plan was created with arkcos_plan_create_tables_only");
    if (nmaps < 1 || nmaps > pl->max_nmaps) return fail(ARKCOS_INVALID_ARG, "nmaps must be in [1, max_nmaps]");
    const size_t full = (size_t)pl->max_nmaps * (size_t)pl->g.npix * elem_size(pl->dtype);
    const size_t bytes = (size_t)nmaps * (size_t)pl->g.npix * elem_size(pl->dtype);
    if (!pl->d_stage_in) CUDA_TRY(cudaMalloc(&pl->d_stage_in, full));
    if (!pl->d_stage_out) CUDA_TRY(cudaMalloc(&pl->d_stage_out, full));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CUDA_TRY(cudaMemcpyAsync(pl->d_stage_in, h_in, bytes, cudaMemcpyHostToDevice, st));
    if (int rc = arkcos_convolve(pl, pl->d_stage_in, pl->d_stage_out, nmaps, cuda_stream)) return rc;
    CUDA_TRY(cudaMemcpyAsync(h_out, pl->d_stage_out, bytes, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return ARKCOS_OK;
}

int arkcos_convolve_host_async(const arkcos_plan* pl, const void* h_in, void* h_out, int nmaps)
{
    if (!pl || !h_in || !h_out) return fail(ARKCOS_INVALID_ARG, "NULL argument");
    if (pl->tables_only) return fail(ARKCOS_INVALID_ARG, "plan was created with arkcos_plan_create_tables_only");
    if (nmaps < 1 || nmaps > pl->max_nmaps) return fail(ARKCOS_INVALID_ARG, "nmaps must be in [1, max_nmaps]");
    const size_t full = (size_t)pl->max_nmaps * (size_t)pl->g.npix * elem_size(pl->dtype);
    const size_t bytes = (size_t)nmaps * (size_t)pl->g.npix * elem_size(pl->dtype);
    if (!pl->s_h2d) {
        for (int b = 0; b < 2; ++b) {
            CUDA_TRY(cudaMalloc(&pl->d_pipe_in[b], full));
            CUDA_TRY(cudaMalloc(&pl->d_pipe_out[b], full));
            CUDA_TRY(cudaEventCreateWithFlags(&pl->ev_h2d[b], cudaEventDisableTiming));
            CUDA_TRY(cudaEventCreateWithFlags(&pl->ev_comp[b], cudaEventDisableTiming));
            CUDA_TRY(cudaEventCreateWithFlags(&pl->ev_d2h[b], cudaEventDisableTiming));
        }
        CUDA_TRY(cudaStreamCreateWithFlags(&pl->s_comp, cudaStreamNonBlocking));
        CUDA_TRY(cudaStreamCreateWithFlags(&pl->s_d2h, cudaStreamNonBlocking));
        CUDA_TRY(cudaStreamCreateWithFlags(&pl->s_h2d, cudaStreamNonBlocking));
    }
    const int b = (int)(pl->pipe_calls & 1);
    const bool reuse = pl->pipe_calls >= 2;
    // upload into set b once the kernels of the call before last have read it
    if (reuse) CUDA_TRY(cudaStreamWaitEvent(pl->s_h2d, pl->ev_comp[b], 0));
    CUDA_TRY(cudaMemcpyAsync(pl->d_pipe_in[b], h_in, bytes, cudaMemcpyHostToDevice, pl->s_h2d));
    CUDA_TRY(cudaEventRecord(pl->ev_h2d[b], pl->s_h2d));
    // kernels: after the upload, and after the download of the call before last has read the output set
    CUDA_TRY(cudaStreamWaitEvent(pl->s_comp, pl->ev_h2d[b], 0));
    if (reuse) CUDA_TRY(cudaStreamWaitEvent(pl->s_comp, pl->ev_d2h[b], 0));
    if (int rc = arkcos_convolve(pl, pl->d_pipe_in[b], pl->d_pipe_out[b], nmaps, (void*)pl->s_comp)) return rc;
    CUDA_TRY(cudaEventRecord(pl->ev_comp[b], pl->s_comp));
    // download
    CUDA_TRY(cudaStreamWaitEvent(pl->s_d2h, pl->ev_comp[b], 0));
    CUDA_TRY(cudaMemcpyAsync(h_out, pl->d_pipe_out[b], bytes, cudaMemcpyDeviceToHost, pl->s_d2h));
    CUDA_TRY(cudaEventRecord(pl->ev_d2h[b], pl->s_d2h));
    ++pl->pipe_calls;
    return ARKCOS_OK;
}

int arkcos_plan_synchronize(const arkcos_plan* pl)
{
    if (!pl) return fail(ARKCOS_INVALID_ARG, "NULL plan");
    if (pl->s_h2d) {
        CUDA_TRY(cudaStreamSynchronize(pl->s_h2d));
        CUDA_TRY(cudaStreamSynchronize(pl->s_comp));
        CUDA_TRY(cudaStreamSynchronize(pl->s_d2h));
    }
    return ARKCOS_OK;
}

int arkcos_plan_destroy(arkcos_plan* pl)
{
    if (!pl) return ARKCOS_OK;
    for (const auto& e : pl->graphs) cudaGraphExecDestroy(e.exec);
    pl->graphs.clear();
    for (int b = 0; b < 2; ++b) {
        if (pl->d_pipe_in[b]) cudaFree(pl->d_pipe_in[b]);
        if (pl->d_pipe_out[b]) cudaFree(pl->d_pipe_out[b]);
        if (pl->ev_h2d[b]) cudaEventDestroy(pl->ev_h2d[b]);
        if (pl->ev_comp[b]) cudaEventDestroy(pl->ev_comp[b]);
        if (pl->ev_d2h[b]) cudaEventDestroy(pl->ev_d2h[b]);
    }
    for (cudaStream_t q : {pl->s_h2d, pl->s_comp, pl->s_d2h}) if (q) cudaStreamDestroy(q);
    void* ptrs[] = {pl->d_rings, pl->d_lens, pl->d_pairs, pl->d_north, pl->d_items[0], pl->d_items[1], pl->d_items[2], pl->d_items[3],
                    pl->d_items[4], pl->d_items[5], pl->d_eqchunks, pl->d_pole, pl->d_chirp, pl->d_phase, pl->d_fft_order[0], pl->d_fft_order[1], pl->d_table, pl->d_table2, pl->d_tw, pl->d_filt,
                    pl->d_W, pl->d_specIn, pl->d_specOut, pl->d_stage_in, pl->d_stage_out,
                    pl->d_cap_chunks, pl->d_cap_chunk_items, pl->d_tc_chunks, pl->d_tc_tiles, pl->d_tc_cols, pl->d_tc_rings, pl->d_tc_items[0], pl->d_tc_items[1], pl->d_tc_items[2], pl->d_goff, pl->d_G, pl->d_pole_scratch, pl->d_nyq, pl->d_direct_items, pl->d_tw3, pl->d_tw16, pl->d_fft3_d2[0], pl->d_fft3_d2[1], pl->d_fft3_b2[0], pl->d_fft3_b2[1], pl->d_wpair, pl->d_fft3_jobs[0][0], pl->d_fft3_jobs[0][1], pl->d_fft3_jobs[0][2], pl->d_fft3_jobs[0][3],
                    pl->d_fft3_jobs[1][0], pl->d_fft3_jobs[1][1], pl->d_fft3_jobs[1][2], pl->d_fft3_jobs[1][3]};
    for (void* p : ptrs) if (p) cudaFree(p);
    for (auto& e : pl->ev) if (e) cudaEventDestroy(e);
    for (auto& e : pl->ev_band) if (e) cudaEventDestroy(e);
    for (auto& d : pl->ev_fft) for (auto& e : d) if (e) cudaEventDestroy(e);
    if (pl->ev_fork) cudaEventDestroy(pl->ev_fork);
    for (auto& e : pl->ev_join) if (e) cudaEventDestroy(e);
    for (auto& q : pl->side) if (q) cudaStreamDestroy(q);
    if (pl->side_rows) cudaStreamDestroy(pl->side_rows);
    if (pl->ev_rows_fork) cudaEventDestroy(pl->ev_rows_fork);
    if (pl->ev_rows_done) cudaEventDestroy(pl->ev_rows_done);
    delete pl;
    return ARKCOS_OK;
}

int64_t arkcos_plan_npix(const arkcos_plan* pl) { return pl ? pl->g.npix : -1; }
int arkcos_plan_nrings(const arkcos_plan* pl) { return pl ? pl->g.R : -1; }
double arkcos_plan_ell_nyquist(const arkcos_plan* pl) { return pl ? pl->ell_nyquist : -1.0; }

int arkcos_plan_ring_info(const arkcos_plan* pl, int ring, double* theta, int* n, double* phi0, int64_t* offset,
                          int* band_lo, int* band_hi, int* mprime)
{
    if (!pl || ring < 0 || ring >= pl->g.R) return fail(ARKCOS_INVALID_ARG, "bad ring");
    const HostGeometry& g = pl->g;
    if (theta) *theta = g.theta[ring];
    if (n) *n = g.n[ring];
    if (phi0) *phi0 = g.phi0[ring];
    if (offset) *offset = g.pix_off[ring];
    if (band_lo) *band_lo = g.band_lo[ring];
    if (band_hi) *band_hi = g.band_hi[ring];
    if (mprime) *mprime = g.mprime[ring];
    return ARKCOS_OK;
}

int arkcos_plan_stats(const arkcos_plan* pl, int64_t* ring_pairs, int64_t* row_samples, double* mac_flops, double* fft_flops,
                      int64_t* workspace_bytes)
{
    if (!pl) return fail(ARKCOS_INVALID_ARG, "NULL plan");
    if (ring_pairs) *ring_pairs = pl->stats.ring_pairs;
    if (row_samples) *row_samples = pl->stats.row_samples;
    if (mac_flops) *mac_flops = pl->stats.mac_flops;
    if (fft_flops) *fft_flops = pl->stats.fft_flops;
    if (workspace_bytes) *workspace_bytes = pl->stats.workspace_bytes;
    return ARKCOS_OK;
}

int arkcos_plan_set_timing(const arkcos_plan* pl, int enable)
{
    if (!pl) return fail(ARKCOS_INVALID_ARG, "NULL plan");
    pl->timing = enable == 2 ? 2 : (enable ? 1 : 0);
    return ARKCOS_OK;
}

int arkcos_plan_get_timing(const arkcos_plan* pl, float* ms4)
{
    if (!pl || !ms4) return fail(ARKCOS_INVALID_ARG, "NULL argument");
    if (!pl->timing) return fail(ARKCOS_INVALID_ARG, "timing is not enabled");
    CUDA_TRY(cudaEventSynchronize(pl->ev[4]));
    for (int k = 0; k < 4; ++k) CUDA_TRY(cudaEventElapsedTime(&ms4[k], pl->ev[k], pl->ev[k + 1]));
    return ARKCOS_OK;
}

int arkcos_plan_band_kernels(const arkcos_plan* pl, int* n, const char** names, double* model_flops, float* last_ms)
{
    // launch names: the class-E and cap runs are band_mac_tc_kernel<KIND> when the plan uses the tensor cores
    static const char* kFp32[9] = {"band_mac_general_kernel", "band_mac_pole_kernel", "band_mac_eq_kernel",
                                   "band_mac_uniform_kernel<12,0>", "band_mac_uniform_kernel<20,0>",
                                   "band_mac_uniform_kernel<32,1>", "band_mac_uniform_kernel<12,1> + band_nyquist_eq_kernel", "band_mac_capchunk_kernel<4,20,0>",
                                   "band_mac_capchunk_kernel<4,20,1>"};
    if (!pl || !n) return fail(ARKCOS_INVALID_ARG, "NULL argument");
    const char* kNames[9];
    for (int k = 0; k < 9; ++k) kNames[k] = kFp32[k];
    if (pl->use_tc) {
        kNames[2] = pl->eq_alt ? "band_mac_tc_kernel<0>" : "band_mac_tc_kernel<1>";
        kNames[7] = "band_mac_tc_kernel<2>";
        kNames[8] = "band_mac_tc_kernel<3>";
    } else if (pl->d_G) {
        kNames[2] = "band_mac_eq_cached_kernel";
        kNames[7] = "band_mac_capchunk_cached_kernel<0>";
        kNames[8] = "band_mac_capchunk_cached_kernel<1>";
    }
    if (pl->npole > 0 && pl->pole_warp_per_mode) kNames[1] = "band_mac_pole_kernel + band_mac_pole_fold_kernel";
    *n = 9;
    for (int k = 0; k < 9; ++k) {
        if (names) names[k] = kNames[k];
        if (model_flops) model_flops[k] = pl->stats.band_flops[k];
    }
    if (last_ms) {
        if (pl->timing != 2) return fail(ARKCOS_INVALID_ARG, "per-kernel timing needs arkcos_plan_set_timing(plan, 2)");
        CUDA_TRY(cudaEventSynchronize(pl->ev_band[9]));
        for (int k = 0; k < 9; ++k) CUDA_TRY(cudaEventElapsedTime(&last_ms[k], pl->ev_band[k], pl->ev_band[k + 1]));
    }
    return ARKCOS_OK;
}

int arkcos_plan_fft_kernels(const arkcos_plan* pl, int* n, const char** names, double* pixels, float* last_ms_forward,
                            float* last_ms_inverse)
{
    static const char* kNames[9] = {"ring_fft3_direct1_kernel<12>", "ring_fft3_bluestein<12>", "ring_fft3_direct1_kernel<11>",
                                    "ring_fft3_bluestein<11>", "ring_fft3_direct1_kernel<10>", "ring_fft3_bluestein<10>",
                                    "ring_fft3_direct1_kernel<9>", "ring_fft3_bluestein<9>", "ring_fft_kernel (shared memory)"};
    if (!pl || !n) return fail(ARKCOS_INVALID_ARG, "NULL argument");
    *n = 9;
    for (int k = 0; k < 9; ++k) {
        if (names) names[k] = kNames[k];
        if (pixels) pixels[k] = pl->stats.fft_pixels[k];
    }
    if (last_ms_forward || last_ms_inverse) {
        if (pl->timing != 2) return fail(ARKCOS_INVALID_ARG, "per-kernel timing needs arkcos_plan_set_timing(plan, 2)");
        CUDA_TRY(cudaEventSynchronize(pl->ev_fft[1][9]));
        for (int k = 0; k < 9; ++k) {
            if (last_ms_forward) CUDA_TRY(cudaEventElapsedTime(&last_ms_forward[k], pl->ev_fft[0][k], pl->ev_fft[0][k + 1]));
            if (last_ms_inverse) CUDA_TRY(cudaEventElapsedTime(&last_ms_inverse[k], pl->ev_fft[1][k], pl->ev_fft[1][k + 1]));
        }
    }
    return ARKCOS_OK;
}

int arkcos_plan_work_model(const arkcos_plan* pl, double* band_pair_modes, double* fft_flops_min, double* tensor_flops,
                           int* memsets_per_map)
{
    if (!pl) return fail(ARKCOS_INVALID_ARG, "NULL plan");
    if (band_pair_modes) *band_pair_modes = pl->stats.mac_pairs_modes;
    if (fft_flops_min) *fft_flops_min = pl->stats.fft_flops_min;
    if (tensor_flops) *tensor_flops = pl->use_tc ? pl->stats.tc_flops : 0.0;
    if (memsets_per_map) *memsets_per_map = pl->ncapitems > 0 ? (int)pl->cap_zero.size() : 0;
    return ARKCOS_OK;
}

int arkcos_plan_tensor_cores(const arkcos_plan* pl, int blocks[3], int* resident_per_sm)
{
    if (!pl) return fail(ARKCOS_INVALID_ARG, "NULL plan");
    if (blocks) for (int c = 0; c < 3; ++c) blocks[c] = pl->use_tc ? pl->ntc_items[c] : 0;
    if (resident_per_sm) *resident_per_sm = pl->use_tc ? pl->tc_blocks_per_sm : 0;
    return pl->use_tc ? 1 : 0;
}

int arkcos_plan_launches_per_convolve(const arkcos_plan* pl)
{
    if (!pl) return -1;
    int n = (pl->opt.cache_kernel_rows || pl->npairs == 0) ? 0 : 1;
    for (int d = 0; d < 2; ++d) {
        n += (pl->nfft_old[d] > 0 ? 1 : 0) + (pl->nfft3_d2[d] > 0 ? 1 : 0) + (pl->nfft3_b2[d] > 0 ? 1 : 0);
        for (int c = 0; c < 4; ++c) n += (pl->nfft3_bluestein[d][c] > 0 ? 1 : 0) + (pl->nfft3[d][c] > pl->nfft3_bluestein[d][c] ? 1 : 0);
    }
    n += (pl->nitems[0] > 0) + (pl->pole_warp_per_mode ? 2 : 1) * (pl->npole > 0) + (pl->neqchunks > 0);
    for (int c = 1; c < kBandClasses; ++c) n += pl->nitems[c] > 0 ? 1 : 0;
    n += pl->ndirect > 0 ? 1 : 0;
    n += pl->nnyq > 0 ? 1 : 0;
    n += (pl->ncapsingle > 0 ? 1 : 0) + (pl->ncapitems > pl->ncapsingle ? 1 : 0);
    return n;
}

int arkcos_probe_fp32_peak(double* tflops, int repeats)
{
    if (!tflops || repeats < 1) return fail(ARKCOS_INVALID_ARG, "bad argument");
    int dev = 0, sms = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int blocks = sms * 8, threads = 256, iters = 1 << 15;
    float* d = nullptr;
    CUDA_TRY(cudaMalloc(&d, (size_t)blocks * threads * sizeof(float)));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    double best = 0.0;
    for (int r = 0; r < repeats + 1; ++r) {
        cudaEventRecord(e0);
        fma_chain_kernel<<<blocks, threads>>>(d, iters, 1.0000001f, 1e-9f);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms > 0) best = std::max(best, 2.0 * 8.0 * iters * (double)blocks * threads / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d);
    CUDA_TRY(cudaGetLastError());
    *tflops = best;
    return ARKCOS_OK;
}

const char* arkcos_strerror(int status)
{
    switch (status) {
        case ARKCOS_OK: return "success";
        case ARKCOS_INVALID_ARG: return "invalid argument";
        case ARKCOS_UNSUPPORTED: return "unsupported request";
        case ARKCOS_CUDA_ERROR: return "CUDA error";
        case ARKCOS_OUT_OF_MEMORY: return "out of memory";
        default: return "unknown status";
    }
}

const char* arkcos_last_error(void) { return g_last_error.c_str(); }

}  // extern "C"
