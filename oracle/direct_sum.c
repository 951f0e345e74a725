/* Oracle #1: brute-force direct sum (fp64).  TEST INFRASTRUCTURE ONLY -- see oracle/__init__.py.
 *
 *   out(p) = sum_{q : gamma_pq < theta_max}  K(gamma_pq) * in(q) * Omega_q
 *
 * This is Eq. 6 of the paper, "s_p = sum_q K(p.q) r_q", with
 *   - the quadrature weight of the input pixel put in, as PAPER.md:99 allows ("the same quadrature
 *     weights can be used in Equation (6)") and BASELINE.json's configs state (Omega_q),
 *   - the compact support of PAPER.md:83 read as the strict inequality gamma < theta_max,
 *   - K(gamma) interpolated linearly from a table over [0, theta_max] ("interpolating it
 *     in O(1) operations from ... precomputed values"; BASELINE.json configs[0] "tabulated on 65536
 *     points over [0, theta_max] with linear interpolation").
 *
 * The angular distance is evaluated in the cancellation-free form of Eq. 9:
 *   x = 2 - 2 cos(gamma) = 4 sin^2((theta_p-theta_q)/2) + 4 sin(theta_p) sin(theta_q) sin^2(dphi/2),
 *   gamma = 2 asin(sqrt(x)/2).
 * (The right-hand side of Eq. 9 equals 2 - 2 cos(alpha) identically; SURVEY.md section 8c reading 3.)
 *
 * Pruning (does not change the result, every pixel pair that survives is still tested with
 * gamma < theta_max): only rings with |theta_i - theta_j| < theta_max, and on such a ring only the
 * phi window that can lie inside the cap, padded by two pixels.
 *
 * No blocking, no ring symmetries, no caching of weights: one K evaluation per pixel pair.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static double kernel_lerp(const double* table, int ntab, double theta_max, double gamma)
{
    /* table[t] = K(t * theta_max / (ntab-1)), t = 0 .. ntab-1 */
    double u = gamma * (double)(ntab - 1) / theta_max;
    long t = (long)floor(u);
    if (t < 0) t = 0;
    if (t > ntab - 2) t = ntab - 2;
    double f = u - (double)t;
    return table[t] + f * (table[t + 1] - table[t]);
}

/* Returns the number of threads used (>= 1), or a negative value on a bad argument.
 *
 * theta, n, phi0, omega : [R]       ring tables (see oracle/geometry.py)
 * offset                : [R+1]     first pixel of each ring
 * table, ntab, theta_max            radial profile
 * in                    : [nmaps][npix]
 * out_rings             : [n_out]   output rings to evaluate
 * out                   : [nmaps][sum_k n[out_rings[k]]]   rings concatenated in the order given
 * nthreads              : <= 0 means "all" (OpenMP default)
 */
int arkcos_oracle_direct_sum(int R, const double* theta, const int64_t* n, const double* phi0,
                             const double* omega, const int64_t* offset,
                             const double* table, int ntab, double theta_max,
                             const double* in, int nmaps, int64_t npix,
                             const int32_t* out_rings, int n_out, double* out, int nthreads)
{
    if (R <= 0 || ntab < 2 || !(theta_max > 0.0) || nmaps <= 0 || n_out < 0) return -1;
    const double two_pi = 6.283185307179586476925286766559;

    int64_t* out_off = (int64_t*)malloc(sizeof(int64_t) * (size_t)(n_out + 1));
    if (!out_off) return -2;
    out_off[0] = 0;
    for (int k = 0; k < n_out; ++k) {
        if (out_rings[k] < 0 || out_rings[k] >= R) { free(out_off); return -1; }
        out_off[k + 1] = out_off[k] + n[out_rings[k]];
    }
    const int64_t nout_pix = out_off[n_out];
    int used = 1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
    used = omp_get_max_threads();
#endif
    const double sh = sin(0.5 * theta_max);
    const double xmax = 4.0 * sh * sh;       /* squared chord of the support radius (pruning only) */

#pragma omp parallel for schedule(dynamic, 1)
    for (int kk = 0; kk < n_out; ++kk) {
        const int i = out_rings[kk];
        const double ti = theta[i], si = sin(ti);
        double* acc = (double*)malloc(sizeof(double) * (size_t)nmaps);
        for (int64_t k = 0; k < n[i]; ++k) {
            const double phip = phi0[i] + two_pi * (double)k / (double)n[i];
            for (int m = 0; m < nmaps; ++m) acc[m] = 0.0;
            for (int j = 0; j < R; ++j) {
                const double dt = ti - theta[j];
                if (!(fabs(dt) < theta_max)) continue;
                const double sd = sin(0.5 * dt);
                const double A = 4.0 * sd * sd;
                const double B = 4.0 * si * sin(theta[j]);
                const int64_t nj = n[j];
                /* phi window: x < xmax  <=>  sin^2(dphi/2) < (xmax - A)/B */
                int64_t l_lo = 0, l_cnt = nj;
                if (B > 0.0) {
                    double ratio = (xmax - A) / B;
                    if (ratio < 0.0) ratio = 0.0;
                    if (ratio < 1.0) {
                        const double dphimax = 2.0 * asin(sqrt(ratio));
                        const double step = two_pi / (double)nj;
                        const double c = (phip - phi0[j]) / step;      /* fractional pixel position */
                        const double hw = dphimax / step + 2.0;         /* half width + padding */
                        if (2.0 * hw + 4.0 < (double)nj) {   /* else: the whole ring, each pixel once */
                            l_lo = (int64_t)floor(c - hw);
                            l_cnt = (int64_t)ceil(c + hw) - l_lo + 1;
                        }
                    }
                }
                for (int64_t ll = 0; ll < l_cnt; ++ll) {
                    int64_t l = (l_lo + ll) % nj;
                    if (l < 0) l += nj;
                    const double phiq = phi0[j] + two_pi * (double)l / (double)nj;
                    const double s2 = sin(0.5 * (phip - phiq));
                    const double x = A + B * s2 * s2;
                    double hx = 0.5 * sqrt(x);
                    if (hx > 1.0) hx = 1.0;
                    const double gamma = 2.0 * asin(hx);
                    if (gamma < theta_max) {
                        const double w = kernel_lerp(table, ntab, theta_max, gamma) * omega[j];
                        const int64_t q = offset[j] + l;
                        for (int m = 0; m < nmaps; ++m) acc[m] += w * in[(int64_t)m * npix + q];
                    }
                }
            }
            for (int m = 0; m < nmaps; ++m) out[(int64_t)m * nout_pix + out_off[kk] + k] = acc[m];
        }
        free(acc);
    }
    free(out_off);
    return used;
}
