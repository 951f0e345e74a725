// Plan-time tools around Eq. 7: Legendre transform of a tabulated radial profile (Eq. 2),
// the mean quadratic error of cutting the profile at an angular distance alpha_cut, and choosers built on it (the smallest
// cut, and the azimuthal wavenumber the kernel-row grid of a polar-cap ring has to resolve).  Host code, no CUDA.
//
// The profile between table nodes is the linear interpolant the convolution itself uses, so every table
// interval is integrated on its own (the integrand is smooth there): Gauss-Legendre panels no longer than a fraction of
// the oscillation length pi / lmax of P_lmax, P_l(cos theta) at all quadrature nodes advanced together by the three-term
// recurrence  (l+1) P_{l+1} = (2l+1) z P_l - l P_{l-1}.
#include <math.h>

#include <algorithm>
#include <string>
#include <vector>

#include "../../include/arkcos.h"

namespace arkcos {
int set_last_error(int code, const std::string& msg);      // arkcos_host.cu
}

namespace {

const double kPi = 3.14159265358979323846264338327950288;

// nodes x_k in (-1, 1) and weights of the q-point Gauss-Legendre rule: Newton iteration on P_q
void gauss_legendre(int q, std::vector<double>& x, std::vector<double>& w)
{
    x.resize(q);
    w.resize(q);
    for (int k = 0; k < q; ++k) {
        double z = cos(kPi * (k + 0.75) / (q + 0.5));
        double dp = 1.0;
        for (int it = 0; it < 100; ++it) {
            double p0 = 1.0, p1 = z;
            for (int l = 1; l < q; ++l) {
                const double p2 = ((2 * l + 1) * z * p1 - l * p0) / (l + 1);
                p0 = p1;
                p1 = p2;
            }
            dp = q * (z * p1 - p0) / (z * z - 1.0);
            const double dz = p1 / dp;
            z -= dz;
            if (fabs(dz) < 1e-16) break;
        }
        x[k] = z;
        w[k] = 2.0 / ((1.0 - z * z) * dp * dp);
    }
}

struct Quadrature {
    std::vector<double> z, f;         // cos(theta_k) and K(theta_k) sin(theta_k) weight_k 2 pi of every node
    std::vector<int> cell_begin;      // nodes of cell c: cell_begin[c] .. cell_begin[c+1]
};

// Nodes for the profile restricted to the cells [edges[c], edges[c+1]) (edges ascending, inside [0, theta_max]).
void build_nodes(const arkcos_kernel& kr, const std::vector<double>& edges, int lmax, Quadrature& Q)
{
    const int n = kr.n;
    const double h = kr.theta_max / (n - 1);
    const double osc = kPi / (lmax + 1.0);
    std::vector<double> x3, w3, x8, w8;
    gauss_legendre(3, x3, w3);
    gauss_legendre(8, x8, w8);
    Q.cell_begin.assign(1, 0);
    for (size_t c = 0; c + 1 < edges.size(); ++c) {
        const double lo = edges[c], hi = edges[c + 1];
        if (hi > lo) {
            int t0 = std::min(std::max((int)floor(lo / h), 0), n - 2);
            for (int t = t0; t <= n - 2 && t * h < hi; ++t) {
                const double a = std::max(lo, t * h), b = std::min(hi, (t + 1) * h);
                if (!(b > a)) continue;
                const double k0 = kr.table[t], k1 = kr.table[t + 1];
                // panels of at most a quarter of the oscillation length; a panel tiny against it needs three nodes only
                const int np = std::max(1, (int)ceil((b - a) / (0.25 * osc)));
                const bool tiny = (b - a) < 0.02 * osc;
                const std::vector<double>&x = tiny ? x3 : x8, &w = tiny ? w3 : w8;
                for (int p = 0; p < np; ++p) {
                    const double pa = a + (b - a) * p / np, pb = a + (b - a) * (p + 1) / np;
                    for (size_t k = 0; k < x.size(); ++k) {
                        const double th = 0.5 * (pa + pb) + 0.5 * (pb - pa) * x[k];
                        const double u = th / h - t;
                        Q.z.push_back(cos(th));
                        Q.f.push_back(2.0 * kPi * (k0 + u * (k1 - k0)) * sin(th) * 0.5 * (pb - pa) * w[k]);
                    }
                }
            }
        }
        Q.cell_begin.push_back((int)Q.z.size());
    }
}

// out[c * (lmax + 1) + l] = sum over the nodes of cell c of f P_l(z); the nodes are advanced through all l in blocks
// that stay in the first-level cache
void legendre_cells(const Quadrature& Q, int lmax, std::vector<double>& out)
{
    const int ncell = (int)Q.cell_begin.size() - 1;
    out.assign((size_t)ncell * (lmax + 1), 0.0);
    constexpr int kBlock = 512;
    double p0[kBlock], p1[kBlock], p2[kBlock];
    for (int c = 0; c < ncell; ++c) {
        double* __restrict__ o = out.data() + (size_t)c * (lmax + 1);
        for (int k0 = Q.cell_begin[c]; k0 < Q.cell_begin[c + 1]; k0 += kBlock) {
            const int nb = std::min(kBlock, Q.cell_begin[c + 1] - k0);
            const double* __restrict__ z = Q.z.data() + k0;
            const double* __restrict__ f = Q.f.data() + k0;
            double a0 = 0.0, a1 = 0.0;
            for (int k = 0; k < nb; ++k) {
                p0[k] = 1.0;
                p1[k] = z[k];
                a0 += f[k];
                a1 += f[k] * z[k];
            }
            o[0] += a0;
            if (lmax >= 1) o[1] += a1;
            double *q0 = p0, *q1 = p1, *q2 = p2;
            for (int l = 1; l < lmax; ++l) {
                const double a = (2.0 * l + 1.0) / (l + 1.0), b = (double)l / (l + 1.0);
                double acc = 0.0;
                for (int k = 0; k < nb; ++k) {
                    q2[k] = a * z[k] * q1[k] - b * q0[k];
                    acc += f[k] * q2[k];
                }
                o[l + 1] += acc;
                double* t = q0;
                q0 = q1;
                q1 = q2;
                q2 = t;
            }
        }
    }
}

int check_kernel(const arkcos_kernel* k)
{
    if (!k || !k->table) return arkcos::set_last_error(ARKCOS_INVALID_ARG, "NULL kernel");
    if (k->n < 2 || !(k->theta_max > 0.0) || !(k->theta_max <= kPi + 1e-12))
        return arkcos::set_last_error(ARKCOS_INVALID_ARG, "kernel: need n >= 2 and 0 < theta_max <= pi");
    return 0;
}

double eq7_sum(const double* dk, const double* c_ell, int lmax)
{
    double s = 0.0;
    for (int l = 0; l <= lmax; ++l) s += (2.0 * l + 1.0) / (4.0 * kPi) * dk[l] * dk[l] * c_ell[l];
    return s;
}

}  // namespace

extern "C" {

int arkcos_kernel_legendre(const arkcos_kernel* kernel, double theta_lo, double theta_hi, int lmax, double* k_ell)
{
    if (int rc = check_kernel(kernel)) return rc;
    if (!k_ell || lmax < 0 || lmax > (1 << 16)) return arkcos::set_last_error(ARKCOS_INVALID_ARG, "need k_ell and 0 <= lmax <= 65536");
    if (!(theta_lo >= 0.0) || !(theta_hi <= kernel->theta_max * (1 + 1e-15)) || theta_hi < theta_lo)
        return arkcos::set_last_error(ARKCOS_INVALID_ARG, "need 0 <= theta_lo <= theta_hi <= theta_max");
    Quadrature Q;
    build_nodes(*kernel, {theta_lo, std::min(theta_hi, kernel->theta_max)}, lmax, Q);
    std::vector<double> out;
    legendre_cells(Q, lmax, out);
    std::copy(out.begin(), out.begin() + lmax + 1, k_ell);
    return ARKCOS_OK;
}

int arkcos_kernel_truncation_error(const arkcos_kernel* kernel, double theta_cut, const double* c_ell, int lmax, double* sigma2,
                                   double* signal2)
{
    if (int rc = check_kernel(kernel)) return rc;
    if (!c_ell || lmax < 0 || lmax > (1 << 16)) return arkcos::set_last_error(ARKCOS_INVALID_ARG, "need c_ell and 0 <= lmax <= 65536");
    if (!(theta_cut >= 0.0)) return arkcos::set_last_error(ARKCOS_INVALID_ARG, "theta_cut must be >= 0");
    const double cut = std::min(theta_cut, kernel->theta_max);
    Quadrature Q;
    build_nodes(*kernel, {0.0, cut, kernel->theta_max}, lmax, Q);
    std::vector<double> cells;
    legendre_cells(Q, lmax, cells);
    const double* inner = cells.data();
    const double* outer = cells.data() + (lmax + 1);
    if (sigma2) *sigma2 = eq7_sum(outer, c_ell, lmax);
    if (signal2) {
        std::vector<double> whole(lmax + 1);
        for (int l = 0; l <= lmax; ++l) whole[l] = inner[l] + outer[l];
        *signal2 = eq7_sum(whole.data(), c_ell, lmax);
    }
    return ARKCOS_OK;
}

int arkcos_kernel_choose_cut(const arkcos_kernel* kernel, const double* c_ell, int lmax, double rel_tol, int ngrid, double* theta_cut,
                             double* sigma2, double* signal2)
{
    if (int rc = check_kernel(kernel)) return rc;
    if (!c_ell || lmax < 0 || lmax > (1 << 16)) return arkcos::set_last_error(ARKCOS_INVALID_ARG, "need c_ell and 0 <= lmax <= 65536");
    if (!(rel_tol >= 0.0) || ngrid < 1 || ngrid > 4096 || !theta_cut)
        return arkcos::set_last_error(ARKCOS_INVALID_ARG, "need rel_tol >= 0, 1 <= ngrid <= 4096, theta_cut");
    std::vector<double> edges(ngrid + 1);
    for (int g = 0; g <= ngrid; ++g) edges[g] = kernel->theta_max * g / ngrid;
    Quadrature Q;
    build_nodes(*kernel, edges, lmax, Q);
    std::vector<double> cells;
    legendre_cells(Q, lmax, cells);
    std::vector<double> tail(lmax + 1, 0.0), whole(lmax + 1, 0.0);
    for (int g = 0; g < ngrid; ++g)
        for (int l = 0; l <= lmax; ++l) whole[l] += cells[(size_t)g * (lmax + 1) + l];
    const double sig = eq7_sum(whole.data(), c_ell, lmax);
    // from the outside in: the cut moves to edges[g] as long as the error of dropping [edges[g], theta_max) stays below the bound
    int best = ngrid;
    double best_s2 = 0.0;
    for (int g = ngrid - 1; g >= 0; --g) {
        for (int l = 0; l <= lmax; ++l) tail[l] += cells[(size_t)g * (lmax + 1) + l];
        const double s2 = eq7_sum(tail.data(), c_ell, lmax);
        if (!(s2 <= rel_tol * rel_tol * sig)) break;
        best = g;
        best_s2 = s2;
    }
    *theta_cut = edges[best];
    if (sigma2) *sigma2 = best_s2;
    if (signal2) *signal2 = sig;
    return ARKCOS_OK;
}

int arkcos_kernel_choose_ell_nyquist(const arkcos_kernel* kernel, const double* c_ell, int lmax, double rel_tol, double* ell_nyquist)
{
    if (int rc = check_kernel(kernel)) return rc;
    if (!c_ell || lmax < 0 || lmax > (1 << 16) || !(rel_tol >= 0.0) || !ell_nyquist)
        return arkcos::set_last_error(ARKCOS_INVALID_ARG, "need c_ell, 0 <= lmax <= 65536, rel_tol >= 0, ell_nyquist");
    Quadrature Q;
    build_nodes(*kernel, {0.0, kernel->theta_max}, lmax, Q);
    std::vector<double> kl;
    legendre_cells(Q, lmax, kl);
    const double sig = eq7_sum(kl.data(), c_ell, lmax);
    double tail = 0.0;
    int l = lmax;
    for (; l > 0; --l) {
        tail += (2.0 * l + 1.0) / (4.0 * kPi) * kl[l] * kl[l] * c_ell[l];
        if (!(tail <= rel_tol * rel_tol * sig)) break;
    }
    *ell_nyquist = (double)l;
    return ARKCOS_OK;
}

}  // extern "C"
