// host_eig.cu -- the projected eigenproblem of the Davidson loop (risp_tda_solve) on the host.
//
// The subspace matrix G = V^T A V is at most a few hundred rows, and an iteration needs only its lowest n_roots eigenpairs.
#include "ctx.h"
#include <algorithm>
#include <cmath>

// The nv lowest eigenpairs only (what a Davidson iteration needs; a full QL accumulation of all vectors costs ~9 n^3 flops, 90 ms
// at n = 315, once per iteration): Householder tridiagonalisation with the reflectors kept, eigenvalues by QL without vectors,
// eigenvectors of T by inverse iteration (pivoted tridiagonal LU, re-orthogonalised against the vectors already found, as
// LAPACK's dstein does for clusters), back-transformed through the reflectors.  z[i*n + j], j < nv; w has all n eigenvalues.
void risp_sym_eig_lowest(std::vector<double> &a, int n, int nv, std::vector<double> &w, std::vector<double> &z)
{
    nv = std::min(nv, n);
    std::vector<double> vs((size_t)n * n, 0.0), betas(n, 0.0), v(n), p(n), d(n), e(n, 0.0);
    for (int k = 0; k + 2 < n; ++k) {
        int len = n - k - 1;
        double nrm = 0.0;
        for (int i = 0; i < len; ++i) { v[i] = a[(size_t)(k + 1 + i) * n + k]; nrm += v[i] * v[i]; }
        nrm = std::sqrt(nrm);
        double tail = 0.0;
        for (int i = 1; i < len; ++i) tail += v[i] * v[i];
        if (tail == 0.0) continue;
        double alpha = v[0] > 0 ? -nrm : nrm;
        v[0] -= alpha;
        double vv = 0.0;
        for (int i = 0; i < len; ++i) vv += v[i] * v[i];
        double beta = 2.0 / vv;
        for (int i = 0; i < len; ++i) {
            double s = 0.0;
            const double *row = &a[(size_t)(k + 1 + i) * n + k + 1];
            for (int j = 0; j < len; ++j) s += row[j] * v[j];
            p[i] = beta * s;
        }
        double K = 0.0;
        for (int i = 0; i < len; ++i) K += v[i] * p[i];
        K *= 0.5 * beta;
        for (int i = 0; i < len; ++i) p[i] -= K * v[i];
        for (int i = 0; i < len; ++i) {
            double *row = &a[(size_t)(k + 1 + i) * n + k + 1];
            const double vi = v[i], pi = p[i];
            for (int j = 0; j < len; ++j) row[j] -= vi * p[j] + pi * v[j];
        }
        a[(size_t)(k + 1) * n + k] = a[(size_t)k * n + k + 1] = alpha;
        for (int i = 1; i < len; ++i) a[(size_t)(k + 1 + i) * n + k] = a[(size_t)k * n + k + 1 + i] = 0.0;
        betas[k] = beta;
        std::copy(v.begin(), v.begin() + len, vs.begin() + (size_t)k * n);
    }
    for (int i = 0; i < n; ++i) d[i] = a[(size_t)i * n + i];
    for (int i = 0; i + 1 < n; ++i) e[i] = a[(size_t)(i + 1) * n + i];
    const std::vector<double> d0 = d, e0 = e;          // T, kept for the inverse iteration
    for (int l = 0; l < n; ++l) {                       // QL, eigenvalues only
        int iter = 0, m;
        do {
            for (m = l; m < n - 1; ++m) {
                double dd = std::fabs(d[m]) + std::fabs(d[m + 1]);
                if (std::fabs(e[m]) <= 2.3e-16 * dd) break;
            }
            if (m != l) {
                if (++iter > 200) break;
                double g = (d[l + 1] - d[l]) / (2.0 * e[l]);
                double r = std::hypot(g, 1.0);
                g = d[m] - d[l] + e[l] / (g + (g >= 0 ? std::fabs(r) : -std::fabs(r)));
                double s = 1.0, c = 1.0, pp = 0.0;
                int i;
                for (i = m - 1; i >= l; --i) {
                    double f = s * e[i], b = c * e[i];
                    e[i + 1] = r = std::hypot(f, g);
                    if (r == 0.0) { d[i + 1] -= pp; e[m] = 0.0; break; }
                    s = f / r; c = g / r;
                    g = d[i + 1] - pp;
                    r = (d[i] - g) * s + 2.0 * c * b;
                    pp = s * r;
                    d[i + 1] = g + pp;
                    g = c * r - b;
                }
                if (r == 0.0 && i >= l) continue;
                d[l] -= pp; e[l] = g; e[m] = 0.0;
            }
        } while (m != l);
    }
    w = d;
    std::sort(w.begin(), w.end());
    double tnorm = 0.0;
    for (int i = 0; i < n; ++i) tnorm = std::max(tnorm, std::fabs(d0[i]) + (i ? std::fabs(e0[i - 1]) : 0.0) + (i + 1 < n ? std::fabs(e0[i]) : 0.0));
    const double eps = 2.2e-16, tiny = std::max(tnorm, 1e-300) * eps;
    z.assign((size_t)n * n, 0.0);
    std::vector<double> X((size_t)nv * n), dl(n), dd(n), du(n), du2(n), x(n);
    std::vector<char> piv(n);
    double lam_prev = 0.0;
    for (int j = 0; j < nv; ++j) {
        double lam = w[j];
        if (j > 0 && lam - lam_prev < 10.0 * tiny) lam = lam_prev + 10.0 * tiny;   // separate numerically equal eigenvalues
        lam_prev = lam;
        // LU of T - lam I with partial pivoting (dgttrf)
        for (int i = 0; i < n; ++i) { dd[i] = d0[i] - lam; dl[i] = du[i] = (i + 1 < n) ? e0[i] : 0.0; du2[i] = 0.0; piv[i] = 0; }
        for (int i = 0; i + 1 < n; ++i) {
            if (std::fabs(dd[i]) >= std::fabs(dl[i])) {
                if (dd[i] == 0.0) dd[i] = tiny;
                const double f = dl[i] / dd[i];
                dl[i] = f; dd[i + 1] -= f * du[i];
            } else {
                const double f = dd[i] / dl[i];
                dd[i] = dl[i]; dl[i] = f;
                const double t = du[i];
                du[i] = dd[i + 1]; dd[i + 1] = t - f * dd[i + 1];
                if (i + 2 < n) { du2[i] = du[i + 1]; du[i + 1] = -f * du[i + 1]; }
                piv[i] = 1;
            }
        }
        if (std::fabs(dd[n - 1]) < tiny) dd[n - 1] = tiny;
        for (int i = 0; i < n - 1; ++i) if (std::fabs(dd[i]) < tiny * 1e-3) dd[i] = tiny;
        unsigned long long seed = 0x9E3779B97F4A7C15ull * (unsigned long long)(j + 1);
        for (int i = 0; i < n; ++i) { seed = seed * 6364136223846793005ull + 1442695040888963407ull; x[i] = ((double)(seed >> 11) / 9007199254740992.0) - 0.5; }
        double *xj = &X[(size_t)j * n];
        for (int it = 0; it < 5; ++it) {
            for (int i = 0; i + 1 < n; ++i) {
                if (!piv[i]) x[i + 1] -= dl[i] * x[i];
                else { const double t = x[i]; x[i] = x[i + 1]; x[i + 1] = t - dl[i] * x[i]; }
            }
            x[n - 1] /= dd[n - 1];
            if (n > 1) x[n - 2] = (x[n - 2] - du[n - 2] * x[n - 1]) / dd[n - 2];
            for (int i = n - 3; i >= 0; --i) x[i] = (x[i] - du[i] * x[i + 1] - du2[i] * x[i + 2]) / dd[i];
            for (int rep = 0; rep < 2; ++rep)
                for (int q = 0; q < j; ++q) {
                    if (w[j] - w[q] > 1e-3 * std::max(tnorm, 1e-300)) continue;      // well separated: orthogonal by themselves
                    const double *xq = &X[(size_t)q * n];
                    double dot = 0.0;
                    for (int i = 0; i < n; ++i) dot += xq[i] * x[i];
                    for (int i = 0; i < n; ++i) x[i] -= dot * xq[i];
                }
            double nr = 0.0;
            for (int i = 0; i < n; ++i) nr += x[i] * x[i];
            nr = 1.0 / std::sqrt(std::max(nr, 1e-300));
            for (int i = 0; i < n; ++i) x[i] *= nr;
        }
        std::copy(x.begin(), x.end(), xj);
        // back-transform: y = H_0 H_1 ... H_{n-3} x
        for (int k = n - 3; k >= 0; --k) {
            if (betas[k] == 0.0) continue;
            const int len = n - k - 1;
            const double *vk = &vs[(size_t)k * n];
            double dot = 0.0;
            for (int i = 0; i < len; ++i) dot += vk[i] * x[k + 1 + i];
            dot *= betas[k];
            for (int i = 0; i < len; ++i) x[k + 1 + i] -= dot * vk[i];
        }
        for (int i = 0; i < n; ++i) z[(size_t)i * n + j] = x[i];
    }
}

// Debug export (include/risp_debug.h): the eigen solver above, pinned against LAPACK in tests/test_host_logic.py.
extern "C" int risp_debug_sym_eig_lowest(int n, int nv, const double *a_in, double *w_out, double *z_out)
{
    if (n <= 0 || nv <= 0 || !a_in || !w_out || !z_out) return RISP_EINVAL;
    std::vector<double> a(a_in, a_in + (size_t)n * n), w, z;
    risp_sym_eig_lowest(a, n, nv, w, z);
    std::memcpy(w_out, w.data(), (size_t)n * 8);
    std::memcpy(z_out, z.data(), (size_t)n * n * 8);
    return RISP_OK;
}
