// solve_tddft.cu -- risp_tddft_solve: lowest excitation energies of full TDDFT-risp, the symplectic problem of Eq. 1
// (PAPER.md:47-58), by a Davidson-like iteration in which "both (A+B) and (A-B) are projected into the subspace"
// (PAPER.md:213-215).
//
// One orthonormal basis b spans the trial space of |X+Y> and |X-Y> (reading G26: the paper mentions "the corresponding expansion
// basis of X+Y and X-Y"; a common basis is the standard form of that scheme).  With P = (A+B) b, Q = (A-B) b and the projected
// matrices M+ = b^T P, M- = b^T Q (M- positive definite for a stable reference), Eq. 1 reduces to the symmetric problem
//     C^T M+ C z = Omega^2 z,   M- = C C^T (Cholesky),   |X+Y> = b C z / sqrt(Omega),   |X-Y> = b M+ (C z) / Omega^(3/2),
// normalised to <X+Y|X-Y> = 1, i.e. X^T X - Y^T Y = 1.  Residuals r1 = (A+B)|X+Y> - Omega |X-Y>, r2 = (A-B)|X-Y> - Omega |X+Y>; both are
// preconditioned with (Omega - Delta)^-1, orthonormalised against b and appended (up to two vectors per unconverged root), at the
// price of ONE risp_matvec_tddft per new vector (it returns both products).  The subspace is device resident (this solver is for
// systems whose T_ia^P' tensor fits in HBM anyway); when it is full the iteration restarts from the orthonormalised {X+Y, X-Y}.
#include "ctx.h"
#include <algorithm>
#include <chrono>
#include <cmath>

void risp_sym_eig_lowest(std::vector<double> &a, int n, int nv, std::vector<double> &w, std::vector<double> &z);   // host_eig.cu

namespace {

__global__ void td_unit_kernel(double *__restrict__ V, long long dim, const long long *__restrict__ idx)
{
    const int j = blockIdx.y;
    const long long hot = idx[j];
    for (long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x; x < dim; x += (long long)gridDim.x * blockDim.x) V[j * dim + x] = x == hot ? 1.0 : 0.0;
}

// t = r / (omega - (eps_a - eps_i)), |denominator| floored at 1e-8; r and t may be the same vector
__global__ void td_precondition_kernel(const double *r, double omega, const double *__restrict__ eps, int nocc, int nvir, double *t)
{
    const double *ev = eps + nocc;
    for (long long i = blockIdx.x; i < nocc; i += gridDim.x) {
        const double ei = eps[i];
        for (int a = threadIdx.x; a < nvir; a += blockDim.x) {
            double den = omega - (ev[a] - ei);
            if (fabs(den) < 1e-8) den = den < 0 ? -1e-8 : 1e-8;
            t[i * nvir + a] = r[i * nvir + a] / den;
        }
    }
}

__global__ void td_scale_rows_kernel(double *__restrict__ T, long long dim, const double *__restrict__ scale)
{
    const int j = blockIdx.y;
    const double s = scale[j];
    for (long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x; x < dim; x += (long long)gridDim.x * blockDim.x) T[j * dim + x] *= s;
}

inline unsigned sgrid(long long n) { return (unsigned)std::min<long long>((n + 255) / 256, 148 * 8); }

struct TdSolver {
    risp_ctx *ctx = nullptr;
    long long dim = 0, slice = 16384;
    int kcap = 0, k = 0;
    double *b = nullptr, *P = nullptr, *Q = nullptr, *T = nullptr, *tmp = nullptr;
    double *dPart = nullptr, *dSmall = nullptr, *dCoef = nullptr, *dScale = nullptr;
    long long *dIdx = nullptr;
    cudaStream_t st = 0;
    DevScratch scr;
    int gram(const double *A, int na, const double *B, int nb, std::vector<double> &out) { return risp_rows_gram(ctx, A, na, B, nb, dim, slice, dPart, dSmall, out, st); }
    int lincomb(const std::vector<double> &coef, int nc, int na, const double *A, double *C, double alpha, double beta)
    {
        // na may exceed the 128-row K tile budget of nothing here: K = na is the contraction length of one GEMM, any size works
        return risp_rows_lincomb(ctx, coef.data(), nc, na, A, C, dim, alpha, beta, dCoef, st);
    }
};

// lower Cholesky factor of the n x n matrix g (ld n) with a relative pivot threshold; ok[j] = 0 marks dropped rows.  Returns L (dropped
// rows / columns are unit vectors so that the triangular solves stay defined).
void host_cholesky(const std::vector<double> &g, int n, double thresh, std::vector<double> &L, std::vector<char> &ok)
{
    L.assign((size_t)n * n, 0.0); ok.assign(n, 1);
    for (int j = 0; j < n; ++j) {
        for (int i = j; i < n; ++i) {
            double s = g[(size_t)i * n + j];
            for (int c = 0; c < j; ++c) s -= L[(size_t)i * n + c] * L[(size_t)j * n + c];
            if (i == j) {
                if (!(s > thresh)) { ok[j] = 0; L[(size_t)j * n + j] = 1.0; break; }
                L[(size_t)j * n + j] = std::sqrt(s);
            } else L[(size_t)i * n + j] = ok[j] ? s / L[(size_t)j * n + j] : 0.0;
        }
        if (!ok[j]) for (int i = 0; i < n; ++i) if (i != j) L[(size_t)i * n + j] = 0.0;
    }
}
void host_lower_inverse(const std::vector<double> &L, int n, std::vector<double> &Li)
{
    Li.assign((size_t)n * n, 0.0);
    for (int c = 0; c < n; ++c) {
        Li[(size_t)c * n + c] = 1.0 / L[(size_t)c * n + c];
        for (int i = c + 1; i < n; ++i) {
            double s = 0.0;
            for (int q = c; q < i; ++q) s += L[(size_t)i * n + q] * Li[(size_t)q * n + c];
            Li[(size_t)i * n + c] = -s / L[(size_t)i * n + i];
        }
    }
}

// orthonormalise the nb vectors in T against b[0, k) and among themselves; result back in T, dependent vectors dropped
int td_orthonormalise(TdSolver &S, double *T, double *tmp, int &nb)
{
    risp_ctx *ctx = S.ctx;
    int rc;
    std::vector<double> g;
    {
        if ((rc = S.gram(T, nb, T, nb, g))) return rc;
        std::vector<double> sc(nb);
        for (int j = 0; j < nb; ++j) { const double n2 = g[(size_t)j * nb + j]; sc[j] = n2 > 0 ? 1.0 / std::sqrt(n2) : 0.0; }
        RISP_CUDA_TRY(cudaMemcpyAsync(S.dScale, sc.data(), (size_t)nb * 8, cudaMemcpyHostToDevice, S.st));
        td_scale_rows_kernel<<<dim3(sgrid(S.dim), nb), 256, 0, S.st>>>(T, S.dim, S.dScale);
        RISP_CUDA_TRY(cudaGetLastError());
        RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
    }
    for (int first = 0; first < S.k; first += 128) {
        const int cnt = std::min(128, S.k - first);
        const double *Vc = S.b + (long long)first * S.dim;
        for (int rep = 0; rep < 2; ++rep) {
            std::vector<double> c;
            if ((rc = S.gram(T, nb, Vc, cnt, c))) return rc;
            if ((rc = S.lincomb(c, nb, cnt, Vc, T, -1.0, 1.0))) return rc;
        }
    }
    double *cur = T, *oth = tmp;
    for (int rep = 0; rep < 2; ++rep) {
        if ((rc = S.gram(cur, nb, cur, nb, g))) return rc;
        std::vector<double> L, Li;
        std::vector<char> ok;
        host_cholesky(g, nb, rep == 0 ? 1e-14 : 1e-4, L, ok);
        host_lower_inverse(L, nb, Li);
        int nk = 0;
        for (int j = 0; j < nb; ++j) nk += ok[j];
        if (nk == 0) { nb = 0; return RISP_OK; }
        std::vector<double> coef((size_t)nk * nb, 0.0);
        int r = 0;
        for (int j = 0; j < nb; ++j) {
            if (!ok[j]) continue;
            for (int c = 0; c < nb; ++c) coef[(size_t)r * nb + c] = ok[c] ? Li[(size_t)j * nb + c] : 0.0;
            ++r;
        }
        if ((rc = S.lincomb(coef, nk, nb, cur, oth, 1.0, 0.0))) return rc;
        std::swap(cur, oth);
        nb = nk;
    }
    return RISP_OK;
}

}  // namespace

extern "C" int risp_tddft_solve(risp_ctx *ctx, int32_t nroots, const risp_solve_options *opt_in, double *omega_out, double *X_out, double *Y_out,
                                risp_solve_info *info)
{
    if (!ctx) return RISP_EINVAL;
    const long long dim = (long long)ctx->nocc * ctx->nvir;
    if (nroots <= 0 || nroots > 32 || 2LL * nroots > dim || !omega_out) { risp_set_error(ctx, "risp_tddft_solve: need 1 <= nroots <= 32 and an output array"); return RISP_EINVAL; }
    if (!(ctx->flags & RISP_FLAG_TDDFT)) { risp_set_error(ctx, "risp_tddft_solve: the context was set up without RISP_FLAG_TDDFT"); return RISP_EINVAL; }
    RISP_CUDA_TRY(cudaSetDevice(ctx->device));
    risp_solve_options opt;
    std::memset(&opt, 0, sizeof(opt));
    if (opt_in) opt = *opt_in;
    const double tol = opt.tol > 0 ? opt.tol : 1e-5;
    const int max_iter = opt.max_iter > 0 ? opt.max_iter : 100;
    int n_guess = opt.n_guess > 0 ? opt.n_guess : 2 * nroots;
    n_guess = (int)std::min<long long>(std::max(n_guess, nroots), dim);
    const int max_sub = std::max(opt.max_sub > 0 ? opt.max_sub : 20 * nroots, 6 * nroots);
    auto t_start = std::chrono::steady_clock::now();
    double sec_mv = 0.0;
    int rc;
    if (ctx->w_Xin) { cudaFree(ctx->w_Xin); ctx->w_Xin = nullptr; }
    if (ctx->w_Sout) { cudaFree(ctx->w_Sout); ctx->w_Sout = nullptr; }
    ctx->xin_cap = 0;
    const int block = std::min(RISP_MS, ctx->max_batch);
    if ((rc = risp_ensure_workspace(ctx, block))) return rc;

    TdSolver S;
    S.ctx = ctx; S.dim = dim;
    S.slice = dim > (1 << 20) ? std::max<long long>(4096, ((dim / 1024) + 4095) / 4096 * 4096) : 16384;
    const int nzmax = (int)(dim / S.slice) + 2;
    const size_t vec = (size_t)dim * 8;
    {
        size_t free_b = 0, total_b = 0;
        RISP_CUDA_TRY(cudaMemGetInfo(&free_b, &total_b));
        size_t room = opt.device_budget_bytes ? std::min(opt.device_budget_bytes, free_b) : (size_t)(0.9 * (double)(free_b - std::min<size_t>((size_t)1 << 30, free_b / 8)));
        const size_t fixed = 4 * (size_t)nroots * vec + ((size_t)nzmax * 128 * 64 + 128 * 64) * 8 + (size_t)(max_sub + 64) * (max_sub + 64) * 8 + ((size_t)1 << 20);
        long long cap = room > fixed ? (long long)((room - fixed) / (3 * vec)) : 0;
        cap = std::min<long long>(cap, max_sub);
        if (cap < 6LL * nroots) { risp_set_error(ctx, "risp_tddft_solve: device memory too small for a subspace of 6 n_roots vectors (b, (A+B) b, (A-B) b)"); return RISP_ENOMEM; }
        S.kcap = (int)cap;
    }
    n_guess = std::min(n_guess, S.kcap - 2 * nroots);
    const int n2 = 2 * nroots;
    RISP_CUDA_TRY(S.scr.alloc(S.b, (size_t)S.kcap * dim));
    RISP_CUDA_TRY(S.scr.alloc(S.P, (size_t)S.kcap * dim));
    RISP_CUDA_TRY(S.scr.alloc(S.Q, (size_t)S.kcap * dim));
    RISP_CUDA_TRY(S.scr.alloc(S.T, (size_t)n2 * dim));
    RISP_CUDA_TRY(S.scr.alloc(S.tmp, (size_t)n2 * dim));
    RISP_CUDA_TRY(S.scr.alloc(S.dPart, (size_t)nzmax * 128 * 64));
    RISP_CUDA_TRY(S.scr.alloc(S.dSmall, (size_t)128 * 64));
    RISP_CUDA_TRY(S.scr.alloc(S.dCoef, (size_t)std::max(S.kcap, 128) * 128));
    RISP_CUDA_TRY(S.scr.alloc(S.dScale, (size_t)128));
    RISP_CUDA_TRY(S.scr.alloc(S.dIdx, (size_t)RISP_MS));
    const double sec_alloc = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();

    const int ld = S.kcap;
    std::vector<double> Mp((size_t)ld * ld, 0.0), Mm((size_t)ld * ld, 0.0);
    int n_sigma = 0, iterations = 0, restarts = 0, sub_max = 0;
    // (A+B) b and (A-B) b for basis vectors [k0, k0 + nb), projected matrices extended
    auto extend = [&](int k0, int nb) -> int {
        auto t0 = std::chrono::steady_clock::now();
        for (int j0 = 0; j0 < nb; j0 += block) {
            const int mb = std::min(block, nb - j0);
            int r = risp_matvec_impl(ctx, mb, S.b + (long long)(k0 + j0) * dim, S.P + (long long)(k0 + j0) * dim, S.st, S.Q + (long long)(k0 + j0) * dim);
            if (r) return r;
        }
        RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
        sec_mv += std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
        n_sigma += nb;
        std::vector<double> blk;
        const int kn = k0 + nb;
        for (int pass = 0; pass < 2; ++pass) {
            std::vector<double> &M = pass == 0 ? Mp : Mm;
            const double *W = (pass == 0 ? S.P : S.Q) + (long long)k0 * dim;
            for (int j0 = 0; j0 < nb; j0 += 64) {
                const int nj = std::min(64, nb - j0);
                for (int first = 0; first < kn; first += 128) {
                    const int cnt = std::min(128, kn - first);
                    int r = S.gram(S.b + (long long)first * dim, cnt, W + (long long)j0 * dim, nj, blk);
                    if (r) return r;
                    for (int i = 0; i < cnt; ++i)
                        for (int j = 0; j < nj; ++j) M[(size_t)(first + i) * ld + k0 + j0 + j] = blk[(size_t)i * nj + j];
                }
            }
            for (int i = 0; i < kn; ++i)           // symmetrise the new block, mirror the new columns
                for (int j = k0; j < kn; ++j) {
                    const double v = i >= k0 ? 0.5 * (M[(size_t)i * ld + j] + M[(size_t)j * ld + i]) : M[(size_t)i * ld + j];
                    M[(size_t)i * ld + j] = M[(size_t)j * ld + i] = v;
                }
        }
        S.k = kn;
        sub_max = std::max(sub_max, S.k);
        return RISP_OK;
    };

    // ---------------- initial guess: unit vectors on the smallest eps_a - eps_i
    {
        std::vector<std::pair<double, long long>> dl;
        const int no_top = (int)std::min<long long>(ctx->nocc, n_guess), nv_bot = (int)std::min<long long>(ctx->nvir, n_guess);
        for (int i = ctx->nocc - no_top; i < ctx->nocc; ++i)
            for (int a = 0; a < nv_bot; ++a) dl.push_back({ctx->h_eps[ctx->nocc + a] - ctx->h_eps[i], (long long)i * ctx->nvir + a});
        std::stable_sort(dl.begin(), dl.end(), [](auto &x, auto &y) { return x.first < y.first || (x.first == y.first && x.second < y.second); });
        for (int g0 = 0; g0 < n_guess; g0 += RISP_MS) {
            const int nb = std::min(RISP_MS, n_guess - g0);
            std::vector<long long> idx(nb);
            for (int j = 0; j < nb; ++j) idx[j] = dl[g0 + j].second;
            RISP_CUDA_TRY(cudaMemcpyAsync(S.dIdx, idx.data(), (size_t)nb * sizeof(long long), cudaMemcpyHostToDevice, S.st));
            td_unit_kernel<<<dim3(sgrid(dim), nb), 256, 0, S.st>>>(S.b + (long long)g0 * dim, dim, S.dIdx);
            RISP_CUDA_TRY(cudaGetLastError());
            RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
        }
        if ((rc = extend(0, n_guess))) return rc;
    }

    std::vector<double> omega(nroots, 0.0), rn(nroots, 0.0), U, V;      // U, V: [k][nroots] subspace coefficients of |X+Y>, |X-Y>
    bool converged = false;
    int n_unconv_prev = nroots;
    for (int it = 1; it <= max_iter; ++it) {
        iterations = it;
        // ---- reduced problem: M- = C C^T, C^T M+ C z = Omega^2 z
        auto reduced = [&]() -> int {
            const int k = S.k;
            std::vector<double> g((size_t)k * k), C, H((size_t)k * k), Tm((size_t)k * k), w, z;
            std::vector<char> ok;
            for (int i = 0; i < k; ++i)
                for (int j = 0; j < k; ++j) g[(size_t)i * k + j] = Mm[(size_t)i * ld + j];
            host_cholesky(g, k, 0.0, C, ok);
            for (int j = 0; j < k; ++j) if (!ok[j]) { risp_set_error(ctx, "risp_tddft_solve: the projected A - B is not positive definite (unstable reference)"); return RISP_ENOTPD; }
            for (int i = 0; i < k; ++i)           // Tm = M+ C
                for (int j = 0; j < k; ++j) {
                    double s = 0.0;
                    for (int q = j; q < k; ++q) s += Mp[(size_t)i * ld + q] * C[(size_t)q * k + j];
                    Tm[(size_t)i * k + j] = s;
                }
            for (int i = 0; i < k; ++i)           // H = C^T Tm
                for (int j = 0; j < k; ++j) {
                    double s = 0.0;
                    for (int q = i; q < k; ++q) s += C[(size_t)q * k + i] * Tm[(size_t)q * k + j];
                    H[(size_t)i * k + j] = s;
                }
            for (int i = 0; i < k; ++i)
                for (int j = 0; j < i; ++j) H[(size_t)i * k + j] = H[(size_t)j * k + i] = 0.5 * (H[(size_t)i * k + j] + H[(size_t)j * k + i]);
            risp_sym_eig_lowest(H, k, nroots, w, z);
            U.assign((size_t)k * nroots, 0.0); V.assign((size_t)k * nroots, 0.0);
            for (int r = 0; r < nroots; ++r) {
                if (!(w[r] > 0)) { risp_set_error(ctx, "risp_tddft_solve: non-positive Omega^2 in the subspace (unstable reference)"); return RISP_ENOTPD; }
                omega[r] = std::sqrt(w[r]);
                const double sc = 1.0 / std::sqrt(omega[r]);
                for (int i = 0; i < k; ++i) {
                    double s = 0.0;
                    for (int q = 0; q <= i; ++q) s += C[(size_t)i * k + q] * z[(size_t)q * k + r];
                    U[(size_t)i * nroots + r] = s * sc;
                }
                for (int i = 0; i < k; ++i) {
                    double s = 0.0;
                    for (int q = 0; q < k; ++q) s += Mp[(size_t)i * ld + q] * U[(size_t)q * nroots + r];
                    V[(size_t)i * nroots + r] = s / omega[r];
                }
            }
            return RISP_OK;
        };
        if ((rc = reduced())) return rc;
        // ---- restart from the orthonormalised {X+Y, X-Y} when the corrections of this iteration would not fit
        if (S.k > n2 && S.k + 2 * std::min(n_unconv_prev, nroots) > S.kcap) {
            const int k = S.k;
            std::vector<double> g((size_t)n2 * n2), L, Li;
            std::vector<char> ok;
            auto col = [&](int c, int i) { return c < nroots ? U[(size_t)i * nroots + c] : V[(size_t)i * nroots + c - nroots]; };
            for (int a = 0; a < n2; ++a)
                for (int c = 0; c < n2; ++c) {
                    double s = 0.0;
                    for (int i = 0; i < k; ++i) s += col(a, i) * col(c, i);
                    g[(size_t)a * n2 + c] = s;
                }
            double gmax = 0.0;
            for (int a = 0; a < n2; ++a) gmax = std::max(gmax, g[(size_t)a * n2 + a]);
            host_cholesky(g, n2, 1e-10 * gmax, L, ok);
            host_lower_inverse(L, n2, Li);
            int nk = 0;
            for (int a = 0; a < n2; ++a) nk += ok[a];
            std::vector<double> coef((size_t)nk * k, 0.0);      // new basis vector r = sum_i coef[r][i] b_i
            int r = 0;
            for (int a = 0; a < n2; ++a) {
                if (!ok[a]) continue;
                for (int c = 0; c <= a; ++c) {
                    if (!ok[c]) continue;
                    const double f = Li[(size_t)a * n2 + c];
                    for (int i = 0; i < k; ++i) coef[(size_t)r * k + i] += f * col(c, i);
                }
                ++r;
            }
            for (double *W : {S.b, S.P, S.Q}) {
                for (int r0 = 0; r0 < nk; r0 += n2) {
                    const int nr = std::min(n2, nk - r0);
                    std::vector<double> cc(coef.begin() + (size_t)r0 * k, coef.begin() + (size_t)(r0 + nr) * k);
                    if ((rc = S.lincomb(cc, nr, k, W, S.tmp, 1.0, 0.0))) return rc;
                    RISP_CUDA_TRY(cudaMemcpyAsync(S.T + (long long)r0 * dim, S.tmp, (size_t)nr * dim * 8, cudaMemcpyDeviceToDevice, S.st));
                }
                RISP_CUDA_TRY(cudaMemcpyAsync(W, S.T, (size_t)nk * dim * 8, cudaMemcpyDeviceToDevice, S.st));
                RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
            }
            for (std::vector<double> *M : {&Mp, &Mm}) {
                std::vector<double> t1((size_t)nk * k, 0.0), t2((size_t)nk * nk, 0.0);
                for (int a = 0; a < nk; ++a)
                    for (int j = 0; j < k; ++j) {
                        double s = 0.0;
                        for (int i = 0; i < k; ++i) s += coef[(size_t)a * k + i] * (*M)[(size_t)i * ld + j];
                        t1[(size_t)a * k + j] = s;
                    }
                for (int a = 0; a < nk; ++a)
                    for (int c = 0; c < nk; ++c) {
                        double s = 0.0;
                        for (int j = 0; j < k; ++j) s += t1[(size_t)a * k + j] * coef[(size_t)c * k + j];
                        t2[(size_t)a * nk + c] = s;
                    }
                std::fill(M->begin(), M->end(), 0.0);
                for (int a = 0; a < nk; ++a)
                    for (int c = 0; c < nk; ++c) (*M)[(size_t)a * ld + c] = 0.5 * (t2[(size_t)a * nk + c] + t2[(size_t)c * nk + a]);
            }
            S.k = nk;
            ++restarts;
            if ((rc = reduced())) return rc;
        }
        // ---- residuals r1 = P u - Omega b v, r2 = Q v - Omega b u  (T = [r1; r2])
        const int k = S.k;
        {
            std::vector<double> c1((size_t)nroots * k), c2((size_t)nroots * k), c3((size_t)nroots * k), c4((size_t)nroots * k);
            for (int r = 0; r < nroots; ++r)
                for (int i = 0; i < k; ++i) {
                    c1[(size_t)r * k + i] = U[(size_t)i * nroots + r]; c2[(size_t)r * k + i] = -omega[r] * V[(size_t)i * nroots + r];
                    c3[(size_t)r * k + i] = V[(size_t)i * nroots + r]; c4[(size_t)r * k + i] = -omega[r] * U[(size_t)i * nroots + r];
                }
            double *T2 = S.T + (long long)nroots * dim;
            if ((rc = S.lincomb(c1, nroots, k, S.P, S.T, 1.0, 0.0)) || (rc = S.lincomb(c2, nroots, k, S.b, S.T, 1.0, 1.0)) ||
                (rc = S.lincomb(c3, nroots, k, S.Q, T2, 1.0, 0.0)) || (rc = S.lincomb(c4, nroots, k, S.b, T2, 1.0, 1.0)))
                return rc;
        }
        std::vector<double> g;
        if ((rc = S.gram(S.T, n2, S.T, n2, g))) return rc;
        std::vector<int> unc;
        for (int r = 0; r < nroots; ++r) {
            rn[r] = std::sqrt(std::max(g[(size_t)r * n2 + r], g[(size_t)(nroots + r) * n2 + nroots + r]));
            if (!(rn[r] < tol)) unc.push_back(r);
        }
        n_unconv_prev = (int)unc.size();
        if (unc.empty()) { converged = true; break; }
        if (it == max_iter) break;
        // ---- corrections: both residuals of every unconverged root, preconditioned, compacted to the front of T (ascending: in place)
        int nb = 0;
        for (int half = 0; half < 2; ++half)
            for (int r : unc) {
                td_precondition_kernel<<<(unsigned)std::min<long long>(ctx->nocc, 148 * 16), 256, 0, S.st>>>(S.T + (long long)(half * nroots + r) * dim, omega[r], ctx->d_eps,
                                                                                                         ctx->nocc, ctx->nvir, S.T + (long long)nb * dim);
                RISP_CUDA_TRY(cudaGetLastError());
                ++nb;
            }
        nb = std::min(nb, S.kcap - S.k);
        if (nb <= 0) continue;                       // full: the next iteration restarts
        if ((rc = td_orthonormalise(S, S.T, S.tmp, nb))) return rc;
        if (nb == 0) break;                          // stagnated
        RISP_CUDA_TRY(cudaMemcpyAsync(S.b + (long long)S.k * dim, S.T, (size_t)nb * dim * 8, cudaMemcpyDeviceToDevice, S.st));
        if ((rc = extend(S.k, nb))) return rc;
    }
    for (int r = 0; r < nroots; ++r) omega_out[r] = omega[r];
    if (X_out || Y_out) {      // X = (|X+Y> + |X-Y>)/2, Y = (|X+Y> - |X-Y>)/2
        const int k = S.k;
        std::vector<double> cx((size_t)nroots * k), cy((size_t)nroots * k);
        for (int r = 0; r < nroots; ++r)
            for (int i = 0; i < k; ++i) {
                cx[(size_t)r * k + i] = 0.5 * (U[(size_t)i * nroots + r] + V[(size_t)i * nroots + r]);
                cy[(size_t)r * k + i] = 0.5 * (U[(size_t)i * nroots + r] - V[(size_t)i * nroots + r]);
            }
        if (X_out && (rc = S.lincomb(cx, nroots, k, S.b, X_out, 1.0, 0.0))) return rc;
        if (Y_out && (rc = S.lincomb(cy, nroots, k, S.b, Y_out, 1.0, 0.0))) return rc;
    }
    if (info) {
        std::memset(info, 0, sizeof(*info));
        info->iterations = iterations; info->restarts = restarts; info->n_sigma = n_sigma; info->converged = converged ? 1 : 0;
        for (int r = 0; r < nroots; ++r) info->resid[r] = rn[r];
        info->sec_total = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
        info->sec_matvec = sec_mv; info->sec_alloc = sec_alloc; info->sec_subspace = info->sec_total - sec_mv - sec_alloc;
        info->subspace_max = sub_max; info->cached_vectors = S.kcap; info->block = block; info->capacity = S.kcap;
    }
    if (!converged) { risp_set_error(ctx, "risp_tddft_solve: not converged within max_iter"); return RISP_ENOTCONV; }
    return RISP_OK;
}
