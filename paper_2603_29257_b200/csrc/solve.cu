// solve.cu -- risp_tda_solve: host-memory-assisted Davidson for the lowest roots of A X = X Omega (Eq. 9).
//
// Placement follows PAPER.md:189-201 (Fig. 2): the expansion vectors V and their images W = A V live in PINNED HOST
// memory; only the newest block, the Ritz vectors and two streaming chunk buffers are device resident.  Every pass
// over the subspace (projection V^T W_new, Ritz reconstruction X = V y / A X = W y, orthogonalisation of the
// corrections) streams V / W through the device in chunks on a side stream, double buffered against the compute
// stream.  When the subspace would outgrow its budget the solver restarts from the current Ritz vectors
// (reading G17: W <- W y by linearity, no extra sigma-build).
// "Assisted": whatever HBM is left after the K tensors and the matvec work space holds the leading part of V and W on the
// device; the vectors beyond it live in pinned host memory (page-locked chunk by chunk by a background thread) and are
// streamed over the host link on the side stream -- none for the small configurations, most of them at 3000 atoms, all of
// them with RISP_SOLVE_NO_CACHE.
// The Davidson recipe itself (guess, preconditioner, Gram-Schmidt) is the "standard" one of DESIGN.md reading G16.
#include "ctx.h"
#include <algorithm>
#include <atomic>
#include <chrono>
#include <cmath>
#include <thread>

namespace {

// ------------------------------------------------------------------------------------------------ device kernels
__global__ void unit_guess_kernel(double *V, long long dim, const long long *idx, int n)
{
    int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < n) V[(long long)j * dim + idx[j]] = 1.0;
}

// res[j] = AX[j] - theta[j] X[j]; partial squared norms per block -> part[j][blockIdx.x]
__global__ void residual_kernel(const double *__restrict__ X, const double *__restrict__ AX, const double *__restrict__ theta,
                                double *__restrict__ res, long long dim, double *__restrict__ part)
{
    const int j = blockIdx.y;
    const double th = theta[j];
    double s = 0.0;
    for (long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x; x < dim; x += (long long)gridDim.x * blockDim.x) {
        double r = AX[j * dim + x] - th * X[j * dim + x];
        res[j * dim + x] = r;
        s += r * r;
    }
    __shared__ double sh[256];
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) part[j * gridDim.x + blockIdx.x] = sh[0];
}

// t[j] = res[src[j]] / (theta[src[j]] - (eps_a - eps_i)), |denominator| floored at 1e-8 (sign kept)
__global__ void precondition_kernel(const double *__restrict__ res, const double *__restrict__ theta, const int *__restrict__ src,
                                    const double *__restrict__ eps, int nocc, int nvir, double *__restrict__ t, long long dim)
{
    const int j = blockIdx.y, sj = src[j];
    const double th = theta[sj];
    for (long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x; x < dim; x += (long long)gridDim.x * blockDim.x) {
        int a = (int)(x % nvir), i = (int)(x / nvir);
        double den = th - (eps[nocc + a] - eps[i]);
        if (fabs(den) < 1e-8) den = den < 0 ? -1e-8 : 1e-8;
        t[j * dim + x] = res[sj * dim + x] / den;
    }
}

__global__ void reduce_partials_kernel(const double *__restrict__ part, int nz, int n, double *__restrict__ out)
{
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    double s = 0.0;
    for (int z = 0; z < nz; ++z) s += part[(long long)z * n + e];
    out[e] = s;
}

// ------------------------------------------------------------------------------------------------ host eigen solver
// Symmetric eigenproblem of the projected matrix (k <= a few hundred): Householder tridiagonalisation followed by the
// implicit-shift QL iteration, eigenvectors accumulated.  a: n x n row-major (destroyed); w ascending; z[i*n + j] = i-th
// component of eigenvector j.
void sym_eig(std::vector<double> &a, int n, std::vector<double> &w, std::vector<double> &z)
{
    // zt[j*n + i] = i-th component of (current) basis vector j: every update below runs over contiguous rows
    std::vector<double> zt((size_t)n * n, 0.0);
    for (int i = 0; i < n; ++i) zt[(size_t)i * n + i] = 1.0;
    std::vector<double> v(n), p(n), d(n), e(n, 0.0), sr(n);
    for (int k = 0; k + 2 < n; ++k) {
        int len = n - k - 1;
        double nrm = 0.0;
        for (int i = 0; i < len; ++i) { v[i] = a[(size_t)(k + 1 + i) * n + k]; nrm += v[i] * v[i]; }
        nrm = std::sqrt(nrm);
        double tail = 0.0;
        for (int i = 1; i < len; ++i) tail += v[i] * v[i];
        if (tail == 0.0) continue;                        // already tridiagonal in this column
        double alpha = v[0] > 0 ? -nrm : nrm;
        v[0] -= alpha;
        double vv = 0.0;
        for (int i = 0; i < len; ++i) vv += v[i] * v[i];
        double beta = 2.0 / vv;
        for (int i = 0; i < len; ++i) {                   // p = beta A22 v
            double s = 0.0;
            const double *row = &a[(size_t)(k + 1 + i) * n + k + 1];
            for (int j = 0; j < len; ++j) s += row[j] * v[j];
            p[i] = beta * s;
        }
        double K = 0.0;
        for (int i = 0; i < len; ++i) K += v[i] * p[i];
        K *= 0.5 * beta;
        for (int i = 0; i < len; ++i) p[i] -= K * v[i];   // w
        for (int i = 0; i < len; ++i) {
            double *row = &a[(size_t)(k + 1 + i) * n + k + 1];
            const double vi = v[i], pi = p[i];
            for (int j = 0; j < len; ++j) row[j] -= vi * p[j] + pi * v[j];
        }
        a[(size_t)(k + 1) * n + k] = a[(size_t)k * n + k + 1] = alpha;
        for (int i = 1; i < len; ++i) a[(size_t)(k + 1 + i) * n + k] = a[(size_t)k * n + k + 1 + i] = 0.0;
        // Q <- Q H: columns k+1.. of Q are rows k+1.. of zt;  s_r = sum_j Q[r][k+1+j] v[j]
        std::fill(sr.begin(), sr.end(), 0.0);
        for (int j = 0; j < len; ++j) {
            const double *zr = &zt[(size_t)(k + 1 + j) * n];
            const double vj = v[j];
            for (int r = 0; r < n; ++r) sr[r] += zr[r] * vj;
        }
        for (int j = 0; j < len; ++j) {
            double *zr = &zt[(size_t)(k + 1 + j) * n];
            const double bv = beta * v[j];
            for (int r = 0; r < n; ++r) zr[r] -= sr[r] * bv;
        }
    }
    for (int i = 0; i < n; ++i) d[i] = a[(size_t)i * n + i];
    for (int i = 0; i + 1 < n; ++i) e[i] = a[(size_t)(i + 1) * n + i];
    // implicit QL with Wilkinson-type shift
    for (int l = 0; l < n; ++l) {
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
                    double *z0 = &zt[(size_t)i * n], *z1 = &zt[(size_t)(i + 1) * n];
                    for (int k = 0; k < n; ++k) {
                        const double f2 = z1[k];
                        z1[k] = s * z0[k] + c * f2;
                        z0[k] = c * z0[k] - s * f2;
                    }
                }
                if (r == 0.0 && i >= l) continue;
                d[l] -= pp; e[l] = g; e[m] = 0.0;
            }
        } while (m != l);
    }
    // sort ascending; z[i*n + j] = i-th component of eigenvector j
    std::vector<int> ord(n);
    for (int i = 0; i < n; ++i) ord[i] = i;
    std::sort(ord.begin(), ord.end(), [&](int x, int y) { return d[x] < d[y]; });
    w.resize(n);
    z.assign((size_t)n * n, 0.0);
    for (int j = 0; j < n; ++j) {
        w[j] = d[ord[j]];
        const double *zr = &zt[(size_t)ord[j] * n];
        for (int i = 0; i < n; ++i) z[(size_t)i * n + j] = zr[i];
    }
}

// The nv lowest eigenpairs only (what a Davidson iteration needs; the full QL accumulation above costs ~9 n^3 flops, 90 ms at
// n = 315, once per iteration): Householder tridiagonalisation with the reflectors kept, eigenvalues by QL without vectors,
// eigenvectors of T by inverse iteration (pivoted tridiagonal LU, re-orthogonalised against the vectors already found, as
// LAPACK's dstein does for clusters), back-transformed through the reflectors.  z[i*n + j], j < nv; w has all n eigenvalues.
void sym_eig_lowest(std::vector<double> &a, int n, int nv, std::vector<double> &w, std::vector<double> &z)
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

// The pinned host copy of the subspace: V and W as chunks of 32 vectors, page-locked by a background thread
// while the first sigma-builds run (pinning 7 GB takes ~2.7 s -- a fifth of a 300-atom solve if done up front).
struct HostStore {
    static constexpr int CHV = 32;
    long long dim = 0;
    int nchunks = 0, device = 0, slots = 0;
    std::vector<double *> v, w;
    std::atomic<int> ready{0}, failed{0}, stop{0};
    std::thread th;
    void start(int dev, long long dim_, int slots_)
    {
        device = dev; dim = dim_; slots = slots_;
        nchunks = (slots + CHV - 1) / CHV;
        v.assign(nchunks, nullptr); w.assign(nchunks, nullptr);
        th = std::thread([this] {
            cudaSetDevice(device);
            for (int c = 0; c < nchunks && !stop.load(); ++c) {
                const size_t nvec = (size_t)std::min(CHV, slots - c * CHV);
                if (cudaHostAlloc((void **)&v[c], nvec * dim * 8, cudaHostAllocDefault) != cudaSuccess ||
                    cudaHostAlloc((void **)&w[c], nvec * dim * 8, cudaHostAllocDefault) != cudaSuccess) { failed.store(1); return; }
                ready.store(c + 1, std::memory_order_release);
            }
        });
    }
    // host address of vector i of V (isW = false) or W; blocks until its chunk is pinned; nullptr if the allocation failed
    double *ptr(bool isW, long long i)
    {
        const int c = (int)(i / CHV);
        while (ready.load(std::memory_order_acquire) <= c) {
            if (failed.load()) return nullptr;
            std::this_thread::yield();
        }
        return (isW ? w[c] : v[c]) + (i % CHV) * dim;
    }
    ~HostStore() { finish(); }
    void finish()
    {
        stop.store(1);
        if (th.joinable()) th.join();
        for (double *p : v) if (p) cudaFreeHost(p);
        for (double *p : w) if (p) cudaFreeHost(p);
        v.clear(); w.clear();
    }
};

struct Solver {
    risp_ctx *ctx;
    long long dim;
    int cap = 0, k = 0, CH = 16;
    HostStore host;                                // pinned host copy of V and W
    double *dB = nullptr, *dWB = nullptr;          // newest block and its image [32][dim]
    double *dX = nullptr, *dAX = nullptr, *dRes = nullptr, *dT = nullptr;   // [nroots][dim]
    double *dChunk[2] = {nullptr, nullptr};        // streaming buffers [CH][dim]
    double *dVc = nullptr, *dWc = nullptr;         // device cache of the first ncache subspace vectors [ncache][dim]
    int ncache = 0;
    long long slice = 16384;                       // split-K slice of the Gram products
    std::vector<double> tmp;
    double *dCoef = nullptr, *dPart = nullptr, *dSmall = nullptr, *dTheta = nullptr;
    int *dSrc = nullptr;
    cudaEvent_t evUp[2], evFree[2], evD2H, evReady;
    double bytes_h2d = 0, bytes_d2h = 0;
    cudaStream_t st = 0;                           // compute stream (default)
};

int gram(Solver &S, const double *A, int na, const double *B, int nb, std::vector<double> &out)
{
    // out[na][nb] = sum_x A[i][x] B[j][x]: split-K batched DMMA GEMM + fixed-order reduction.  The smaller operand goes to the
    // M side (16-row tiles exist, the N tile is always 128 wide); the product is HBM-bound: it reads (na + nb) dim doubles.
    risp_ctx *ctx = S.ctx;
    const bool swap = na > nb;
    const double *P = swap ? B : A, *Q = swap ? A : B;
    const int np = swap ? nb : na, nq = swap ? na : nb;
    const long long slice = S.slice;
    int nfull = (int)(S.dim / slice);
    long long tail = S.dim - (long long)nfull * slice;
    int nz = nfull + (tail ? 1 : 0);
    if (nfull) {
        GemmDesc d = gemm_desc(np, nq, (int)slice, P, S.dim, true, Q, S.dim, true, S.dPart, nq);
        d.nb1 = nfull; d.sA1 = slice; d.sB1 = slice; d.sC1 = (long long)np * nq;
        RISP_CUDA_TRY(risp_dgemm(d, S.st));
    }
    if (tail) {
        GemmDesc d = gemm_desc(np, nq, (int)tail, P + (long long)nfull * slice, S.dim, true, Q + (long long)nfull * slice, S.dim, true,
                               S.dPart + (long long)nfull * np * nq, nq);
        RISP_CUDA_TRY(risp_dgemm(d, S.st));
    }
    reduce_partials_kernel<<<(np * nq + 127) / 128, 128, 0, S.st>>>(S.dPart, nz, np * nq, S.dSmall);
    out.resize((size_t)na * nb);
    if (!swap) {
        RISP_CUDA_TRY(cudaMemcpyAsync(out.data(), S.dSmall, (size_t)na * nb * 8, cudaMemcpyDeviceToHost, S.st));
        RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
    } else {
        S.tmp.resize((size_t)na * nb);
        RISP_CUDA_TRY(cudaMemcpyAsync(S.tmp.data(), S.dSmall, (size_t)na * nb * 8, cudaMemcpyDeviceToHost, S.st));
        RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
        for (int i = 0; i < na; ++i)
            for (int j = 0; j < nb; ++j) out[(size_t)i * nb + j] = S.tmp[(size_t)j * na + i];
    }
    return RISP_OK;
}

// C[nc][dim] = alpha * coef[nc][na] * A[na][dim] + beta * C
int lincomb(Solver &S, const std::vector<double> &coef, int nc, int na, const double *A, double *C, double alpha, double beta)
{
    risp_ctx *ctx = S.ctx;
    RISP_CUDA_TRY(cudaMemcpyAsync(S.dCoef, coef.data(), (size_t)nc * na * 8, cudaMemcpyHostToDevice, S.st));
    GemmDesc d = gemm_desc(nc, (int)std::min<long long>(S.dim, 1 << 30), na, S.dCoef, na, true, A, S.dim, false, C, S.dim, alpha, beta);
    RISP_CUDA_TRY(risp_dgemm(d, S.st));
    RISP_CUDA_TRY(cudaStreamSynchronize(S.st));   // coef is a host temporary
    return RISP_OK;
}

// pass over subspace vectors [0, n): the first ncache come from the device cache `dc` (chunks of up to 128), the others are
// streamed from the pinned host store (V or W) in chunks on the side stream; fn(dev_ptr, first, count) runs on the compute stream
template <class F>
int stream_pass(Solver &S, bool isW, const double *dc, int n, F &&fn)
{
    risp_ctx *ctx = S.ctx;
    int rc;
    const int nc = std::min(n, S.ncache);
    for (int first = 0; first < nc; first += 128)
        if ((rc = fn(dc + (long long)first * S.dim, first, std::min(128, nc - first)))) return rc;
    const int rest = n - nc;
    int nchunk = (rest + S.CH - 1) / S.CH;
    auto upload = [&](int c) -> int {
        int b = c & 1, first = nc + c * S.CH, cnt = std::min(S.CH, n - first);
        RISP_CUDA_TRY(cudaStreamWaitEvent(ctx->side, S.evFree[b], 0));
        for (int done = 0; done < cnt;) {           // a block of CH vectors may straddle two pinned chunks
            const int i = first + done - S.ncache, seg = std::min(cnt - done, HostStore::CHV - i % HostStore::CHV);
            const double *h = S.host.ptr(isW, i);
            if (!h) { risp_set_error(ctx, "risp_tda_solve: pinned host allocation of the subspace failed"); return RISP_ENOMEM; }
            RISP_CUDA_TRY(cudaMemcpyAsync(S.dChunk[b] + (long long)done * S.dim, h, (size_t)seg * S.dim * 8, cudaMemcpyHostToDevice, ctx->side));
            done += seg;
        }
        RISP_CUDA_TRY(cudaEventRecord(S.evUp[b], ctx->side));
        S.bytes_h2d += (double)cnt * S.dim * 8;
        return RISP_OK;
    };
    if (nchunk > 0 && (rc = upload(0))) return rc;
    for (int c = 0; c < nchunk; ++c) {
        if (c + 1 < nchunk && (rc = upload(c + 1))) return rc;
        int b = c & 1, first = nc + c * S.CH, cnt = std::min(S.CH, n - first);
        RISP_CUDA_TRY(cudaStreamWaitEvent(S.st, S.evUp[b], 0));
        if ((rc = fn(S.dChunk[b], first, cnt))) return rc;
        RISP_CUDA_TRY(cudaEventRecord(S.evFree[b], S.st));
    }
    return RISP_OK;
}

// store device vectors src[0, n) as subspace vectors [k, k+n): into the device cache while it reaches, beyond it into the
// pinned host store (side stream, after the compute stream has produced them)
int store_vectors(Solver &S, bool isW, double *dc, int k, const double *src, int n)
{
    risp_ctx *ctx = S.ctx;
    const int nc = std::max(0, std::min(n, S.ncache - k));       // vectors that land in the device cache
    if (nc > 0) RISP_CUDA_TRY(cudaMemcpyAsync(dc + (long long)k * S.dim, src, (size_t)nc * S.dim * 8, cudaMemcpyDeviceToDevice, S.st));
    if (nc == n) return RISP_OK;
    RISP_CUDA_TRY(cudaEventRecord(S.evReady, S.st));
    RISP_CUDA_TRY(cudaStreamWaitEvent(ctx->side, S.evReady, 0));
    for (int done = nc; done < n;) {
        const int i = k + done - S.ncache, seg = std::min(n - done, HostStore::CHV - i % HostStore::CHV);
        double *h = S.host.ptr(isW, i);
        if (!h) { risp_set_error(ctx, "risp_tda_solve: pinned host allocation of the subspace failed"); return RISP_ENOMEM; }
        RISP_CUDA_TRY(cudaMemcpyAsync(h, src + (long long)done * S.dim, (size_t)seg * S.dim * 8, cudaMemcpyDeviceToHost, ctx->side));
        S.bytes_d2h += (double)seg * S.dim * 8;
        done += seg;
    }
    return RISP_OK;
}

}  // namespace

extern "C" int risp_tda_solve(risp_ctx *ctx, int32_t nroots, const risp_solve_options *opt_in, double *omega_out, double *X_out,
                              risp_solve_info *info)
{
    if (!ctx) return RISP_EINVAL;
    const long long dim = (long long)ctx->nocc * ctx->nvir;
    if (nroots <= 0 || nroots > RISP_MAX_ROOTS || nroots > dim || !omega_out) { risp_set_error(ctx, "risp_tda_solve: bad nroots or NULL output"); return RISP_EINVAL; }
    RISP_CUDA_TRY(cudaSetDevice(ctx->device));
    risp_solve_options opt;
    std::memset(&opt, 0, sizeof(opt));
    if (opt_in) opt = *opt_in;
    const double tol = opt.tol > 0 ? opt.tol : 1e-5;
    const int max_iter = opt.max_iter > 0 ? opt.max_iter : 100;
    int n_guess = opt.n_guess > 0 ? opt.n_guess : 2 * nroots;
    n_guess = (int)std::min<long long>(std::max(n_guess, nroots), dim);
    int max_sub = opt.max_sub > 0 ? opt.max_sub : 20 * nroots;
    auto t_start = std::chrono::steady_clock::now();
    double sec_mv = 0.0;

    Solver S;
    S.ctx = ctx; S.dim = dim;
    const int nbmax = std::max(n_guess, nroots);
    auto DA = [&](double *&p, size_t n) -> int { RISP_CUDA_TRY(cudaMalloc((void **)&p, n * 8)); return RISP_OK; };
    int rc;
    if ((rc = DA(S.dB, (size_t)nbmax * dim)) || (rc = DA(S.dWB, (size_t)nbmax * dim)) || (rc = DA(S.dX, (size_t)nroots * dim)) ||
        (rc = DA(S.dAX, (size_t)nroots * dim)) || (rc = DA(S.dRes, (size_t)nroots * dim)) || (rc = DA(S.dT, (size_t)nroots * dim)) ||
        (rc = DA(S.dChunk[0], (size_t)S.CH * dim)) || (rc = DA(S.dChunk[1], (size_t)S.CH * dim)))
        return rc;
    S.slice = dim > (1 << 20) ? 4096 : 16384;      // enough slices to give every SM a tile
    const int nzmax = (int)(dim / S.slice) + 2;
    if ((rc = DA(S.dPart, std::max((size_t)nzmax * 128 * 64, (size_t)RISP_MAX_ROOTS * 256))) || (rc = DA(S.dSmall, (size_t)128 * 64 + 4096)) ||
        (rc = DA(S.dTheta, (size_t)RISP_MAX_ROOTS)))
        return rc;
    RISP_CUDA_TRY(cudaMalloc((void **)&S.dSrc, RISP_MAX_ROOTS * sizeof(int)));
    for (int b = 0; b < 2; ++b) { RISP_CUDA_TRY(cudaEventCreateWithFlags(&S.evUp[b], cudaEventDisableTiming)); RISP_CUDA_TRY(cudaEventCreateWithFlags(&S.evFree[b], cudaEventDisableTiming)); }
    RISP_CUDA_TRY(cudaEventCreateWithFlags(&S.evD2H, cudaEventDisableTiming));
    RISP_CUDA_TRY(cudaEventCreateWithFlags(&S.evReady, cudaEventDisableTiming));

    // subspace capacity: the user's max_sub, bounded by what HBM (left once the matvec work space for the largest
    // block exists) and the pinned-host budget can hold together; vectors [0, ncache) live on the device, the others on the host
    int slots = 0;
    {
        int rcw = risp_ensure_workspace(ctx, std::min(nbmax, RISP_MS));
        if (rcw) return rcw;
        size_t free_b = 0, total_b = 0;
        RISP_CUDA_TRY(cudaMemGetInfo(&free_b, &total_b));
        const size_t keep = (size_t)1 << 30, pervec = 2 * (size_t)dim * 8;
        size_t room = free_b > keep ? (size_t)(0.9 * (double)(free_b - keep)) : 0;
        long long dev_vecs = (opt.flags & 1) ? 0 : (long long)(room / pervec);      // flags bit 0: no device cache (testing the streamed path)
        if (opt.flags & 2) dev_vecs = std::min<long long>(dev_vecs, nroots + 2);     // flags bit 1: tiny cache (testing the mixed path)
        const long long host_vecs = (long long)(ctx->host_budget / pervec);
        slots = (int)std::min<long long>((long long)max_sub + nroots, dev_vecs + host_vecs);
        slots = std::max(slots, std::max(n_guess, 2 * nroots) + nroots);
        S.cap = slots - nroots;                     // room to append one more block before the restart decision
        S.ncache = (int)std::min<long long>(slots, dev_vecs);
        if (S.ncache > 0) {
            RISP_CUDA_TRY(cudaMalloc((void **)&S.dVc, (size_t)S.ncache * dim * 8));
            RISP_CUDA_TRY(cudaMalloc((void **)&S.dWc, (size_t)S.ncache * dim * 8));
        }
        // vectors beyond the cache live in pinned host memory only; nothing is pinned when everything fits in HBM
        if (slots > S.ncache) S.host.start(ctx->device, dim, slots - S.ncache);
        const int small = std::max(slots, 64);
        if ((rc = DA(S.dCoef, (size_t)small * small))) return rc;
    }

    auto cleanup = [&]() {
        cudaDeviceSynchronize();
        S.host.finish();
        double *bufs[] = {S.dB, S.dWB, S.dX, S.dAX, S.dRes, S.dT, S.dChunk[0], S.dChunk[1], S.dCoef, S.dPart, S.dSmall, S.dTheta};
        for (double *b : bufs) if (b) cudaFree(b);
        if (S.dSrc) cudaFree(S.dSrc);
        for (int b = 0; b < 2; ++b) { cudaEventDestroy(S.evUp[b]); cudaEventDestroy(S.evFree[b]); }
        cudaEventDestroy(S.evD2H); cudaEventDestroy(S.evReady);
        if (S.dVc) cudaFree(S.dVc);
        if (S.dWc) cudaFree(S.dWc);
    };
#define SOLVE_TRY(x) do { int rc_ = (x); if (rc_) { cleanup(); return rc_; } } while (0)

    // ---------------- initial guess: unit vectors on the smallest eps_a - eps_i
    int nb = n_guess;
    {
        std::vector<std::pair<double, long long>> dl;
        // the n_guess smallest differences: occupied from the top, virtual from the bottom
        int no_top = (int)std::min<long long>(ctx->nocc, n_guess), nv_bot = (int)std::min<long long>(ctx->nvir, n_guess);
        for (int i = ctx->nocc - no_top; i < ctx->nocc; ++i)
            for (int a = 0; a < nv_bot; ++a) dl.push_back({ctx->h_eps[ctx->nocc + a] - ctx->h_eps[i], (long long)i * ctx->nvir + a});
        std::stable_sort(dl.begin(), dl.end(), [](auto &x, auto &y) { return x.first < y.first || (x.first == y.first && x.second < y.second); });
        std::vector<long long> idx(nb);
        for (int j = 0; j < nb; ++j) idx[j] = dl[j].second;
        long long *d_idx = nullptr;
        RISP_CUDA_TRY(cudaMalloc((void **)&d_idx, nb * sizeof(long long)));
        RISP_CUDA_TRY(cudaMemcpy(d_idx, idx.data(), nb * sizeof(long long), cudaMemcpyHostToDevice));
        RISP_CUDA_TRY(cudaMemsetAsync(S.dB, 0, (size_t)nb * dim * 8, S.st));
        unit_guess_kernel<<<(nb + 63) / 64, 64, 0, S.st>>>(S.dB, dim, d_idx, nb);
        RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
        cudaFree(d_idx);
    }

    std::vector<double> G;          // projected matrix, k x k, row-major with leading dimension ldg
    const int ldg = slots;
    G.assign((size_t)ldg * ldg, 0.0);
    std::vector<double> theta(nroots, 0.0), rn(nroots, 0.0), yv;
    int iterations = 0, restarts = 0, n_sigma = 0, sub_max = 0;
    bool converged = false;
    S.k = 0;

    const double sec_alloc = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
    for (int it = 1; it <= max_iter; ++it) {
        iterations = it;
        // ---- W_B = A B
        {
            auto t0 = std::chrono::steady_clock::now();
            for (int b0 = 0; b0 < nb; b0 += RISP_MS) {
                int mb = std::min(RISP_MS, nb - b0);
                SOLVE_TRY(risp_ensure_workspace(ctx, mb));
                SOLVE_TRY(risp_matvec_impl(ctx, mb, S.dB + (long long)b0 * dim, S.dWB + (long long)b0 * dim, S.st));
            }
            RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
            sec_mv += std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
            n_sigma += nb;
        }
        // ---- projected matrix: G[0:k][k:k+nb] = V_old^T W_B (stream V_old), G[k:,k:] = B^T W_B
        {
            const int k = S.k;
            std::vector<double> blk;
            SOLVE_TRY(stream_pass(S, false, S.dVc, k, [&](const double *Vc, int first, int cnt) -> int {
                int r = gram(S, Vc, cnt, S.dWB, nb, blk);
                if (r) return r;
                for (int i = 0; i < cnt; ++i)
                    for (int j = 0; j < nb; ++j) G[(size_t)(first + i) * ldg + k + j] = G[(size_t)(k + j) * ldg + first + i] = blk[(size_t)i * nb + j];
                return RISP_OK;
            }));
            SOLVE_TRY(gram(S, S.dB, nb, S.dWB, nb, blk));
            for (int i = 0; i < nb; ++i)
                for (int j = 0; j < nb; ++j) G[(size_t)(k + i) * ldg + k + j] = 0.5 * (blk[(size_t)i * nb + j] + blk[(size_t)j * nb + i]);
            // append B, W_B to the pinned host subspace (side stream)
            SOLVE_TRY(store_vectors(S, false, S.dVc, k, S.dB, nb));
            SOLVE_TRY(store_vectors(S, true, S.dWc, k, S.dWB, nb));
            RISP_CUDA_TRY(cudaEventRecord(S.evD2H, ctx->side));
            S.k += nb;
            sub_max = std::max(sub_max, S.k);
        }
        // ---- Ritz pairs of the projected matrix
        const int k = S.k;
        {
            std::vector<double> a((size_t)k * k), w;
            for (int i = 0; i < k; ++i)
                for (int j = 0; j < k; ++j) a[(size_t)i * k + j] = G[(size_t)i * ldg + j];
            sym_eig_lowest(a, k, nroots, w, yv);
            for (int j = 0; j < nroots; ++j) theta[j] = w[j];
        }
        // ---- X = V y, AX = W y (stream V and W; needs the appended block on the host)
        RISP_CUDA_TRY(cudaEventSynchronize(S.evD2H));
        for (int pass = 0; pass < 2; ++pass) {
            double *dst = pass == 0 ? S.dX : S.dAX;
            bool first_chunk = true;
            SOLVE_TRY(stream_pass(S, pass != 0, pass == 0 ? S.dVc : S.dWc, k, [&](const double *Vc, int first, int cnt) -> int {
                std::vector<double> coef((size_t)nroots * cnt);
                for (int j = 0; j < nroots; ++j)
                    for (int i = 0; i < cnt; ++i) coef[(size_t)j * cnt + i] = yv[(size_t)(first + i) * k + j];
                int r = lincomb(S, coef, nroots, cnt, Vc, dst, 1.0, first_chunk ? 0.0 : 1.0);
                first_chunk = false;
                return r;
            }));
        }
        // ---- residuals
        {
            RISP_CUDA_TRY(cudaMemcpyAsync(S.dTheta, theta.data(), nroots * 8, cudaMemcpyHostToDevice, S.st));
            const int gx = 256;
            residual_kernel<<<dim3(gx, nroots), 256, 0, S.st>>>(S.dX, S.dAX, S.dTheta, S.dRes, dim, S.dPart);
            std::vector<double> part((size_t)nroots * gx);
            RISP_CUDA_TRY(cudaMemcpyAsync(part.data(), S.dPart, part.size() * 8, cudaMemcpyDeviceToHost, S.st));
            RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
            for (int j = 0; j < nroots; ++j) {
                double s = 0.0;
                for (int b = 0; b < gx; ++b) s += part[(size_t)j * gx + b];
                rn[j] = std::sqrt(s);
            }
        }
        std::vector<int> src;
        for (int j = 0; j < nroots; ++j) if (!(rn[j] < tol)) src.push_back(j);
        if (src.empty()) { converged = true; break; }
        if (it == max_iter) break;
        // ---- restart from the Ritz vectors when the next block would not fit
        if (k + (int)src.size() > S.cap) {
            SOLVE_TRY(store_vectors(S, false, S.dVc, 0, S.dX, nroots));
            SOLVE_TRY(store_vectors(S, true, S.dWc, 0, S.dAX, nroots));
            RISP_CUDA_TRY(cudaEventRecord(S.evD2H, ctx->side));
            RISP_CUDA_TRY(cudaEventSynchronize(S.evD2H));
            std::fill(G.begin(), G.end(), 0.0);
            for (int j = 0; j < nroots; ++j) G[(size_t)j * ldg + j] = theta[j];
            S.k = nroots;
            ++restarts;
        }
        // ---- corrections t_j = r_j / (theta_j - Delta), normalised
        nb = (int)src.size();
        {
            RISP_CUDA_TRY(cudaMemcpyAsync(S.dSrc, src.data(), nb * sizeof(int), cudaMemcpyHostToDevice, S.st));
            precondition_kernel<<<dim3(256, nb), 256, 0, S.st>>>(S.dRes, S.dTheta, S.dSrc, ctx->d_eps, ctx->nocc, ctx->nvir, S.dT, dim);
            RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
        }
        auto normalise_rows = [&](double *T, int n, std::vector<double> &norms) -> int {
            std::vector<double> g;
            int r = gram(S, T, n, T, n, g);
            if (r) return r;
            norms.resize(n);
            std::vector<double> coef((size_t)n * n, 0.0);
            for (int j = 0; j < n; ++j) { norms[j] = std::sqrt(g[(size_t)j * n + j]); coef[(size_t)j * n + j] = norms[j] > 0 ? 1.0 / norms[j] : 0.0; }
            // scale in place through a temporary: B = coef * T, then copy back
            r = lincomb(S, coef, n, n, T, S.dB, 1.0, 0.0);
            if (r) return r;
            RISP_CUDA_TRY(cudaMemcpyAsync(T, S.dB, (size_t)n * dim * 8, cudaMemcpyDeviceToDevice, S.st));
            return RISP_OK;
        };
        std::vector<double> norms;
        SOLVE_TRY(normalise_rows(S.dT, nb, norms));
        // ---- orthogonalise against V: per streamed chunk, two projections (block Gram-Schmidt with re-orthogonalisation)
        SOLVE_TRY(stream_pass(S, false, S.dVc, S.k, [&](const double *Vc, int first, int cnt) -> int {
            for (int rep = 0; rep < 2; ++rep) {
                std::vector<double> c;
                int r = gram(S, S.dT, nb, Vc, cnt, c);       // c[j][i] = t_j . v_i
                if (r) return r;
                r = lincomb(S, c, nb, cnt, Vc, S.dT, -1.0, 1.0);
                if (r) return r;
            }
            return RISP_OK;
        }));
        // ---- orthonormalise the corrections among themselves: Cholesky of their Gram matrix, twice; drop dependent ones
        {
            std::vector<int> keep(nb);
            for (int j = 0; j < nb; ++j) keep[j] = j;
            for (int rep = 0; rep < 2; ++rep) {
                std::vector<double> g;
                SOLVE_TRY(gram(S, S.dT, nb, S.dT, nb, g));
                // after projection the rows have norm <= 1; a row whose remaining norm is tiny is (numerically) inside span(V)
                std::vector<double> L((size_t)nb * nb, 0.0);
                std::vector<char> ok(nb, 1);
                for (int j = 0; j < nb; ++j) {
                    for (int i = j; i < nb; ++i) {
                        double s = g[(size_t)i * nb + j];
                        for (int c = 0; c < j; ++c) s -= L[(size_t)i * nb + c] * L[(size_t)j * nb + c];
                        if (i == j) {
                            if (!(s > (rep == 0 ? 1e-16 : 1e-4))) { ok[j] = 0; L[(size_t)j * nb + j] = 1.0; break; }
                            L[(size_t)j * nb + j] = std::sqrt(s);
                        } else L[(size_t)i * nb + j] = ok[j] ? s / L[(size_t)j * nb + j] : 0.0;
                    }
                    if (!ok[j]) for (int i = 0; i < nb; ++i) if (i != j) L[(size_t)i * nb + j] = 0.0;
                }
                // Linv (lower), rows of dropped vectors zeroed
                std::vector<double> Li((size_t)nb * nb, 0.0);
                for (int c = 0; c < nb; ++c) {
                    Li[(size_t)c * nb + c] = 1.0 / L[(size_t)c * nb + c];
                    for (int i = c + 1; i < nb; ++i) {
                        double s = 0.0;
                        for (int q = c; q < i; ++q) s += L[(size_t)i * nb + q] * Li[(size_t)q * nb + c];
                        Li[(size_t)i * nb + c] = -s / L[(size_t)i * nb + i];
                    }
                }
                std::vector<int> newkeep;
                std::vector<double> coef;
                int nk = 0;
                for (int j = 0; j < nb; ++j) if (ok[j]) ++nk;
                coef.assign((size_t)nk * nb, 0.0);
                int r = 0;
                for (int j = 0; j < nb; ++j) {
                    if (!ok[j]) continue;
                    for (int c = 0; c < nb; ++c) coef[(size_t)r * nb + c] = ok[c] ? Li[(size_t)j * nb + c] : 0.0;
                    newkeep.push_back(keep[j]);
                    ++r;
                }
                if (nk == 0) { nb = 0; break; }
                SOLVE_TRY(lincomb(S, coef, nk, nb, S.dT, S.dB, 1.0, 0.0));
                RISP_CUDA_TRY(cudaMemcpyAsync(S.dT, S.dB, (size_t)nk * dim * 8, cudaMemcpyDeviceToDevice, S.st));
                RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
                nb = nk; keep = newkeep;
            }
        }
        if (nb == 0) break;     // nothing new to add: stagnated
        RISP_CUDA_TRY(cudaMemcpyAsync(S.dB, S.dT, (size_t)nb * dim * 8, cudaMemcpyDeviceToDevice, S.st));
        RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
    }
    for (int j = 0; j < nroots; ++j) omega_out[j] = theta[j];
    if (X_out) RISP_CUDA_TRY(cudaMemcpy(X_out, S.dX, (size_t)nroots * dim * 8, cudaMemcpyDeviceToDevice));
    if (info) {
        std::memset(info, 0, sizeof(*info));
        info->iterations = iterations; info->restarts = restarts; info->n_sigma = n_sigma; info->converged = converged ? 1 : 0;
        for (int j = 0; j < nroots; ++j) info->resid[j] = rn[j];
        info->sec_total = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
        info->sec_matvec = sec_mv; info->sec_subspace = info->sec_total - sec_mv - sec_alloc; info->sec_alloc = sec_alloc;
        info->bytes_h2d = S.bytes_h2d; info->bytes_d2h = S.bytes_d2h; info->subspace_max = sub_max; info->cached_vectors = S.ncache;
    }
    cleanup();
    if (!converged) { risp_set_error(ctx, "risp_tda_solve: not converged within max_iter"); return RISP_ENOTCONV; }
    return RISP_OK;
}

// Debug export: the host eigen solver of the projected matrix (tests/test_host_logic.py pins it against LAPACK).
extern "C" int risp_debug_sym_eig(int n, const double *a_in, double *w_out, double *z_out)
{
    if (n <= 0 || !a_in || !w_out || !z_out) return RISP_EINVAL;
    std::vector<double> a(a_in, a_in + (size_t)n * n), w, z;
    sym_eig(a, n, w, z);
    std::memcpy(w_out, w.data(), (size_t)n * 8);
    std::memcpy(z_out, z.data(), (size_t)n * n * 8);
    return RISP_OK;
}

// Debug export: the lowest-nv variant used inside the Davidson loop.
extern "C" int risp_debug_sym_eig_lowest(int n, int nv, const double *a_in, double *w_out, double *z_out)
{
    if (n <= 0 || nv <= 0 || !a_in || !w_out || !z_out) return RISP_EINVAL;
    std::vector<double> a(a_in, a_in + (size_t)n * n), w, z;
    sym_eig_lowest(a, n, nv, w, z);
    std::memcpy(w_out, w.data(), (size_t)n * 8);
    std::memcpy(z_out, z.data(), (size_t)n * n * 8);
    return RISP_OK;
}
