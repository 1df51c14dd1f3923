// solve.cu -- risp_tda_solve: host-memory-assisted Davidson for the lowest roots of A X = X Omega (Eq. 9).
//
// Placement follows PAPER.md:189-201 (Fig. 2): the expansion vectors V and their images W = A V live in PINNED HOST memory and are
// "uploaded on demand"; when the subspace would outgrow its budget the solver restarts from the current Ritz vectors
// (reading G17: W <- W y by linearity, no extra sigma-build).  "Assisted" on a 180 GB part: whatever HBM is left
// after the K tensors, the matvec work space and the solver's own blocks caches the leading vectors of V and W on the device;
// only the vectors beyond that cache live in pinned host memory (page-locked piece by piece by a background thread) and are
// streamed over the host link on the side stream, double buffered against the compute stream -- none of them at 100-300 atoms,
// most of them at 3000 atoms, all of them with RISP_SOLVE_NO_CACHE.
//
// Device footprint of the solver itself: TWO blocks of `block` vectors (trial vectors / their images; between sigma-builds the
// same two buffers hold the Ritz vectors X = V y and A X = W y of a chunk of roots, then the residuals and corrections in
// place), two streaming buffers of CH vectors when a host part exists, and small scratch.  Roots are worked through in chunks
// of `block`, so the footprint does not grow with n_roots or n_guess: at 3000 atoms (1.06 GB per vector) block = 5 costs
// 10.6 GB + 8.5 GB of streaming buffers instead of the ~160 GB a 30-vector block with separate X / AX / residual / correction
// arrays would take.
//
// The Davidson recipe itself (guess, preconditioner, Gram-Schmidt) is the "standard" one of DESIGN.md reading G16.
#include "ctx.h"
#include <algorithm>
#include <atomic>
#include <chrono>
#include <cmath>
#include <thread>

void risp_sym_eig_lowest(std::vector<double> &a, int n, int nv, std::vector<double> &w, std::vector<double> &z);   // host_eig.cu

namespace {

// ------------------------------------------------------------------------------------------------ device kernels
__device__ __forceinline__ double hash_noise(unsigned long long seed, unsigned long long j, unsigned long long x)
{
    unsigned long long z = seed + 0x9E3779B97F4A7C15ull * (j + 1) + 0xD1B54A32D192ED03ull * (x + 1);      // splitmix64 finaliser
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    z ^= z >> 31;
    return (double)(z >> 11) * (2.0 / 9007199254740992.0) - 1.0;                                           // uniform in [-1, 1)
}

// V[j] = e_{idx[j]} (+ amp * seeded noise)
__global__ void guess_kernel(double *__restrict__ V, long long dim, const long long *__restrict__ idx, double amp, unsigned long long seed, int j0)
{
    const int j = blockIdx.y;
    const long long hot = idx[j];
    for (long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x; x < dim; x += (long long)gridDim.x * blockDim.x)
        V[j * dim + x] = (x == hot ? 1.0 : 0.0) + (amp != 0.0 ? amp * hash_noise(seed, (unsigned long long)(j0 + j), (unsigned long long)x) : 0.0);
}

// in place: AX[j] <- AX[j] - theta[j] X[j]; partial squared norms per block -> part[j][blockIdx.x]
__global__ void residual_kernel(const double *__restrict__ X, double *__restrict__ AX, const double *__restrict__ theta, long long dim,
                                double *__restrict__ part)
{
    const int j = blockIdx.y;
    const double th = theta[j];
    double s = 0.0;
    for (long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x; x < dim; x += (long long)gridDim.x * blockDim.x) {
        const double r = AX[j * dim + x] - th * X[j * dim + x];
        AX[j * dim + x] = r;
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

// t[dst] = r[src] / (theta - (eps_a - eps_i)), |denominator| floored at 1e-8 (sign kept); dst <= src, element-wise, so it may
// run in place.  One launch per vector, in ascending order: the compaction never overwrites a residual that is still needed.
__global__ void precondition_kernel(const double *r, double theta, const double *__restrict__ eps, int nocc, int nvir, double *t, long long rows)
{
    const double *ev = eps + nocc;
    for (long long i = blockIdx.x; i < rows; i += gridDim.x) {
        const double ei = eps[i];
        const double *src = r + i * nvir;
        double *dst = t + i * nvir;
        for (int a = threadIdx.x; a < nvir; a += blockDim.x) {
            double den = theta - (ev[a] - ei);
            if (fabs(den) < 1e-8) den = den < 0 ? -1e-8 : 1e-8;
            dst[a] = src[a] / den;
        }
    }
}

__global__ void scale_rows_kernel(double *__restrict__ T, long long dim, const double *__restrict__ scale)
{
    const int j = blockIdx.y;
    const double s = scale[j];
    for (long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x; x < dim; x += (long long)gridDim.x * blockDim.x) T[j * dim + x] *= s;
}

__global__ void reduce_partials_kernel(const double *__restrict__ part, int nz, int n, double *__restrict__ out)
{
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    double s = 0.0;
    for (int z = 0; z < nz; ++z) s += part[(long long)z * n + e];
    out[e] = s;
}

__global__ void f64_to_f32_kernel(const double *__restrict__ a, float *__restrict__ b, long long n)
{
    for (long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x; x < n; x += (long long)gridDim.x * blockDim.x) b[x] = (float)a[x];
}
__global__ void f32_to_f64_kernel(const float *__restrict__ a, double *__restrict__ b, long long n)
{
    for (long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x; x < n; x += (long long)gridDim.x * blockDim.x) b[x] = (double)a[x];
}
__global__ void round_to_f32_kernel(double *__restrict__ a, long long n)
{
    for (long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x; x < n; x += (long long)gridDim.x * blockDim.x) a[x] = (double)(float)a[x];
}

inline unsigned stream_grid(long long n) { return (unsigned)std::min<long long>((n + 255) / 256, 148 * 8); }

// ------------------------------------------------------------------------------------------------ pinned host store
// The host-resident part of V and W, in pieces of `pv` vectors that a background thread page-locks while the
// first sigma-builds run (pinning 7 GB takes ~2.7 s -- a fifth of a 300-atom solve if done up front).  esize = 8, or 4 with
// RISP_SOLVE_HOST_FP32.
struct HostStore {
    long long dim = 0;
    int pv = 32, npieces = 0, device = 0, slots = 0, esize = 8;
    std::vector<void *> v, w;
    std::atomic<int> ready{0}, failed{0}, stop{0};
    std::thread th;
    void start(int dev, long long dim_, int slots_, int esize_)
    {
        device = dev; dim = dim_; slots = slots_; esize = esize_;
        pv = (int)std::max<long long>(1, std::min<long long>(32, ((long long)2 << 30) / (dim * esize)));     // pieces of <= 2 GiB
        npieces = (slots + pv - 1) / pv;
        v.assign(npieces, nullptr); w.assign(npieces, nullptr);
        th = std::thread([this] {
            cudaSetDevice(device);
            for (int c = 0; c < npieces && !stop.load(); ++c) {
                const size_t nvec = (size_t)std::min(pv, slots - c * pv);
                if (cudaHostAlloc(&v[c], nvec * dim * esize, cudaHostAllocDefault) != cudaSuccess ||
                    cudaHostAlloc(&w[c], nvec * dim * esize, cudaHostAllocDefault) != cudaSuccess) { (void)cudaGetLastError(); failed.store(1); return; }
                ready.store(c + 1, std::memory_order_release);
            }
        });
    }
    // host address of vector i of V (isW = false) or W; blocks until its piece is pinned; nullptr if the allocation failed
    char *ptr(bool isW, long long i)
    {
        const int c = (int)(i / pv);
        while (ready.load(std::memory_order_acquire) <= c) {
            if (failed.load()) return nullptr;
            std::this_thread::yield();
        }
        return (char *)(isW ? w[c] : v[c]) + (i % pv) * dim * esize;
    }
    int run(long long i) const { return pv - (int)(i % pv); }     // vectors contiguous in memory from vector i on
    ~HostStore() { finish(); }
    void finish()
    {
        stop.store(1);
        if (th.joinable()) th.join();
        for (void *p : v) if (p) cudaFreeHost(p);
        for (void *p : w) if (p) cudaFreeHost(p);
        v.clear(); w.clear();
    }
};

// Everything the solver allocates; the destructor releases all of it, so every early return of risp_tda_solve is leak free.
struct Solver {
    risp_ctx *ctx = nullptr;
    long long dim = 0;
    int nroots = 0, block = 0, cap = 0, slots = 0, k = 0, CH = 16, ncache = 0;
    bool fp32_host = false;
    HostStore host;
    double *bufA = nullptr, *bufB = nullptr;           // the two blocks [block][dim]
    double *dChunk[2] = {nullptr, nullptr};            // FP64 streaming buffers [CH][dim] (FP32 mode: only [0], fed from dStage32)
    float *dStage32[2] = {nullptr, nullptr};           // FP32 mode: raw chunks as they arrive from the host [CH][dim]
    float *dStore32 = nullptr;                         // FP32 mode: a block converted for its way to the host [block][dim]
    double *dVc = nullptr, *dWc = nullptr;             // device cache of the first ncache subspace vectors [ncache][dim]
    long long slice = 16384;                           // split-K slice of the Gram products
    int nzmax = 0;
    std::vector<double> tmp;
    double *dCoef = nullptr, *dPart = nullptr, *dSmall = nullptr, *dTheta = nullptr;
    long long *dIdx = nullptr;
    cudaEvent_t evUp[2] = {nullptr, nullptr}, evFree[2] = {nullptr, nullptr}, evD2H = nullptr, evReady = nullptr;
    double bytes_h2d = 0, bytes_d2h = 0;
    cudaStream_t st = 0;                               // compute stream (default)
    std::vector<void *> owned;
    ~Solver()
    {
        cudaDeviceSynchronize();
        host.finish();
        for (void *p : owned) cudaFree(p);
        cudaEvent_t evs[] = {evUp[0], evUp[1], evFree[0], evFree[1], evD2H, evReady};
        for (cudaEvent_t e : evs) if (e) cudaEventDestroy(e);
    }
    template <class T>
    int alloc(T *&p, size_t count)
    {
        p = nullptr;
        if (count == 0) return RISP_OK;
        RISP_CUDA_TRY(cudaMalloc((void **)&p, count * sizeof(T)));
        owned.push_back(p);
        return RISP_OK;
    }
};

#define KERNEL_CHECK() RISP_CUDA_TRY(cudaGetLastError())

// out[na][nb] = sum_x A[i][x] B[j][x]; needs min(na, nb) <= 64 and max(na, nb) <= 128 (scratch size); callers chunk accordingly
int gram(Solver &S, const double *A, int na, const double *B, int nb, std::vector<double> &out)
{
    return risp_rows_gram(S.ctx, A, na, B, nb, S.dim, S.slice, S.dPart, S.dSmall, out, S.st);
}

// C[nc][dim] = alpha * coef[nc][na] * A[na][dim] + beta * C
int lincomb(Solver &S, const std::vector<double> &coef, int nc, int na, const double *A, double *C, double alpha, double beta)
{
    return risp_rows_lincomb(S.ctx, coef.data(), nc, na, A, C, S.dim, alpha, beta, S.dCoef, S.st);
}

// pass over subspace vectors [0, n): the first ncache come from the device cache (chunks of up to 128), the others are streamed
// from the pinned host store (V or W) in chunks of CH on the side stream; fn(dev_ptr, first, count) runs on the compute stream
template <class F>
int stream_pass(Solver &S, bool isW, int n, F &&fn)
{
    risp_ctx *ctx = S.ctx;
    int rc;
    const double *dc = isW ? S.dWc : S.dVc;
    const int nc = std::min(n, S.ncache);
    for (int first = 0; first < nc; first += 128)
        if ((rc = fn(dc + (long long)first * S.dim, first, std::min(128, nc - first)))) return rc;
    const int rest = n - nc;
    if (rest <= 0) return RISP_OK;
    const int nchunk = (rest + S.CH - 1) / S.CH;
    const int es = S.host.esize;
    auto upload = [&](int c) -> int {
        const int b = c & 1, first = nc + c * S.CH, cnt = std::min(S.CH, n - first);
        RISP_CUDA_TRY(cudaStreamWaitEvent(ctx->side, S.evFree[b], 0));
        char *dst = S.fp32_host ? (char *)S.dStage32[b] : (char *)S.dChunk[b];
        for (int done = 0; done < cnt;) {           // a chunk of CH vectors may straddle pinned pieces
            const long long i = first + done - S.ncache;
            const int seg = std::min(cnt - done, S.host.run(i));
            const char *h = S.host.ptr(isW, i);
            if (!h) { risp_set_error(ctx, "risp_tda_solve: pinned host allocation of the subspace failed"); return RISP_ENOMEM; }
            RISP_CUDA_TRY(cudaMemcpyAsync(dst + (size_t)done * S.dim * es, h, (size_t)seg * S.dim * es, cudaMemcpyHostToDevice, ctx->side));
            done += seg;
        }
        RISP_CUDA_TRY(cudaEventRecord(S.evUp[b], ctx->side));
        S.bytes_h2d += (double)cnt * S.dim * es;
        return RISP_OK;
    };
    if (nchunk > 0 && (rc = upload(0))) return rc;
    for (int c = 0; c < nchunk; ++c) {
        if (c + 1 < nchunk && (rc = upload(c + 1))) return rc;
        const int b = c & 1, first = nc + c * S.CH, cnt = std::min(S.CH, n - first);
        RISP_CUDA_TRY(cudaStreamWaitEvent(S.st, S.evUp[b], 0));
        const double *src = S.dChunk[b];
        if (S.fp32_host) {
            f32_to_f64_kernel<<<stream_grid((long long)cnt * S.dim), 256, 0, S.st>>>(S.dStage32[b], S.dChunk[0], (long long)cnt * S.dim);
            KERNEL_CHECK();
            RISP_CUDA_TRY(cudaEventRecord(S.evFree[b], S.st));    // the raw chunk is consumed; the FP64 copy is ordered on the compute stream
            src = S.dChunk[0];
        }
        if ((rc = fn(src, first, cnt))) return rc;
        if (!S.fp32_host) RISP_CUDA_TRY(cudaEventRecord(S.evFree[b], S.st));
    }
    return RISP_OK;
}

// store device vectors src[0, n) as subspace vectors [k, k+n): into the device cache while it reaches, beyond it into the pinned
// host store (side stream, after the compute stream has produced them).  The compute stream then waits for the copies, so the
// caller may overwrite src right away.
int store_vectors(Solver &S, bool isW, int k, const double *src, int n)
{
    risp_ctx *ctx = S.ctx;
    double *dc = isW ? S.dWc : S.dVc;
    const int nc = std::max(0, std::min(n, S.ncache - k));       // vectors that land in the device cache
    if (nc > 0) RISP_CUDA_TRY(cudaMemcpyAsync(dc + (long long)k * S.dim, src, (size_t)nc * S.dim * 8, cudaMemcpyDeviceToDevice, S.st));
    if (nc == n) return RISP_OK;
    const int es = S.host.esize;
    const char *from = (const char *)(src + (long long)nc * S.dim);
    if (S.fp32_host) {
        f64_to_f32_kernel<<<stream_grid((long long)(n - nc) * S.dim), 256, 0, S.st>>>(src + (long long)nc * S.dim, S.dStore32, (long long)(n - nc) * S.dim);
        KERNEL_CHECK();
        from = (const char *)S.dStore32;
    }
    RISP_CUDA_TRY(cudaEventRecord(S.evReady, S.st));
    RISP_CUDA_TRY(cudaStreamWaitEvent(ctx->side, S.evReady, 0));
    for (int done = nc; done < n;) {
        const long long i = k + done - S.ncache;
        const int seg = std::min(n - done, S.host.run(i));
        char *h = S.host.ptr(isW, i);
        if (!h) { risp_set_error(ctx, "risp_tda_solve: pinned host allocation of the subspace failed"); return RISP_ENOMEM; }
        RISP_CUDA_TRY(cudaMemcpyAsync(h, from + (size_t)(done - nc) * S.dim * es, (size_t)seg * S.dim * es, cudaMemcpyDeviceToHost, ctx->side));
        S.bytes_d2h += (double)seg * S.dim * es;
        done += seg;
    }
    RISP_CUDA_TRY(cudaEventRecord(S.evD2H, ctx->side));
    RISP_CUDA_TRY(cudaStreamWaitEvent(S.st, S.evD2H, 0));
    return RISP_OK;
}

// subspace vector `from` -> slot `to` (restart: the Ritz vectors parked in the tail slots become vectors 0 .. nroots-1);
// any combination of device cache and pinned host memory
int move_slot(Solver &S, bool isW, int from, int to)
{
    risp_ctx *ctx = S.ctx;
    double *dc = isW ? S.dWc : S.dVc;
    const bool fd = from < S.ncache, td = to < S.ncache;
    const size_t es = S.host.esize;
    if (fd && td) { RISP_CUDA_TRY(cudaMemcpyAsync(dc + (long long)to * S.dim, dc + (long long)from * S.dim, (size_t)S.dim * 8, cudaMemcpyDeviceToDevice, S.st)); return RISP_OK; }
    if (!fd && !td) {
        char *a = S.host.ptr(isW, from - S.ncache), *b = S.host.ptr(isW, to - S.ncache);
        if (!a || !b) { risp_set_error(ctx, "risp_tda_solve: pinned host allocation of the subspace failed"); return RISP_ENOMEM; }
        RISP_CUDA_TRY(cudaStreamSynchronize(ctx->side));
        std::memcpy(b, a, (size_t)S.dim * es);
        return RISP_OK;
    }
    // host tail slot -> device cache slot (the cache is the leading part, so the opposite direction does not occur)
    char *a = S.host.ptr(isW, from - S.ncache);
    if (!a) { risp_set_error(ctx, "risp_tda_solve: pinned host allocation of the subspace failed"); return RISP_ENOMEM; }
    RISP_CUDA_TRY(cudaStreamSynchronize(ctx->side));
    if (!S.fp32_host) { RISP_CUDA_TRY(cudaMemcpyAsync(dc + (long long)to * S.dim, a, (size_t)S.dim * 8, cudaMemcpyHostToDevice, S.st)); }
    else {
        RISP_CUDA_TRY(cudaMemcpyAsync(S.dStage32[0], a, (size_t)S.dim * 4, cudaMemcpyHostToDevice, S.st));
        f32_to_f64_kernel<<<stream_grid(S.dim), 256, 0, S.st>>>(S.dStage32[0], dc + (long long)to * S.dim, S.dim);
        KERNEL_CHECK();
    }
    S.bytes_h2d += (double)S.dim * es;
    RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
    return RISP_OK;
}

// dst[nc][dim] = sum_i y[first + i][c0 + j] * (V or W)[first + i]  over the whole subspace of size ky  (X = V y, A X = W y)
int ritz_vectors(Solver &S, bool isW, const std::vector<double> &yv, int ky, int ncol_y, int c0, int nc, double *dst)
{
    bool first_chunk = true;
    return stream_pass(S, isW, ky, [&](const double *Vc, int first, int cnt) -> int {
        std::vector<double> coef((size_t)nc * cnt);
        for (int j = 0; j < nc; ++j)
            for (int i = 0; i < cnt; ++i) coef[(size_t)j * cnt + i] = yv[(size_t)(first + i) * ncol_y + c0 + j];
        int r = lincomb(S, coef, nc, cnt, Vc, dst, 1.0, first_chunk ? 0.0 : 1.0);
        first_chunk = false;
        return r;
    });
}

// Orthonormalise the nb vectors in T against the stored subspace [0, S.k) and among themselves (reading G16: two passes of block
// Gram-Schmidt against V, Cholesky-based orthonormalisation inside the block, dependent vectors dropped).  `tmp` is a second
// block buffer; the result is back in T.  Returns the number of vectors kept through nb.
int orthonormalise(Solver &S, double *T, double *tmp, int &nb)
{
    risp_ctx *ctx = S.ctx;
    int rc;
    std::vector<double> g;
    // normalise first: the preconditioned residuals span many orders of magnitude
    {
        std::vector<double> sc(nb);
        for (int j0 = 0; j0 < nb; j0 += 64) {       // diagonal of the Gram matrix, block by block
            const int nj = std::min(64, nb - j0);
            if ((rc = gram(S, T + (long long)j0 * S.dim, nj, T + (long long)j0 * S.dim, nj, g))) return rc;
            for (int j = 0; j < nj; ++j) { const double n2 = g[(size_t)j * nj + j]; sc[j0 + j] = n2 > 0 ? 1.0 / std::sqrt(n2) : 0.0; }
        }
        RISP_CUDA_TRY(cudaMemcpyAsync(S.dTheta, sc.data(), (size_t)nb * 8, cudaMemcpyHostToDevice, S.st));
        scale_rows_kernel<<<dim3(stream_grid(S.dim), nb), 256, 0, S.st>>>(T, S.dim, S.dTheta);
        KERNEL_CHECK();
        RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
    }
    if ((rc = stream_pass(S, false, S.k, [&](const double *Vc, int first, int cnt) -> int {
            for (int rep = 0; rep < 2; ++rep) {
                std::vector<double> c;
                int r = gram(S, T, nb, Vc, cnt, c);       // c[j][i] = t_j . v_i
                if (r) return r;
                r = lincomb(S, c, nb, cnt, Vc, T, -1.0, 1.0);
                if (r) return r;
            }
            return RISP_OK;
        }))) return rc;
    double *cur = T, *oth = tmp;
    for (int rep = 0; rep < 2; ++rep) {
        if ((rc = gram(S, cur, nb, cur, nb, g))) return rc;
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
        std::vector<double> Li((size_t)nb * nb, 0.0);       // L^-1 (lower)
        for (int c = 0; c < nb; ++c) {
            Li[(size_t)c * nb + c] = 1.0 / L[(size_t)c * nb + c];
            for (int i = c + 1; i < nb; ++i) {
                double s = 0.0;
                for (int q = c; q < i; ++q) s += L[(size_t)i * nb + q] * Li[(size_t)q * nb + c];
                Li[(size_t)i * nb + c] = -s / L[(size_t)i * nb + i];
            }
        }
        int nk = 0;
        for (int j = 0; j < nb; ++j) if (ok[j]) ++nk;
        if (nk == 0) { nb = 0; return RISP_OK; }
        std::vector<double> coef((size_t)nk * nb, 0.0);
        int r = 0;
        for (int j = 0; j < nb; ++j) {
            if (!ok[j]) continue;
            for (int c = 0; c < nb; ++c) coef[(size_t)r * nb + c] = ok[c] ? Li[(size_t)j * nb + c] : 0.0;
            ++r;
        }
        if ((rc = lincomb(S, coef, nk, nb, cur, oth, 1.0, 0.0))) return rc;
        std::swap(cur, oth);
        nb = nk;
    }
    // two swaps: the result is back in T
    return RISP_OK;
}

}  // namespace

// ---- dense row-block products shared by the TDA and the TDDFT solver (declared in ctx.h)
// out[na][nb] = sum_x A[i][x] B[j][x]: split-K batched DMMA GEMM + fixed-order reduction.  The smaller operand goes to the M side
// (16-row tiles exist, the N tile is always 128 wide); the product is HBM-bound: it reads (na + nb) dim doubles.
// dPart: [dim / slice + 2][128 * 64] doubles, dSmall: [128 * 64].
int risp_rows_gram(risp_ctx *ctx, const double *A, int na, const double *B, int nb, long long dim, long long slice, double *dPart, double *dSmall,
                   std::vector<double> &out, cudaStream_t st)
{
    const bool swap = na > nb;
    const double *P = swap ? B : A, *Q = swap ? A : B;
    const int np = swap ? nb : na, nq = swap ? na : nb;
    if (np > 64 || nq > 128) { risp_set_error(ctx, "risp solver: internal Gram block too large"); return RISP_EINVAL; }
    int nfull = (int)(dim / slice);
    long long tail = dim - (long long)nfull * slice;
    int nz = nfull + (tail ? 1 : 0);
    if (nfull) {
        GemmDesc d = gemm_desc(np, nq, (int)slice, P, dim, true, Q, dim, true, dPart, nq);
        d.nb1 = nfull; d.sA1 = slice; d.sB1 = slice; d.sC1 = (long long)np * nq;
        RISP_CUDA_TRY(risp_dgemm(d, st));
    }
    if (tail) {
        GemmDesc d = gemm_desc(np, nq, (int)tail, P + (long long)nfull * slice, dim, true, Q + (long long)nfull * slice, dim, true,
                               dPart + (long long)nfull * np * nq, nq);
        RISP_CUDA_TRY(risp_dgemm(d, st));
    }
    reduce_partials_kernel<<<(np * nq + 127) / 128, 128, 0, st>>>(dPart, nz, np * nq, dSmall);
    RISP_CUDA_TRY(cudaGetLastError());
    out.resize((size_t)na * nb);
    if (!swap) {
        RISP_CUDA_TRY(cudaMemcpyAsync(out.data(), dSmall, (size_t)na * nb * 8, cudaMemcpyDeviceToHost, st));
        RISP_CUDA_TRY(cudaStreamSynchronize(st));
    } else {
        std::vector<double> tmp((size_t)na * nb);
        RISP_CUDA_TRY(cudaMemcpyAsync(tmp.data(), dSmall, (size_t)na * nb * 8, cudaMemcpyDeviceToHost, st));
        RISP_CUDA_TRY(cudaStreamSynchronize(st));
        for (int i = 0; i < na; ++i)
            for (int j = 0; j < nb; ++j) out[(size_t)i * nb + j] = tmp[(size_t)j * na + i];
    }
    return RISP_OK;
}

int risp_rows_lincomb(risp_ctx *ctx, const double *coef_host, int nc, int na, const double *A, double *C, long long dim, double alpha, double beta,
                      double *dCoef, cudaStream_t st)
{
    RISP_CUDA_TRY(cudaMemcpyAsync(dCoef, coef_host, (size_t)nc * na * 8, cudaMemcpyHostToDevice, st));
    GemmDesc d = gemm_desc(nc, (int)std::min<long long>(dim, 1 << 30), na, dCoef, na, true, A, dim, false, C, dim, alpha, beta);
    RISP_CUDA_TRY(risp_dgemm(d, st));
    RISP_CUDA_TRY(cudaStreamSynchronize(st));   // coef is a host temporary
    return RISP_OK;
}

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
    const int max_sub = std::max(opt.max_sub > 0 ? opt.max_sub : 20 * nroots, 2 * nroots);
    auto t_start = std::chrono::steady_clock::now();
    double sec_mv = 0.0;
    int rc;

    Solver S;
    S.ctx = ctx; S.dim = dim; S.nroots = nroots;
    S.fp32_host = (opt.flags & RISP_SOLVE_HOST_FP32) != 0;
    const size_t vec = (size_t)dim * 8;

    // ---------------- block size and memory plan
    // the staging copies of risp_matvec_host are not needed here and are re-created on demand
    if (ctx->w_Xin) { cudaFree(ctx->w_Xin); ctx->w_Xin = nullptr; }
    if (ctx->w_Sout) { cudaFree(ctx->w_Sout); ctx->w_Sout = nullptr; }
    ctx->xin_cap = 0;
    int block = std::min(std::min(std::max(n_guess, nroots), RISP_MS), ctx->max_batch);
    if (opt.max_block > 0) block = std::min(block, opt.max_block);
    block = std::max(block, 1);
    if ((rc = risp_ensure_workspace(ctx, block))) return rc;
    S.slice = dim > (1 << 20) ? std::max<long long>(4096, ((dim / 1024) + 4095) / 4096 * 4096) : 16384;   // ~1000 slices: every SM has tiles
    S.nzmax = (int)(dim / S.slice) + 2;
    const size_t small_bytes = ((size_t)S.nzmax * 128 * 64 + 128 * 64 + 4096) * 8 + ((size_t)1 << 20);
    size_t hostvec_bytes = S.fp32_host ? (size_t)dim * 4 : vec;
    const long long host_vecs = (long long)(ctx->host_budget / (2 * hostvec_bytes));
    {
        size_t free_b = 0, total_b = 0;
        RISP_CUDA_TRY(cudaMemGetInfo(&free_b, &total_b));
        size_t room;
        if (opt.device_budget_bytes) room = std::min(opt.device_budget_bytes, free_b);
        else { const size_t keep = std::min<size_t>((size_t)1 << 30, free_b / 8); room = (size_t)(0.9 * (double)(free_b - keep)); }
        const long long want = (long long)max_sub + nroots;
        const long long dev_limit = (opt.flags & RISP_SOLVE_NO_CACHE) ? 0 : ((opt.flags & RISP_SOLVE_TINY_CACHE) ? nroots + 2 : (1ll << 40));
        for (;; block = (block + 1) / 2) {
            const size_t fixed = 2 * (size_t)block * vec + small_bytes + (size_t)(want + 64) * (want + 64) * 8;
            if (fixed <= room) {
                const size_t left = room - fixed;
                if (dev_limit >= want && (size_t)want * 2 * vec <= left) { S.slots = (int)want; S.ncache = (int)want; S.CH = 0; break; }      // all of V, W in HBM
                S.CH = vec >= ((size_t)1 << 30) ? 2 : (vec >= ((size_t)256 << 20) ? 4 : 16);      // >= 1 GiB per H2D copy either way
                const size_t stream_bytes = 2 * (size_t)S.CH * vec + (S.fp32_host ? (size_t)block * dim * 4 : 0);
                if (stream_bytes <= left) {
                    const long long dev_vecs = std::min<long long>(dev_limit, (long long)((left - stream_bytes) / (2 * vec)));
                    const long long slots = std::min(want, dev_vecs + host_vecs);
                    if (slots >= 3ll * nroots) { S.slots = (int)slots; S.ncache = (int)std::min(slots, dev_vecs); break; }
                }
            }
            if (block == 1) {
                risp_set_error(ctx, "risp_tda_solve: device memory / pinned-host budget too small for two single-vector blocks, the streaming buffers and a subspace of 3 n_roots vectors");
                return RISP_ENOMEM;
            }
        }
    }
    S.block = block; S.cap = S.slots - nroots;
    n_guess = std::min(n_guess, S.cap);
    if ((rc = risp_ensure_workspace(ctx, block))) return rc;
    if ((rc = S.alloc(S.bufA, (size_t)block * dim)) || (rc = S.alloc(S.bufB, (size_t)block * dim))) return rc;
    if ((rc = S.alloc(S.dPart, std::max((size_t)S.nzmax * 128 * 64, (size_t)RISP_MAX_ROOTS * 256))) || (rc = S.alloc(S.dSmall, (size_t)128 * 64)) ||
        (rc = S.alloc(S.dTheta, (size_t)RISP_MAX_ROOTS)) || (rc = S.alloc(S.dIdx, (size_t)RISP_MS)) ||
        (rc = S.alloc(S.dCoef, (size_t)std::max(S.slots, 128) * std::max(S.slots, 128))))
        return rc;
    if (S.slots > S.ncache) {
        if (!S.fp32_host) { if ((rc = S.alloc(S.dChunk[0], (size_t)S.CH * dim)) || (rc = S.alloc(S.dChunk[1], (size_t)S.CH * dim))) return rc; }
        else {
            if ((rc = S.alloc(S.dChunk[0], (size_t)S.CH * dim)) || (rc = S.alloc(S.dStage32[0], (size_t)S.CH * dim)) ||
                (rc = S.alloc(S.dStage32[1], (size_t)S.CH * dim)) || (rc = S.alloc(S.dStore32, (size_t)block * dim)))
                return rc;
        }
        S.host.start(ctx->device, dim, S.slots - S.ncache, S.fp32_host ? 4 : 8);
    }
    if (S.ncache > 0) { if ((rc = S.alloc(S.dVc, (size_t)S.ncache * dim)) || (rc = S.alloc(S.dWc, (size_t)S.ncache * dim))) return rc; }
    for (int b = 0; b < 2; ++b) { RISP_CUDA_TRY(cudaEventCreateWithFlags(&S.evUp[b], cudaEventDisableTiming)); RISP_CUDA_TRY(cudaEventCreateWithFlags(&S.evFree[b], cudaEventDisableTiming)); }
    RISP_CUDA_TRY(cudaEventCreateWithFlags(&S.evD2H, cudaEventDisableTiming));
    RISP_CUDA_TRY(cudaEventCreateWithFlags(&S.evReady, cudaEventDisableTiming));

    std::vector<double> G;          // projected matrix, row-major with leading dimension ldg
    const int ldg = S.slots;
    G.assign((size_t)ldg * ldg, 0.0);
    std::vector<double> theta(nroots, 0.0), rn(nroots, 0.0), yv;
    int iterations = 0, restarts = 0, n_sigma = 0, sub_max = 0, ky = 0;
    bool converged = false;
    S.k = 0;

    // W_B = A B for the nb vectors in Bbuf (image into Wbuf), projected matrix extended, both appended to the subspace
    auto append_block = [&](double *Bbuf, double *Wbuf, int nb) -> int {
        int r;
        if (S.fp32_host) {      // V must be stored exactly: round the trial vectors before their images are computed
            round_to_f32_kernel<<<stream_grid((long long)nb * dim), 256, 0, S.st>>>(Bbuf, (long long)nb * dim);
            KERNEL_CHECK();
        }
        auto t0 = std::chrono::steady_clock::now();
        if ((r = risp_matvec_impl(ctx, nb, Bbuf, Wbuf, S.st))) return r;
        RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
        sec_mv += std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
        n_sigma += nb;
        const int k = S.k;
        std::vector<double> blk;
        // G[0:k][k:k+nb] = V_old^T W_B (stream V_old), G[k:, k:] = B^T W_B symmetrised
        if ((r = stream_pass(S, false, k, [&](const double *Vc, int first, int cnt) -> int {
                int q = gram(S, Vc, cnt, Wbuf, nb, blk);
                if (q) return q;
                for (int i = 0; i < cnt; ++i)
                    for (int j = 0; j < nb; ++j) G[(size_t)(first + i) * ldg + k + j] = G[(size_t)(k + j) * ldg + first + i] = blk[(size_t)i * nb + j];
                return RISP_OK;
            }))) return r;
        if ((r = gram(S, Bbuf, nb, Wbuf, nb, blk))) return r;
        for (int i = 0; i < nb; ++i)
            for (int j = 0; j < nb; ++j) G[(size_t)(k + i) * ldg + k + j] = 0.5 * (blk[(size_t)i * nb + j] + blk[(size_t)j * nb + i]);
        if ((r = store_vectors(S, false, k, Bbuf, nb))) return r;
        if ((r = store_vectors(S, true, k, Wbuf, nb))) return r;
        S.k += nb;
        sub_max = std::max(sub_max, S.k);
        return RISP_OK;
    };

    const double sec_alloc = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();

    // ---------------- initial guess: unit vectors on the smallest eps_a - eps_i, block by block
    {
        std::vector<std::pair<double, long long>> dl;
        const int no_top = (int)std::min<long long>(ctx->nocc, n_guess), nv_bot = (int)std::min<long long>(ctx->nvir, n_guess);
        for (int i = ctx->nocc - no_top; i < ctx->nocc; ++i)
            for (int a = 0; a < nv_bot; ++a) dl.push_back({ctx->h_eps[ctx->nocc + a] - ctx->h_eps[i], (long long)i * ctx->nvir + a});
        std::stable_sort(dl.begin(), dl.end(), [](auto &x, auto &y) { return x.first < y.first || (x.first == y.first && x.second < y.second); });
        const bool perturbed = (opt.flags & RISP_SOLVE_PERTURBED_GUESS) != 0;
        const double amp = perturbed ? 0.3 * std::sqrt(3.0 / (double)dim) : 0.0;     // uniform noise in [-amp, amp): norm 0.3
        for (int g0 = 0; g0 < n_guess; g0 += block) {
            int nb = std::min(block, n_guess - g0);
            std::vector<long long> idx(nb);
            for (int j = 0; j < nb; ++j) idx[j] = dl[g0 + j].second;
            RISP_CUDA_TRY(cudaMemcpyAsync(S.dIdx, idx.data(), (size_t)nb * sizeof(long long), cudaMemcpyHostToDevice, S.st));
            guess_kernel<<<dim3(stream_grid(dim), nb), 256, 0, S.st>>>(S.bufA, dim, S.dIdx, amp, 0x5EEDull + 977ull * (unsigned long long)nroots, g0);
            KERNEL_CHECK();
            RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
            if (perturbed && (rc = orthonormalise(S, S.bufA, S.bufB, nb))) return rc;
            if (nb > 0 && (rc = append_block(S.bufA, S.bufB, nb))) return rc;
        }
    }

    int n_unconv_prev = nroots;
    for (int it = 1; it <= max_iter; ++it) {
        iterations = it;
        // ---- Ritz pairs of the projected matrix
        const int k = S.k;
        {
            std::vector<double> a((size_t)k * k), w;
            for (int i = 0; i < k; ++i)
                for (int j = 0; j < k; ++j) a[(size_t)i * k + j] = G[(size_t)i * ldg + j];
            risp_sym_eig_lowest(a, k, nroots, w, yv);
            for (int j = 0; j < nroots; ++j) theta[j] = w[j];
            ky = k;
        }
        // ---- restart from the Ritz vectors when the corrections of this iteration would not fit: X and A X of all
        //      roots are parked in the tail slots chunk by chunk, then become vectors 0 .. nroots-1
        if (k > nroots && k + std::min(n_unconv_prev, nroots) > S.cap) {
            for (int c0 = 0; c0 < nroots; c0 += block) {
                const int nc = std::min(block, nroots - c0);
                if ((rc = ritz_vectors(S, false, yv, ky, ky, c0, nc, S.bufA))) return rc;
                if ((rc = ritz_vectors(S, true, yv, ky, ky, c0, nc, S.bufB))) return rc;
                if ((rc = store_vectors(S, false, S.cap + c0, S.bufA, nc))) return rc;
                if ((rc = store_vectors(S, true, S.cap + c0, S.bufB, nc))) return rc;
            }
            RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
            for (int j = 0; j < nroots; ++j) {
                if ((rc = move_slot(S, false, S.cap + j, j))) return rc;
                if ((rc = move_slot(S, true, S.cap + j, j))) return rc;
            }
            RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
            std::fill(G.begin(), G.end(), 0.0);
            for (int j = 0; j < nroots; ++j) G[(size_t)j * ldg + j] = theta[j];
            S.k = nroots; ky = nroots;
            yv.assign((size_t)nroots * nroots, 0.0);
            for (int j = 0; j < nroots; ++j) yv[(size_t)j * nroots + j] = 1.0;
            ++restarts;
        }
        // ---- per chunk of roots: X = V y, A X = W y, residual, correction, orthonormalisation, sigma-build, append
        int n_unconv = 0, appended = 0;
        for (int c0 = 0; c0 < nroots; c0 += block) {
            const int nc = std::min(block, nroots - c0);
            if ((rc = ritz_vectors(S, false, yv, ky, ky, c0, nc, S.bufA))) return rc;
            if ((rc = ritz_vectors(S, true, yv, ky, ky, c0, nc, S.bufB))) return rc;
            RISP_CUDA_TRY(cudaMemcpyAsync(S.dTheta, theta.data() + c0, (size_t)nc * 8, cudaMemcpyHostToDevice, S.st));
            const int gx = 256;
            residual_kernel<<<dim3(gx, nc), 256, 0, S.st>>>(S.bufA, S.bufB, S.dTheta, dim, S.dPart);
            KERNEL_CHECK();
            std::vector<double> part((size_t)nc * gx);
            RISP_CUDA_TRY(cudaMemcpyAsync(part.data(), S.dPart, part.size() * 8, cudaMemcpyDeviceToHost, S.st));
            RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
            std::vector<int> src;
            for (int j = 0; j < nc; ++j) {
                double s = 0.0;
                for (int b = 0; b < gx; ++b) s += part[(size_t)j * gx + b];
                rn[c0 + j] = std::sqrt(s);
                if (!(rn[c0 + j] < tol)) src.push_back(j);
            }
            n_unconv += (int)src.size();
            if (src.empty() || it == max_iter) continue;
            int nb = std::min((int)src.size(), S.cap - S.k);     // no room left: the rest waits for the restart of the next iteration
            if (nb <= 0) continue;
            // corrections t_j = r_j / (theta_j - Delta), compacted to the front of bufB (ascending, in place)
            for (int j = 0; j < nb; ++j) {
                precondition_kernel<<<(unsigned)std::min<long long>(ctx->nocc, 148 * 16), 256, 0, S.st>>>(
                    S.bufB + (long long)src[j] * dim, theta[c0 + src[j]], ctx->d_eps, ctx->nocc, ctx->nvir, S.bufB + (long long)j * dim, ctx->nocc);
                KERNEL_CHECK();
            }
            if ((rc = orthonormalise(S, S.bufB, S.bufA, nb))) return rc;
            if (nb == 0) continue;
            if ((rc = append_block(S.bufB, S.bufA, nb))) return rc;
            appended += nb;
        }
        n_unconv_prev = n_unconv;
        if (opt.flags & RISP_SOLVE_LOG_STDERR) {
            double rmax = 0.0;
            for (int j = 0; j < nroots; ++j) rmax = std::max(rmax, rn[j]);
            std::fprintf(stderr, "[risp_tda_solve] it %d  subspace %d  unconverged %d  max residual %.3e  omega_1 %.8f Ha  sigma-builds %d  restarts %d  %.1f s\n", it, S.k,
                         n_unconv, rmax, theta[0], n_sigma, restarts, std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count());
            std::fflush(stderr);
        }
        if (n_unconv == 0) { converged = true; break; }
        if (it == max_iter) break;
        if (opt.max_seconds > 0 && std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count() > (double)opt.max_seconds) break;
        if (appended == 0 && S.k < S.cap) break;     // nothing new to add although there is room: stagnated
    }
    for (int j = 0; j < nroots; ++j) omega_out[j] = theta[j];
    if (X_out) {
        // X_out may be as large as the solver's own blocks: built chunk by chunk through bufA
        for (int c0 = 0; c0 < nroots; c0 += block) {
            const int nc = std::min(block, nroots - c0);
            if ((rc = ritz_vectors(S, false, yv, ky, ky, c0, nc, S.bufA))) return rc;
            RISP_CUDA_TRY(cudaMemcpyAsync(X_out + (long long)c0 * dim, S.bufA, (size_t)nc * dim * 8,
                                          (opt.flags & RISP_SOLVE_X_OUT_HOST) ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, S.st));
            RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
        }
        RISP_CUDA_TRY(cudaStreamSynchronize(S.st));
    }
    if (info) {
        std::memset(info, 0, sizeof(*info));
        info->iterations = iterations; info->restarts = restarts; info->n_sigma = n_sigma; info->converged = converged ? 1 : 0;
        for (int j = 0; j < nroots; ++j) info->resid[j] = rn[j];
        info->sec_total = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
        info->sec_matvec = sec_mv; info->sec_subspace = info->sec_total - sec_mv - sec_alloc; info->sec_alloc = sec_alloc;
        info->bytes_h2d = S.bytes_h2d; info->bytes_d2h = S.bytes_d2h; info->subspace_max = sub_max; info->cached_vectors = S.ncache;
        info->block = block; info->capacity = S.slots;
        info->bytes_host_subspace = (double)(S.slots - S.ncache) * 2.0 * (double)hostvec_bytes;
    }
    if (!converged) { risp_set_error(ctx, "risp_tda_solve: not converged within max_iter"); return RISP_ENOTCONV; }
    return RISP_OK;
}
