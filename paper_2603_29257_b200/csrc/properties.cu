// properties.cu -- risp_transition_properties: transition dipoles, oscillator and rotatory strengths of TDA states
// (Eq. 5-8; in TDA Y = 0).
//
//   mu_0n = scale sum_ia r_ia X_nia                (Eq. 7)        f_0n = 2/3 Omega_n mu_0n . mu_0n     (Eq. 5)
//   m_0n  = scale sum_ia (r x nabla)_ia X_nia      (Eq. 8)        R_0n = 1/2 mu_0n . m_0n              (Eq. 6)
//
// One-electron integrals only: per operator component the AO matrix is filled on the kept shell pairs by the Obara-Saika
// overlap recursion (one thread per shell pair; moments through x - O = (x - A) + (A - O), the gradient acting on the ket through
// d/dx [x_B^j e^{-b x_B^2}] = j x_B^{j-1} e^{..} - 2b x_B^{j+1} e^{..}), transformed to the occupied-virtual block by two DMMA
// GEMMs, and contracted with all n vectors by one split-K GEMM with a fixed-order reduction.  Nothing is kept between calls
// except the small shell table.
#include "ctx.h"
#include <algorithm>
#include <cmath>

using namespace risp_eri;

namespace {

struct OneShell { double x, y, z; int l, nprim, poff, ao; };

// 1D overlaps S[i][j] = <x_A^i e^{-a x_A^2} | x_B^j e^{-b x_B^2}>, i <= IA, j <= JB (Obara-Saika)
template <int IA, int JB>
__device__ __forceinline__ void overlap_1d(double p, double hp, double PA, double PB, double s00, double (&S)[IA + 1][JB + 1])
{
    S[0][0] = s00;
#pragma unroll
    for (int i = 0; i < IA; ++i) S[i + 1][0] = PA * S[i][0] + (i > 0 ? i * hp * S[i - 1][0] : 0.0);
#pragma unroll
    for (int j = 0; j < JB; ++j)
#pragma unroll
        for (int i = 0; i <= IA; ++i)
            S[i][j + 1] = PB * S[i][j] + (i > 0 ? i * hp * S[i - 1][j] : 0.0) + (j > 0 ? j * hp * S[i][j - 1] : 0.0);
    (void)p;
}

__device__ __forceinline__ void cart_exps(int l, int k, int (&e)[3])
{
    // cidx order of eri.cuh within one degree: (ex, ey, ez) with ex descending, then ey descending
    int c = 0;
    for (int ex = l; ex >= 0; --ex)
        for (int ey = l - ex; ey >= 0; --ey, ++c)
            if (c == k) { e[0] = ex; e[1] = ey; e[2] = l - ex - ey; return; }
}

// AO matrix of ONE operator component comp (0-2: (r-O)_k, 3-5: ((r-O) x nabla)_k) on the kept pairs of one class; the mirror image
// carries the sign of the operator's symmetry (+ for r, - for r x nabla)
template <int LA, int LB>
__global__ void __launch_bounds__(128) oneel_kernel(const ShellPair *__restrict__ pairs, int npairs, const OneShell *__restrict__ shl,
                                                    const double *__restrict__ pexp, const double *__restrict__ pd, int comp, double Ox, double Oy,
                                                    double Oz, double *__restrict__ out, long long ld)
{
    const int pi = blockIdx.x * blockDim.x + threadIdx.x;
    if (pi >= npairs) return;
    const ShellPair sp = pairs[pi];
    const OneShell A = shl[sp.shA], B = shl[sp.shB];
    constexpr int NA = ncart(LA), NB = ncart(LB);
    double cart[NA][NB];
#pragma unroll
    for (int i = 0; i < NA; ++i)
#pragma unroll
        for (int j = 0; j < NB; ++j) cart[i][j] = 0.0;
    const double Ac[3] = {A.x, A.y, A.z}, Bc[3] = {B.x, B.y, B.z}, O[3] = {Ox, Oy, Oz};
    const double R2 = sp.ABx * sp.ABx + sp.ABy * sp.ABy + sp.ABz * sp.ABz;
    const int k = comp % 3, k1 = (k + 1) % 3, k2 = (k + 2) % 3;      // L_k = r_k1 d_k2 - r_k2 d_k1
    for (int ka = 0; ka < A.nprim; ++ka)
        for (int kb = 0; kb < B.nprim; ++kb) {
            const double a = pexp[A.poff + ka], b = pexp[B.poff + kb], p = a + b, ip = 1.0 / p, hp = 0.5 * ip;
            const double pre = pd[A.poff + ka] * pd[B.poff + kb] * exp(-a * b * ip * R2);
            const double s00 = sqrt(3.14159265358979323846 * ip);
            double S[3][LA + 2][LB + 2];
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const double P = (a * Ac[d] + b * Bc[d]) * ip;
                overlap_1d<LA + 1, LB + 1>(p, hp, P - Ac[d], P - Bc[d], s00, S[d]);
            }
#pragma unroll
            for (int x = 0; x < NA; ++x)
#pragma unroll
                for (int y = 0; y < NB; ++y) {
                    int u[3], v[3];
                    cart_exps(LA, x, u); cart_exps(LB, y, v);
                    auto Sd = [&](int d) { return S[d][u[d]][v[d]]; };
                    auto Md = [&](int d) { return S[d][u[d] + 1][v[d]] + (Ac[d] - O[d]) * S[d][u[d]][v[d]]; };
                    auto Dd = [&](int d) { return (v[d] > 0 ? v[d] * S[d][u[d]][v[d] - 1] : 0.0) - 2.0 * b * S[d][u[d]][v[d] + 1]; };
                    double val;
                    if (comp < 3) val = Md(k) * Sd(k1) * Sd(k2);
                    else val = Sd(k) * (Md(k1) * Dd(k2) - Dd(k1) * Md(k2));
                    cart[x][y] = fma(pre, val, cart[x][y]);
                }
        }
    const double sign = comp < 3 ? 1.0 : -1.0;
#pragma unroll
    for (int i = 0; i < 2 * LA + 1; ++i)
#pragma unroll
        for (int j = 0; j < 2 * LB + 1; ++j) {
            double s = 0.0;
#pragma unroll
            for (int x = 0; x < NA; ++x)
#pragma unroll
                for (int y = 0; y < NB; ++y) {
                    const double c = sph_coef(LA, i, x) * sph_coef(LB, j, y);
                    if (c != 0.0) s = fma(c, cart[x][y], s);
                }
            out[(long long)(sp.aoA + i) * ld + sp.aoB + j] = s;
            if (sp.shA != sp.shB) out[(long long)(sp.aoB + j) * ld + sp.aoA + i] = sign * s;
        }
}

__global__ void reduce_slices_kernel(const double *__restrict__ part, int nz, int n, double *__restrict__ out)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    double s = 0.0;
    for (int z = 0; z < nz; ++z) s += part[(long long)z * n + e];
    out[e] = s;
}

template <class F>
void dispatch(int la, int lb, F &&f)
{
    if (la == 0) f(std::integral_constant<int, 0>{}, std::integral_constant<int, 0>{});
    else if (la == 1 && lb == 0) f(std::integral_constant<int, 1>{}, std::integral_constant<int, 0>{});
    else if (la == 1) f(std::integral_constant<int, 1>{}, std::integral_constant<int, 1>{});
    else if (lb == 0) f(std::integral_constant<int, 2>{}, std::integral_constant<int, 0>{});
    else if (lb == 1) f(std::integral_constant<int, 2>{}, std::integral_constant<int, 1>{});
    else f(std::integral_constant<int, 2>{}, std::integral_constant<int, 2>{});
}

// the shell table of the one-electron kernel (uploaded once per context)
int ensure_shell_table(risp_ctx *ctx)
{
    if (ctx->d_oneel_shl) return RISP_OK;
    std::vector<OneShell> h(ctx->nshl);
    for (int s = 0; s < ctx->nshl; ++s) {
        const int at = ctx->h_shl_atom[s];
        h[s] = OneShell{ctx->h_xyz[3 * at], ctx->h_xyz[3 * at + 1], ctx->h_xyz[3 * at + 2], ctx->h_shl_l[s], ctx->h_shl_nprim[s], ctx->h_shl_poff[s], ctx->h_shl_ao[s]};
    }
    RISP_CUDA_TRY(cudaMalloc(&ctx->d_oneel_shl, h.size() * sizeof(OneShell)));
    RISP_CUDA_TRY(cudaMemcpy(ctx->d_oneel_shl, h.data(), h.size() * sizeof(OneShell), cudaMemcpyHostToDevice));
    RISP_CUDA_TRY(cudaMalloc((void **)&ctx->d_prim_exp, ctx->h_prim_exp.size() * 8));
    RISP_CUDA_TRY(cudaMalloc((void **)&ctx->d_prim_d, ctx->h_prim_d.size() * 8));
    RISP_CUDA_TRY(cudaMemcpy(ctx->d_prim_exp, ctx->h_prim_exp.data(), ctx->h_prim_exp.size() * 8, cudaMemcpyHostToDevice));
    RISP_CUDA_TRY(cudaMemcpy(ctx->d_prim_d, ctx->h_prim_d.data(), ctx->h_prim_d.size() * 8, cudaMemcpyHostToDevice));
    return RISP_OK;
}

int fill_component(risp_ctx *ctx, int comp, const double *O, double *ao, cudaStream_t st)
{
    RISP_CUDA_TRY(cudaMemsetAsync(ao, 0, (size_t)ctx->nao * ctx->ldao * 8, st));
    for (int c = 0; c < 6; ++c) {
        const PairClass &pc = ctx->cls[c];
        if (!pc.npairs) continue;
        dispatch(pc.la, pc.lb, [&](auto LA, auto LB) {
            oneel_kernel<decltype(LA)::value, decltype(LB)::value><<<(pc.npairs + 127) / 128, 128, 0, st>>>(
                pc.d_pairs, pc.npairs, (const OneShell *)ctx->d_oneel_shl, ctx->d_prim_exp, ctx->d_prim_d, comp, O[0], O[1], O[2], ao, ctx->ldao);
        });
        RISP_CUDA_TRY(cudaGetLastError());
    }
    return RISP_OK;
}

}  // namespace

extern "C" int risp_transition_properties(risp_ctx *ctx, int32_t n, const double *X_dev, const double *omega_hartree, const double *origin_bohr,
                                          double scale, double *mu_out, double *m_out, double *f_out, double *R_out)
{
    if (!ctx) return RISP_EINVAL;
    if (n <= 0 || !X_dev || (f_out && !omega_hartree)) { risp_set_error(ctx, "risp_transition_properties: need n >= 1, X, and omega for f"); return RISP_EINVAL; }
    RISP_CUDA_TRY(cudaSetDevice(ctx->device));
    int rc;
    if ((rc = ensure_shell_table(ctx))) return rc;
    const double O[3] = {origin_bohr ? origin_bohr[0] : 0.0, origin_bohr ? origin_bohr[1] : 0.0, origin_bohr ? origin_bohr[2] : 0.0};
    if (!(scale > 0.0)) scale = std::sqrt(2.0);          // reading G24: closed-shell singlet, <X|X> = 1
    const int nao = ctx->nao, nocc = ctx->nocc, nvir = ctx->nvir;
    const long long dim = (long long)nocc * nvir, ldao = ctx->ldao, ldvir = ctx->ldvir;
    cudaStream_t st = 0;
    DevScratch scr;
    double *ao = nullptr, *T = nullptr, *P = nullptr, *part = nullptr, *res = nullptr;
    const long long slice = dim > (1 << 20) ? std::max<long long>(4096, ((dim / 1024) + 4095) / 4096 * 4096) : 16384;
    const int nfull = (int)(dim / slice), nz = nfull + (dim % slice ? 1 : 0), NCH = 64;
    RISP_CUDA_TRY(scr.alloc(ao, (size_t)nao * ldao));
    RISP_CUDA_TRY(scr.alloc(T, (size_t)nao * ldvir));
    RISP_CUDA_TRY(scr.alloc(P, (size_t)6 * dim + 2));
    RISP_CUDA_TRY(scr.alloc(part, (size_t)nz * 6 * NCH));
    RISP_CUDA_TRY(scr.alloc(res, (size_t)6 * NCH));
    for (int c = 0; c < 6; ++c) {
        if ((rc = fill_component(ctx, c, O, ao, st))) return rc;
        // r_ia = C_occ^T (r_AO C_vir)
        GemmDesc d1 = gemm_desc(nao, nvir, nao, ao, ldao, true, ctx->d_Cvir, ldvir, false, T, ldvir);
        RISP_CUDA_TRY(risp_dgemm(d1, st));
        GemmDesc d2 = gemm_desc(nocc, nvir, nao, ctx->d_Cocc, ctx->ldocc, false, T, ldvir, false, P + (size_t)c * dim, nvir);
        RISP_CUDA_TRY(risp_dgemm(d2, st));
    }
    std::vector<double> h((size_t)6 * NCH), mu((size_t)n * 3), mm((size_t)n * 3);
    for (int n0 = 0; n0 < n; n0 += NCH) {
        const int nn = std::min(NCH, n - n0);
        const double *Xc = X_dev + (size_t)n0 * dim;
        if (nfull) {
            GemmDesc d = gemm_desc(6, nn, (int)slice, P, dim, true, Xc, dim, true, part, nn);
            d.nb1 = nfull; d.sA1 = slice; d.sB1 = slice; d.sC1 = 6LL * nn;
            RISP_CUDA_TRY(risp_dgemm(d, st));
        }
        if (dim % slice) {
            const long long o = (long long)nfull * slice;
            GemmDesc d = gemm_desc(6, nn, (int)(dim - o), P + o, dim, true, Xc + o, dim, true, part + (size_t)nfull * 6 * nn, nn);
            RISP_CUDA_TRY(risp_dgemm(d, st));
        }
        reduce_slices_kernel<<<(6 * nn + 127) / 128, 128, 0, st>>>(part, nz, 6 * nn, res);
        RISP_CUDA_TRY(cudaGetLastError());
        RISP_CUDA_TRY(cudaMemcpyAsync(h.data(), res, (size_t)6 * nn * 8, cudaMemcpyDeviceToHost, st));
        RISP_CUDA_TRY(cudaStreamSynchronize(st));
        for (int j = 0; j < nn; ++j)
            for (int k = 0; k < 3; ++k) { mu[(size_t)(n0 + j) * 3 + k] = scale * h[(size_t)k * nn + j]; mm[(size_t)(n0 + j) * 3 + k] = scale * h[(size_t)(3 + k) * nn + j]; }
    }
    for (int j = 0; j < n; ++j) {
        const double *u = &mu[(size_t)j * 3], *v = &mm[(size_t)j * 3];
        if (mu_out) std::copy(u, u + 3, mu_out + (size_t)j * 3);
        if (m_out) std::copy(v, v + 3, m_out + (size_t)j * 3);
        if (f_out) f_out[j] = 2.0 / 3.0 * omega_hartree[j] * (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);      // Eq. 5
        if (R_out) R_out[j] = 0.5 * (u[0] * v[0] + u[1] * v[1] + u[2] * v[2]);                                // Eq. 6
    }
    return RISP_OK;
}

// Debug export (include/risp_debug.h): the six AO matrices <mu|(r-O)_k|nu>, <mu|((r-O) x nabla)_k|nu> on the kept shell pairs,
// out_host[6][nao][nao]
extern "C" int risp_debug_oneel_ao(risp_ctx *ctx, const double *origin_bohr, double *out_host)
{
    if (!ctx || !out_host) return RISP_EINVAL;
    RISP_CUDA_TRY(cudaSetDevice(ctx->device));
    int rc;
    if ((rc = ensure_shell_table(ctx))) return rc;
    const double O[3] = {origin_bohr ? origin_bohr[0] : 0.0, origin_bohr ? origin_bohr[1] : 0.0, origin_bohr ? origin_bohr[2] : 0.0};
    DevScratch scr;
    double *ao = nullptr;
    RISP_CUDA_TRY(scr.alloc(ao, (size_t)ctx->nao * ctx->ldao));
    for (int c = 0; c < 6; ++c) {
        if ((rc = fill_component(ctx, c, O, ao, 0))) return rc;
        RISP_CUDA_TRY(cudaMemcpy2D(out_host + (size_t)c * ctx->nao * ctx->nao, (size_t)ctx->nao * 8, ao, (size_t)ctx->ldao * 8, (size_t)ctx->nao * 8, ctx->nao,
                                   cudaMemcpyDeviceToHost));
    }
    return RISP_OK;
}
