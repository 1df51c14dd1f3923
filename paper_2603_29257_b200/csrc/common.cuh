// common.cuh -- shared declarations of the librisp CUDA sources (sm_100a, FP64).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>
#include "../../include/risp.h"

#define RISP_CUDA_TRY(expr)                                                                         \
    do {                                                                                            \
        cudaError_t e_ = (expr);                                                                    \
        if (e_ != cudaSuccess) {                                                                    \
            risp_set_error(ctx, std::string(#expr) + ": " + cudaGetErrorString(e_) + " at " +       \
                                    __FILE__ + ":" + std::to_string(__LINE__));                     \
            return e_ == cudaErrorMemoryAllocation ? RISP_ENOMEM : RISP_ECUDA;                      \
        }                                                                                           \
    } while (0)

struct risp_ctx;
void risp_set_error(risp_ctx *ctx, const std::string &msg);

// ---------------------------------------------------------------------------------------------------
// FP64 tensor-core GEMM (DMMA m8n8k4), gemm.cu
//   C[b](m,n) = alpha * sum_k A[b](m,k) B[b](k,n) + beta * C[b](m,n),  C row-major with leading dimension ldc.
//   a_kc: A(m,k) = A[m*lda + k] (K contiguous) else A[k*lda + m];  b_kc: B(k,n) = B[n*ldb + k] else B[k*ldb + n].
//   Two-level batch: batch index z = z1*nb2 + z2, operand offsets z1*s?1 + z2*s?2 (elements).
struct GemmDesc {
    int M, N, K;
    const double *A; long long lda;
    const double *B; long long ldb;
    double *C; long long ldc;
    double alpha, beta;
    int nb1, nb2;
    long long sA1, sA2, sB1, sB2, sC1, sC2;
    bool a_kc, b_kc;
    // optional split of the C rows: row r lives at (r / c_rpg) * c_gstride + (r % c_rpg) * ldc  (c_rpg = 0: plain r * ldc)
    int c_rpg; long long c_gstride;
    // optional split of the C columns: column c lives at (c / c_cpg) * c_cgstride + (c % c_cpg)  (c_cpg = 0: plain c).  Lets one GEMM
    // over N = (P, a) write the per-P blocks M^P[j][a] of Eq. 22 without padding N to the tile width per P.
    int c_cpg; long long c_cgstride;
};

#ifdef __CUDACC__
// epilogue store of the two adjacent accumulator columns (col, col + 1) a DMMA thread holds
__device__ __forceinline__ void risp_store_c_pair(const GemmDesc &d, double *Cp, long long row_off, int col, double v0, double v1, bool vec_ok)
{
    if (col >= d.N) return;
    long long o0 = col, o1 = col + 1;
    bool adjacent = true;
    if (d.c_cpg > 0) {
        const int g = col / d.c_cpg, a = col - g * d.c_cpg;
        o0 = (long long)g * d.c_cgstride + a;
        adjacent = a + 1 < d.c_cpg;
        o1 = adjacent ? o0 + 1 : (long long)(g + 1) * d.c_cgstride;
    }
    double *c0 = Cp + row_off + o0;
    const bool has1 = col + 1 < d.N;
    if (vec_ok && has1 && adjacent && ((o0 & 1) == 0)) {
        double2 v;
        if (d.beta != 0.0) {
            v = *reinterpret_cast<double2 *>(c0);
            v.x = d.alpha * v0 + d.beta * v.x; v.y = d.alpha * v1 + d.beta * v.y;
        } else { v.x = d.alpha * v0; v.y = d.alpha * v1; }
        *reinterpret_cast<double2 *>(c0) = v;
    } else {
        c0[0] = d.alpha * v0 + (d.beta != 0.0 ? d.beta * c0[0] : 0.0);
        if (has1) { double *c1 = Cp + row_off + o1; c1[0] = d.alpha * v1 + (d.beta != 0.0 ? d.beta * c1[0] : 0.0); }
    }
}
#endif
cudaError_t risp_dgemm(const GemmDesc &d, cudaStream_t st);
void risp_dgemm_set_variant(int v);   // tile configuration (debug / tuning only)
inline GemmDesc gemm_desc(int M, int N, int K, const double *A, long long lda, bool a_kc, const double *B, long long ldb, bool b_kc,
                          double *C, long long ldc, double alpha = 1.0, double beta = 0.0)
{
    GemmDesc d;
    d.M = M; d.N = N; d.K = K; d.A = A; d.lda = lda; d.B = B; d.ldb = ldb; d.C = C; d.ldc = ldc;
    d.alpha = alpha; d.beta = beta; d.nb1 = 1; d.nb2 = 1;
    d.sA1 = d.sA2 = d.sB1 = d.sB2 = d.sC1 = d.sC2 = 0; d.a_kc = a_kc; d.b_kc = b_kc; d.c_rpg = 0; d.c_gstride = 0; d.c_cpg = 0; d.c_cgstride = 0;
    return d;
}
