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
    int variant;   // 1: TMA kernel (gemm_tma.cu) whenever the operands allow it; 0: always the cp.async kernel (tests, tuning)
};

#ifdef __CUDACC__
// epilogue store of the two adjacent accumulator columns (col, col + 1) a DMMA thread holds
__device__ __forceinline__ void risp_store_c_pair(const GemmDesc &d, double *Cp, long long row_off, int col, double v0, double v1, bool vec_ok)
{
    if (col >= d.N) return;
    double *c0 = Cp + row_off + col;
    const bool has1 = col + 1 < d.N;
    if (vec_ok && has1) {
        double2 v;
        if (d.beta != 0.0) {
            v = *reinterpret_cast<double2 *>(c0);
            v.x = d.alpha * v0 + d.beta * v.x; v.y = d.alpha * v1 + d.beta * v.y;
        } else { v.x = d.alpha * v0; v.y = d.alpha * v1; }
        *reinterpret_cast<double2 *>(c0) = v;
    } else {
        c0[0] = d.alpha * v0 + (d.beta != 0.0 ? d.beta * c0[0] : 0.0);
        if (has1) c0[1] = d.alpha * v1 + (d.beta != 0.0 ? d.beta * c0[1] : 0.0);
    }
}
#endif
cudaError_t risp_dgemm(const GemmDesc &d, cudaStream_t st);

// ---------------------------------------------------------------------------------------------------
// Single-precision-mode GEMM on tcgen05 (gemm_tc.cu): operands are three bf16 planes each (x = x1 + x2 + x3), both K-contiguous,
//   acc(r, c) = sum_k A[z](r, k) B[z](c, k)   in FP32,   stored transposed:
//   out(r, c) at z*sC + (rpg ? (r / rpg)*gstride + r % rpg : r) + c*ldc;  out_kind 0: FP64 (accumulate: += ), 1: three bf16 planes.
// Leading dimensions, plane and batch strides are in elements and multiples of 8; sA / sB = 0: the operand is shared by the batch.
struct TcGemmDesc {
    int M, N, K, nb;
    const void *A; long long lda, planeA, sA;
    const void *B; long long ldb, planeB, sB;
    void *C; long long ldc, sC, planeC;
    int out_kind, rpg; long long gstride; int accumulate;
    int seg_kb = 0;          // stages per accumulation segment (0: the default, 1)
    int shape = 0;           // 0: 128 x 256 tiles, 32 k per stage (64-byte swizzle rows); 1: 128 x 128 tiles, 64 k per stage (128-byte rows);
                             // 2: CTA pair (cta_group::2), 256 x 256 tile per pair, 32 k per stage, four stages
};
cudaError_t risp_tcgemm(const TcGemmDesc &d, cudaStream_t st);
cudaError_t risp_split_rows_bf3(const double *X, long long ldx, long long rows, int n, void *out, long long ldo, long long plane, int rpg,
                                long long gstride, cudaStream_t st);
cudaError_t risp_split_transpose_bf3(const double *X, long long ldx, int rows, int n, void *out, long long ldo, long long plane, cudaStream_t st);
cudaError_t risp_expand_sym_bf3(const double *packed, long long tri, int n, int np, void *full, long long row_stride, long long p_stride, long long plane,
                                cudaStream_t st);
inline GemmDesc gemm_desc(int M, int N, int K, const double *A, long long lda, bool a_kc, const double *B, long long ldb, bool b_kc,
                          double *C, long long ldc, double alpha = 1.0, double beta = 0.0)
{
    GemmDesc d;
    d.M = M; d.N = N; d.K = K; d.A = A; d.lda = lda; d.B = B; d.ldb = ldb; d.C = C; d.ldc = ldc;
    d.alpha = alpha; d.beta = beta; d.nb1 = 1; d.nb2 = 1;
    d.sA1 = d.sA2 = d.sB1 = d.sB2 = d.sC1 = d.sC2 = 0; d.a_kc = a_kc; d.b_kc = b_kc; d.c_rpg = 0; d.c_gstride = 0; d.variant = 1;
    return d;
}
