/*
 * risp_debug.h -- test and tuning exports of librisp.so that are NOT part of the method's boundary (include/risp.h).
 *
 * They exist so that tests/ and bench.py can reach pieces of the library directly: the FP64 tensor-core GEMM that carries
 * every dense contraction (Eq. 12, 17, 22, 23), the host eigen solver of the Davidson subspace
 * (PAPER.md:189-201), the work-space planner, and the FP64 arithmetic yardsticks the roofline fractions are quoted against.
 * All pointers named *_dev are DEVICE pointers; nothing here keeps state outside the context it is given.
 */
#ifndef RISP_DEBUG_H
#define RISP_DEBUG_H

#include "risp.h"

#ifdef __cplusplus
extern "C" {
#endif

/* C[b](m,n) = alpha sum_k A[b](m,k) B[b](k,n) + beta C[b](m,n), row-major C with leading dimension ldc, `nbatch` problems at
 * element strides sA, sB, sC.  a_kc != 0: A(m,k) = A[m*lda + k], else A[k*lda + m]; likewise b_kc.  variant 1: the TMA/mbarrier
 * kernel whenever the operands allow it (16-byte aligned bases, even leading dimensions), 0: the cp.async kernel.  c_rpg > 0:
 * row r of C lives at (r / c_rpg) * c_gstride + (r % c_rpg) * ldc (the split-row epilogue that writes M^P of Eq. 22).
 * Asynchronous on `stream`.  Returns RISP_OK or RISP_ECUDA. */
int risp_debug_dgemm(int M, int N, int K, const double *A_dev, long long lda, int a_kc, const double *B_dev, long long ldb, int b_kc,
                     double *C_dev, long long ldc, double alpha, double beta, int nbatch, long long sA, long long sB, long long sC,
                     int variant, int c_rpg, long long c_gstride, void *stream);

/* Lowest `nv` eigenpairs of the symmetric n x n HOST matrix a (row-major): w_out[n] all eigenvalues ascending,
 * z_out[i*n + j] = i-th component of eigenvector j (j < nv).  The solver of the projected Davidson problem. */
int risp_debug_sym_eig_lowest(int n, int nv, const double *a_host, double *w_out, double *z_out);

/* Override the work-space plan of the following risp_matvec calls: trial vectors per J sub-batch, AO rows per panel, K aux
 * functions per chunk (0 keeps the automatic choice).  Synchronises the device and drops the current work space. */
int risp_debug_force_plan(risp_ctx *ctx, int mj, int prow, int pc);

/* FP64 yardsticks, measured on the device of `ctx` (or device 0 if ctx == NULL), each timed with CUDA events over `reps`
 * launches after one warm-up:
 *   which = 0  register-resident DFMA chains on every SM (the FP64 ALU peak the integral passes are quoted against), flop/s
 *   which = 1  register-resident DMMA.8x8x4 chains on every SM (the FP64 tensor issue ceiling), flop/s
 *   which = 2  device-to-device copy of `bytes` bytes (read + write counted), bytes/s
 * Returns the rate through *out. */
int risp_debug_yardstick(risp_ctx *ctx, int which, size_t bytes, int reps, double *out);

/* The six one-electron AO matrices behind risp_transition_properties (Eq. 7-8), on the kept shell pairs:
 * out_host[6][nao][nao] = <mu|(r-O)_k|nu> for k = x, y, z, then <mu|((r-O) x nabla)_k|nu>.  origin_bohr: HOST [3] or NULL. */
int risp_debug_oneel_ao(risp_ctx *ctx, const double *origin_bohr, double *out_host);

/* The GEMM of the single-precision mode (RISP_PRECISION_FP32_K; Eq. 22-23 on the tcgen05 tensor cores with operands carried as
 * three bf16 terms, FP32 accumulation) on its own:  C[z][c][r] (+)= sum_k A[z][r][k] B[z][c][k]  for z < nbatch, all DEVICE FP64,
 * A [nbatch][M][K], B [nbatch][N][K], C [nbatch][N][M] contiguous.  via_planes != 0 routes the result through the three-bf16-plane
 * store that feeds Eq. 23; seg_kb = number of 32-k stages accumulated in tensor memory before the partial sum is added, rounded to
 * nearest, to the FP32 running sum in registers (0: the default of the library); shape 0: 128 x 256 tiles with 32 k per stage,
 * 1: 128 x 128 tiles with 64 k per stage, 2: CTA pair (cta_group::2) on a 256 x 256 tile with 32 k per stage.  Synchronous.  Returns RISP_OK, RISP_EINVAL,
 * RISP_ENOMEM or RISP_ECUDA. */
int risp_debug_tcgemm(int32_t M, int32_t N, int32_t K, int32_t nbatch, const double *A_dev, const double *B_dev, double *C_dev,
                      int32_t accumulate, int32_t via_planes, int32_t seg_kb, int32_t shape, void *stream);

/* Tile shape (see risp_debug_tcgemm; -1: the library's choice) and stages per accumulation segment (0: the library's choice) of the
 * Eq. 22 and Eq. 23 launches of the following risp_matvec calls in RISP_PRECISION_FP32_K. */
int risp_debug_set_tc_plan(risp_ctx *ctx, int32_t eq22_shape, int32_t eq22_seg, int32_t eq23_shape, int32_t eq23_seg);

#ifdef __cplusplus
}
#endif
#endif /* RISP_DEBUG_H */
