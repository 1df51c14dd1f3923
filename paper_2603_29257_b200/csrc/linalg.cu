// linalg.cu -- Cholesky factorisation and triangular inverse of the auxiliary metrics (P|Q) on the device.
//
// The RI metric enters the sigma-build as (P|Q)^-1 (Eq. 3, 15, 20).  The matrices are small
// (N_auxJ <= ~6000), so a blocked right-looking Cholesky with 32-wide panels is enough: diagonal block in one warp,
// panel solve one thread per row, trailing update by the DMMA GEMM.  L^-1 is then built block row by block row, so
// that the per-matvec solve R~ = L^-T (L^-1 R) is two small GEMMs instead of a chain of dependent launches.
#include "ctx.h"

namespace {
constexpr int NB = 32;

// factor the nb x nb diagonal block at (k0,k0); write L_kk in place (upper part zeroed) and its inverse to Dinv[32][32]
__global__ void chol_diag_kernel(double *A, int n, int k0, int nb, double *Dinv, int *info)
{
    __shared__ double a[NB][NB + 1];
    __shared__ double x[NB][NB + 1];
    const int t = threadIdx.x;
    for (int j = 0; j < NB; ++j) a[t][j] = (t < nb && j < nb) ? A[(long long)(k0 + t) * n + k0 + j] : (t == j ? 1.0 : 0.0);
    __syncwarp();
    for (int j = 0; j < nb; ++j) {
        double piv = a[j][j];
        if (!(piv > 0.0)) { if (t == 0 && *info == 0) *info = k0 + j + 1; piv = 1.0; }
        piv = sqrt(piv);
        __syncwarp();
        if (t == j) a[j][j] = piv;
        if (t > j) a[t][j] /= piv;
        __syncwarp();
        if (t > j)
            for (int c = j + 1; c <= t; ++c) a[t][c] -= a[t][j] * a[c][j];
        __syncwarp();
    }
    for (int j = 0; j < NB; ++j) if (j > t) a[t][j] = 0.0;
    __syncwarp();
    // inverse: thread t solves L x = e_t
    for (int i = 0; i < NB; ++i) x[i][t] = 0.0;
    x[t][t] = 1.0 / a[t][t];
    for (int i = t + 1; i < NB; ++i) {
        double s = 0.0;
        for (int c = t; c < i; ++c) s += a[i][c] * x[c][t];
        x[i][t] = -s / a[i][i];
    }
    __syncwarp();
    for (int j = 0; j < NB; ++j) {
        if (t < nb && j < nb) A[(long long)(k0 + t) * n + k0 + j] = a[t][j];
        Dinv[t * NB + j] = x[t][j];
    }
}

// rows i >= k0+nb: A[i][k0:k0+nb] <- A[i][k0:k0+nb] * L_kk^-T ; also zero the upper block A[k0:k0+nb][i]
__global__ void chol_panel_kernel(double *A, int n, int k0, int nb, const double *Dinv)
{
    __shared__ double d[NB * NB];
    for (int i = threadIdx.x; i < NB * NB; i += blockDim.x) d[i] = Dinv[i];
    __syncthreads();
    int i = k0 + nb + blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double r[NB], o[NB];
    for (int c = 0; c < nb; ++c) r[c] = A[(long long)i * n + k0 + c];
    for (int j = 0; j < nb; ++j) {
        double s = 0.0;
        for (int c = 0; c <= j; ++c) s += r[c] * d[j * NB + c];
        o[j] = s;
    }
    for (int j = 0; j < nb; ++j) {
        A[(long long)i * n + k0 + j] = o[j];
        A[(long long)(k0 + j) * n + i] = 0.0;
    }
}

// block row i0 of X = L^-1:  X[i0+r][0:i0] <- Dinv * T (T currently stored there), X[i0 blk][i0 blk] <- Dinv
__global__ void trinv_row_kernel(double *X, int n, int i0, int nb, const double *Dinv)
{
    __shared__ double d[NB * NB];
    for (int i = threadIdx.x; i < NB * NB; i += blockDim.x) d[i] = Dinv[i];
    __syncthreads();
    int c = blockIdx.x * blockDim.x + threadIdx.x;   // column
    if (c >= i0 + nb) return;
    if (c >= i0) {
        for (int r = 0; r < nb; ++r) X[(long long)(i0 + r) * n + c] = d[r * NB + (c - i0)];
        return;
    }
    double t[NB];
    for (int r = 0; r < nb; ++r) t[r] = X[(long long)(i0 + r) * n + c];
    for (int r = 0; r < nb; ++r) {
        double s = 0.0;
        for (int k = 0; k <= r; ++k) s += d[r * NB + k] * t[k];
        X[(long long)(i0 + r) * n + c] = s;
    }
}
// C[p][lane] = sum_q op(A)(p,q) B[q][lane], A lower triangular [n][n], B and C [n][32].  TRANS: op(A) = A^T.
// One CTA per output row; its 8 warps split the q range (two partial sums each), the 32 lanes are the 32 trial-vector slots of
// R / R~ (Eq. 15); the partial sums are added in a fixed order.
template <bool TRANS>
__global__ void __launch_bounds__(256) tri_mat32_kernel(const double *__restrict__ A, int n, const double *__restrict__ B, double *__restrict__ C)
{
    __shared__ double part[8][32];
    const int lane = threadIdx.x, w = threadIdx.y, p = blockIdx.x;
    const int q0 = TRANS ? p : 0, q1 = TRANS ? n : p + 1;
    double a0 = 0.0, a1 = 0.0;
    int q = q0 + w;
    for (; q + 8 < q1; q += 16) {
        const double x0 = TRANS ? A[(long long)q * n + p] : A[(long long)p * n + q];
        const double x1 = TRANS ? A[(long long)(q + 8) * n + p] : A[(long long)p * n + q + 8];
        a0 = fma(x0, B[(long long)q * 32 + lane], a0);
        a1 = fma(x1, B[(long long)(q + 8) * 32 + lane], a1);
    }
    if (q < q1) a0 = fma(TRANS ? A[(long long)q * n + p] : A[(long long)p * n + q], B[(long long)q * 32 + lane], a0);
    part[w][lane] = a0 + a1;
    __syncthreads();
    if (w == 0) {
        double s = 0.0;
#pragma unroll
        for (int ww = 0; ww < 8; ++ww) s += part[ww][lane];
        C[(long long)p * 32 + lane] = s;
    }
}
}  // namespace

// R~ = L^-T (L^-1 R) with the precomputed lower-triangular L^-1; R, tmp, Rt are [n][32]
cudaError_t risp_metric_solve32(const double *Linv, int n, const double *R, double *tmp, double *Rt, cudaStream_t st)
{
    dim3 block(32, 8), grid(n);
    tri_mat32_kernel<false><<<grid, block, 0, st>>>(Linv, n, R, tmp);
    tri_mat32_kernel<true><<<grid, block, 0, st>>>(Linv, n, tmp, Rt);
    return cudaGetLastError();
}

cudaError_t risp_cholesky_inverse(double *A, double *Linv, int n, int *info_host, cudaStream_t st)
{
    *info_host = 0;
    if (n <= 0) return cudaSuccess;
    const int nblk = (n + NB - 1) / NB;
    double *Dinv = nullptr;
    int *d_info = nullptr;
    cudaError_t e;
    if ((e = cudaMalloc(&Dinv, (size_t)nblk * NB * NB * sizeof(double))) != cudaSuccess) return e;
    if ((e = cudaMalloc(&d_info, sizeof(int))) != cudaSuccess) { cudaFree(Dinv); return e; }
    cudaMemsetAsync(d_info, 0, sizeof(int), st);
    for (int b = 0; b < nblk && e == cudaSuccess; ++b) {
        int k0 = b * NB, nb = n - k0 < NB ? n - k0 : NB;
        chol_diag_kernel<<<1, NB, 0, st>>>(A, n, k0, nb, Dinv + (size_t)b * NB * NB, d_info);
        int rest = n - k0 - nb;
        if (rest > 0) {
            chol_panel_kernel<<<(rest + 127) / 128, 128, 0, st>>>(A, n, k0, nb, Dinv + (size_t)b * NB * NB);
            const double *panel = A + (long long)(k0 + nb) * n + k0;
            GemmDesc d = gemm_desc(rest, rest, nb, panel, n, true, panel, n, true, A + (long long)(k0 + nb) * n + (k0 + nb), n, -1.0, 1.0);
            e = risp_dgemm(d, st);
        }
    }
    if (e == cudaSuccess) e = cudaMemsetAsync(Linv, 0, (size_t)n * n * sizeof(double), st);
    for (int b = 0; b < nblk && e == cudaSuccess; ++b) {
        int i0 = b * NB, nb = n - i0 < NB ? n - i0 : NB;
        if (i0 > 0) {
            // T = -L[i0 blk][0:i0] * X[0:i0][0:i0]
            GemmDesc d = gemm_desc(nb, i0, i0, A + (long long)i0 * n, n, true, Linv, n, false, Linv + (long long)i0 * n, n, -1.0, 0.0);
            e = risp_dgemm(d, st);
        }
        trinv_row_kernel<<<(i0 + nb + 127) / 128, 128, 0, st>>>(Linv, n, i0, nb, Dinv + (size_t)b * NB * NB);
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(info_host, d_info, sizeof(int), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = cudaGetLastError();
    cudaFree(Dinv); cudaFree(d_info);
    return e;
}
