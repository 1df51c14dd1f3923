// elementwise.cu -- the HBM-bound steps of the sigma-build: diagonal term, window gather / scatter (Eq. 10,
// PAPER.md:92, 142-148) and the packed <-> full conversion of the symmetric K tensors (Eq. 20-21).
#include "ctx.h"

namespace {
// Xk[m][no][ldk] = X[m][o0+i][v0+a]
__global__ void gather_window_kernel(const double *__restrict__ X, double *__restrict__ Xk, long long total, int nocc, int nvir,
                                     int o0, int no, int v0, int nv, int ldk)
{
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        int a = (int)(t % nv);
        long long r = t / nv;
        int i = (int)(r % no);
        long long mi = r / no;
        Xk[r * ldk + a] = X[(mi * nocc + o0 + i) * (long long)nvir + v0 + a];
    }
}

// sigma = (eps_a - eps_i) X   (the J and K terms are accumulated onto it afterwards)
__global__ void diag_sigma_kernel(const double *__restrict__ X, const double *__restrict__ eps, double *__restrict__ sigma, long long total,
                                  int nocc, int nvir)
{
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        int a = (int)(t % nvir);
        int i = (int)((t / nvir) % nocc);
        sigma[t] = (eps[nocc + a] - eps[i]) * X[t];
    }
}

// sigma[m][o0+i][v0+a] -= K'[m][i][a]   (K acts only inside the window; reading G7)
__global__ void sub_window_kernel(const double *__restrict__ Kk, double *__restrict__ sigma, long long total, int nocc, int nvir, int o0,
                                  int no, int v0, int nv, int ldk)
{
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        int a = (int)(t % nv);
        long long r = t / nv;
        int i = (int)(r % no);
        long long mi = r / no;
        sigma[(mi * nocc + o0 + i) * (long long)nvir + v0 + a] -= Kk[r * ldk + a];
    }
}

__global__ void scatter_window_kernel(const double *__restrict__ Kk, double *__restrict__ Kf, long long total, int nocc, int nvir, int o0,
                                      int no, int v0, int nv, int ldk)
{
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        int a = (int)(t % nvir);
        long long r = t / nvir;
        int i = (int)(r % nocc);
        long long mi = r / nocc;
        double v = 0.0;
        if (i >= o0 && i < o0 + no && a >= v0 && a < v0 + nv) v = Kk[(mi * no + (i - o0)) * (long long)ldk + (a - v0)];
        Kf[t] = v;
    }
}

// packed[p][r(r+1)/2 + c] = full[p][r][c], c <= r
__global__ void pack_sym_kernel(const double *__restrict__ full, long long full_stride, int ld, int n, double *__restrict__ packed, long long tri)
{
    const int r = blockIdx.y, c = blockIdx.x * blockDim.x + threadIdx.x, p = blockIdx.z;
    if (c <= r) packed[(long long)p * tri + (long long)r * (r + 1) / 2 + c] = full[(long long)p * full_stride + (long long)r * ld + c];
}

// full[p*p_stride + r*row_stride + c] = packed[p][max(r,c), min(r,c)]: 32x32 tiles through shared memory so that both the packed
// reads and the mirrored writes are coalesced
__global__ void __launch_bounds__(256) expand_sym_kernel(const double *__restrict__ packed, long long tri, int n, double *__restrict__ full,
                                                         long long row_stride, long long p_stride)
{
    __shared__ double s[32][33];
    const int t = blockIdx.x, p = blockIdx.y;
    int tr = (int)((sqrt(8.0 * t + 1.0) - 1.0) * 0.5);
    while ((tr + 1) * (tr + 2) / 2 <= t) ++tr;
    while (tr * (tr + 1) / 2 > t) --tr;
    const int tc = t - tr * (tr + 1) / 2;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const double *pk = packed + (long long)p * tri;
    double *out = full + (long long)p * p_stride;
    for (int rr = ty; rr < 32; rr += 8) {
        const int r = tr * 32 + rr, c = tc * 32 + tx;
        s[rr][tx] = (r < n && c <= r) ? pk[(long long)r * (r + 1) / 2 + c] : 0.0;
    }
    __syncthreads();
    for (int rr = ty; rr < 32; rr += 8) {
        const int r = tr * 32 + rr, c = tc * 32 + tx;
        if (r < n && c < n) out[(long long)r * row_stride + c] = (c <= r) ? s[rr][tx] : s[tx][rr];
        if (tr != tc) {
            const int r2 = tc * 32 + rr, c2 = tr * 32 + tx;
            if (r2 < n && c2 < n) out[(long long)r2 * row_stride + c2] = s[tx][rr];
        }
    }
}

inline unsigned grid_for(long long total)
{
    long long g = (total + 255) / 256;
    return (unsigned)(g > 148LL * 16 ? 148 * 16 : (g < 1 ? 1 : g));
}
}  // namespace

cudaError_t risp_gather_window(const double *X, double *Xk, int m, int nocc, int nvir, int o0, int no, int v0, int nv, int ldk, cudaStream_t st)
{
    long long total = (long long)m * no * nv;
    if (total == 0) return cudaSuccess;
    gather_window_kernel<<<grid_for(total), 256, 0, st>>>(X, Xk, total, nocc, nvir, o0, no, v0, nv, ldk);
    return cudaGetLastError();
}
cudaError_t risp_diag_sigma(const double *X, const double *eps, double *sigma, int m, int nocc, int nvir, cudaStream_t st)
{
    long long total = (long long)m * nocc * nvir;
    if (total == 0) return cudaSuccess;
    diag_sigma_kernel<<<grid_for(total), 256, 0, st>>>(X, eps, sigma, total, nocc, nvir);
    return cudaGetLastError();
}
cudaError_t risp_sub_window(const double *Kk, double *sigma, int m, int nocc, int nvir, int o0, int no, int v0, int nv, int ldk, cudaStream_t st)
{
    long long total = (long long)m * no * nv;
    if (total == 0) return cudaSuccess;
    sub_window_kernel<<<grid_for(total), 256, 0, st>>>(Kk, sigma, total, nocc, nvir, o0, no, v0, nv, ldk);
    return cudaGetLastError();
}
cudaError_t risp_scatter_window(const double *Kk, double *Kf, int m, int nocc, int nvir, int o0, int no, int v0, int nv, int ldk, cudaStream_t st)
{
    long long total = (long long)m * nocc * nvir;
    if (total == 0) return cudaSuccess;
    scatter_window_kernel<<<grid_for(total), 256, 0, st>>>(Kk, Kf, total, nocc, nvir, o0, no, v0, nv, ldk);
    return cudaGetLastError();
}
cudaError_t risp_pack_sym(const double *full, long long full_stride, int ld, int n, int np, double *packed, long long tri, cudaStream_t st)
{
    if (n <= 0 || np <= 0) return cudaSuccess;
    dim3 grid((n + 255) / 256, n, np);
    pack_sym_kernel<<<grid, 256, 0, st>>>(full, full_stride, ld, n, packed, tri);
    return cudaGetLastError();
}
cudaError_t risp_expand_sym(const double *packed, long long tri, int n, int np, double *full, long long row_stride, long long p_stride,
                            cudaStream_t st)
{
    if (n <= 0 || np <= 0) return cudaSuccess;
    const int nt = (n + 31) / 32;
    dim3 grid(nt * (nt + 1) / 2, np);
    expand_sym_kernel<<<grid, 256, 0, st>>>(packed, tri, n, full, row_stride, p_stride);
    return cudaGetLastError();
}
