// elementwise.cu -- the HBM-bound steps of the sigma-build: diagonal term, window gather / scatter (Eq. 10,
// PAPER.md:92, 142-148) and the packed <-> full conversion of the symmetric K tensors (Eq. 20-21).
#include "ctx.h"

namespace {
// The three streaming kernels work row by row (one (vector, occupied) row of X / sigma per CTA pass): no 64-bit divisions per
// element, 16-byte accesses where the row start allows, rows strided over the grid.
// Xk[m][no][ldk] = X[m][o0+i][v0+a]
__global__ void __launch_bounds__(256) gather_window_kernel(const double *__restrict__ X, double *__restrict__ Xk, long long rows, int nocc, int nvir,
                                                            int o0, int no, int v0, int nv, int ldk)
{
    for (long long r = blockIdx.x; r < rows; r += gridDim.x) {
        const long long mi = r / no;
        const int i = (int)(r - mi * no);
        const double *src = X + (mi * nocc + o0 + i) * (long long)nvir + v0;
        double *dst = Xk + r * ldk;
        for (int a = threadIdx.x; a < nv; a += blockDim.x) dst[a] = src[a];
    }
}

// sigma = (eps_a - eps_i) X   (the J and K terms are accumulated onto it afterwards)
__global__ void __launch_bounds__(256) diag_sigma_kernel(const double *__restrict__ X, const double *__restrict__ eps, double *__restrict__ sigma,
                                                         long long rows, int nocc, int nvir)
{
    const double *ev = eps + nocc;
    for (long long r = blockIdx.x; r < rows; r += gridDim.x) {
        const double ei = eps[(int)(r % nocc)];
        const double *x = X + r * nvir;
        double *s = sigma + r * nvir;
        if ((((size_t)x | (size_t)s) & 15) == 0) {
            const int n2 = nvir >> 1;
            for (int a = threadIdx.x; a < n2; a += blockDim.x) {
                const double2 xv = reinterpret_cast<const double2 *>(x)[a];
                double2 o;
                o.x = (ev[2 * a] - ei) * xv.x; o.y = (ev[2 * a + 1] - ei) * xv.y;
                reinterpret_cast<double2 *>(s)[a] = o;
            }
            if ((nvir & 1) && threadIdx.x == 0) s[nvir - 1] = (ev[nvir - 1] - ei) * x[nvir - 1];
        } else {
            for (int a = threadIdx.x; a < nvir; a += blockDim.x) s[a] = (ev[a] - ei) * x[a];
        }
    }
}

// sigma[m][o0+i][v0+a] -= K'[m][i][a]   (K acts only inside the window; reading G7)
__global__ void __launch_bounds__(256) sub_window_kernel(const double *__restrict__ Kk, double *__restrict__ sigma, long long rows, int nocc, int nvir,
                                                         int o0, int no, int v0, int nv, int ldk)
{
    for (long long r = blockIdx.x; r < rows; r += gridDim.x) {
        const long long mi = r / no;
        const int i = (int)(r - mi * no);
        double *dst = sigma + (mi * nocc + o0 + i) * (long long)nvir + v0;
        const double *src = Kk + r * ldk;
        for (int a = threadIdx.x; a < nv; a += blockDim.x) dst[a] -= src[a];
    }
}

// sigma[m][o0+i][v0+a] += scale * K'[m][i][a]   (the (ib|ja) term of full TDDFT enters A+B and A-B with opposite signs, Eq. 2)
__global__ void __launch_bounds__(256) axpy_window_kernel(const double *__restrict__ Kk, double scale, double *__restrict__ sigma, long long rows, int nocc,
                                                          int nvir, int o0, int no, int v0, int nv, int ldk)
{
    for (long long r = blockIdx.x; r < rows; r += gridDim.x) {
        const long long mi = r / no;
        const int i = (int)(r - mi * no);
        double *dst = sigma + (mi * nocc + o0 + i) * (long long)nvir + v0;
        const double *src = Kk + r * ldk;
        for (int a = threadIdx.x; a < nv; a += blockDim.x) dst[a] = fma(scale, src[a], dst[a]);
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

inline unsigned rows_grid(long long rows) { return (unsigned)(rows < 148LL * 32 ? rows : 148 * 32); }
inline unsigned grid_for(long long total)
{
    long long g = (total + 255) / 256;
    return (unsigned)(g > 148LL * 16 ? 148 * 16 : (g < 1 ? 1 : g));
}
}  // namespace

cudaError_t risp_gather_window(const double *X, double *Xk, int m, int nocc, int nvir, int o0, int no, int v0, int nv, int ldk, cudaStream_t st)
{
    long long rows = (long long)m * no;
    if (rows == 0 || nv == 0) return cudaSuccess;
    gather_window_kernel<<<rows_grid(rows), nv >= 256 ? 256 : 128, 0, st>>>(X, Xk, rows, nocc, nvir, o0, no, v0, nv, ldk);
    return cudaGetLastError();
}
cudaError_t risp_diag_sigma(const double *X, const double *eps, double *sigma, int m, int nocc, int nvir, cudaStream_t st)
{
    long long rows = (long long)m * nocc;
    if (rows == 0 || nvir == 0) return cudaSuccess;
    diag_sigma_kernel<<<rows_grid(rows), nvir >= 512 ? 256 : 128, 0, st>>>(X, eps, sigma, rows, nocc, nvir);
    return cudaGetLastError();
}
cudaError_t risp_sub_window(const double *Kk, double *sigma, int m, int nocc, int nvir, int o0, int no, int v0, int nv, int ldk, cudaStream_t st)
{
    long long rows = (long long)m * no;
    if (rows == 0 || nv == 0) return cudaSuccess;
    sub_window_kernel<<<rows_grid(rows), nv >= 256 ? 256 : 128, 0, st>>>(Kk, sigma, rows, nocc, nvir, o0, no, v0, nv, ldk);
    return cudaGetLastError();
}
cudaError_t risp_axpy_window(const double *Kk, double scale, double *sigma, int m, int nocc, int nvir, int o0, int no, int v0, int nv, int ldk, cudaStream_t st)
{
    long long rows = (long long)m * no;
    if (rows == 0 || nv == 0) return cudaSuccess;
    axpy_window_kernel<<<rows_grid(rows), nv >= 256 ? 256 : 128, 0, st>>>(Kk, scale, sigma, rows, nocc, nvir, o0, no, v0, nv, ldk);
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
