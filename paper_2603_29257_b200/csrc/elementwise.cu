// elementwise.cu -- the HBM-bound steps of the sigma-build: window gather, sigma assembly (Eq. 10).
#include "ctx.h"

namespace {
// Xk[m][no][nv] = X[m][o0+i][v0+a]
__global__ void gather_window_kernel(const double *__restrict__ X, double *__restrict__ Xk, long long total, int nocc, int nvir,
                                     int o0, int no, int v0, int nv)
{
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        int a = (int)(t % nv);
        long long r = t / nv;
        int i = (int)(r % no);
        long long mi = r / no;
        Xk[t] = X[(mi * nocc + o0 + i) * (long long)nvir + v0 + a];
    }
}

// sigma = (eps_a - eps_i) X + 2 J - K' (K' only inside the window; reading G7)
__global__ void assemble_sigma_kernel(const double *__restrict__ X, const double *__restrict__ J, const double *__restrict__ Kk,
                                      const double *__restrict__ eps, double *__restrict__ sigma, long long total, int nocc, int nvir,
                                      int o0, int no, int v0, int nv, int has_K)
{
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        int a = (int)(t % nvir);
        long long r = t / nvir;
        int i = (int)(r % nocc);
        long long mi = r / nocc;
        double s = (eps[nocc + a] - eps[i]) * X[t] + 2.0 * J[t];
        if (has_K && i >= o0 && i < o0 + no && a >= v0 && a < v0 + nv) s -= Kk[(mi * no + (i - o0)) * (long long)nv + (a - v0)];
        sigma[t] = s;
    }
}

__global__ void scatter_window_kernel(const double *__restrict__ Kk, double *__restrict__ Kf, long long total, int nocc, int nvir, int o0,
                                      int no, int v0, int nv)
{
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        int a = (int)(t % nvir);
        long long r = t / nvir;
        int i = (int)(r % nocc);
        long long mi = r / nocc;
        double v = 0.0;
        if (i >= o0 && i < o0 + no && a >= v0 && a < v0 + nv) v = Kk[(mi * no + (i - o0)) * (long long)nv + (a - v0)];
        Kf[t] = v;
    }
}
inline unsigned grid_for(long long total)
{
    long long g = (total + 255) / 256;
    return (unsigned)(g > 148LL * 16 ? 148 * 16 : (g < 1 ? 1 : g));
}
}  // namespace

cudaError_t risp_gather_window(const double *X, double *Xk, int m, int nocc, int nvir, int o0, int no, int v0, int nv, cudaStream_t st)
{
    long long total = (long long)m * no * nv;
    if (total == 0) return cudaSuccess;
    gather_window_kernel<<<grid_for(total), 256, 0, st>>>(X, Xk, total, nocc, nvir, o0, no, v0, nv);
    return cudaGetLastError();
}
cudaError_t risp_assemble_sigma(const double *X, const double *J, const double *Kk, const double *eps, double *sigma, int m, int nocc, int nvir,
                                int o0, int no, int v0, int nv, int has_K, cudaStream_t st)
{
    long long total = (long long)m * nocc * nvir;
    if (total == 0) return cudaSuccess;
    assemble_sigma_kernel<<<grid_for(total), 256, 0, st>>>(X, J, Kk, eps, sigma, total, nocc, nvir, o0, no, v0, nv, has_K);
    return cudaGetLastError();
}
cudaError_t risp_scatter_window(const double *Kk, double *Kf, int m, int nocc, int nvir, int o0, int no, int v0, int nv, cudaStream_t st)
{
    long long total = (long long)m * nocc * nvir;
    if (total == 0) return cudaSuccess;
    scatter_window_kernel<<<grid_for(total), 256, 0, st>>>(Kk, Kf, total, nocc, nvir, o0, no, v0, nv);
    return cudaGetLastError();
}
