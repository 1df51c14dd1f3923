// gemm.cu -- FP64 GEMM on the sm_100a tensor cores (DMMA.8x8x4 via mma.sync.m8n8k4.f64).
//
// Used for every dense contraction of the sigma-build: the AO<->MO transforms of the J path (Eq. 12, 17,
// PAPER.md:109, 123) and the exchange contractions M^P = X T_ab^P, K += T_ij^P M^P (Eq. 22-23).
// There is no tcgen05 path for FP64 on sm_100a; the native FP64 tensor instruction is the warp-level DMMA.
//
// Tiling: CTA tile 128x128x16, 8 warps as 2(m) x 4(n), warp tile 64x32 = 8x4 DMMA tiles (64 FP64 accumulators
// per thread), operands staged in shared memory by a 4-stage cp.async pipeline, padded pitches chosen so the
// fragment loads (8-byte LDS) are bank-conflict free for both operand orientations.
#include "common.cuh"

namespace {

constexpr int BM = 128, BN = 128, BK = 16, STAGES = 4, NTHREADS = 256;
constexpr int PITCH_KC = BK + 4;    // tile stored [mn][k]
constexpr int PITCH_MC = BM + 4;    // tile stored [k][mn]
constexpr int TILE_KC = BM * PITCH_KC;
constexpr int TILE_MC = BK * PITCH_MC;
constexpr int TILE_ELEMS = (TILE_KC > TILE_MC ? TILE_KC : TILE_MC);

__device__ __forceinline__ void cp_async8(double *smem_dst, const double *gsrc, bool pred)
{
    unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    int sz = pred ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(s), "l"(gsrc), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ void dmma(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

// load one BMxBK (or BNxBK) operand tile; KC: operand(mn,k) = src[mn*ld + k], else src[k*ld + mn]
template <bool KC>
__device__ __forceinline__ void load_tile(double *dst, const double *src, long long ld, int mn0, int k0, int MN, int K, int tid)
{
    if (KC) {
#pragma unroll
        for (int i = 0; i < (BM * BK) / NTHREADS; ++i) {
            int idx = tid + i * NTHREADS;
            int k = idx % BK, r = idx / BK;
            bool ok = (mn0 + r < MN) && (k0 + k < K);
            const double *g = ok ? src + (long long)(mn0 + r) * ld + (k0 + k) : src;
            cp_async8(dst + r * PITCH_KC + k, g, ok);
        }
    } else {
#pragma unroll
        for (int i = 0; i < (BM * BK) / NTHREADS; ++i) {
            int idx = tid + i * NTHREADS;
            int r = idx % BM, k = idx / BM;
            bool ok = (mn0 + r < MN) && (k0 + k < K);
            const double *g = ok ? src + (long long)(k0 + k) * ld + (mn0 + r) : src;
            cp_async8(dst + k * PITCH_MC + r, g, ok);
        }
    }
}

template <bool AKC, bool BKC>
__global__ void __launch_bounds__(NTHREADS, 1) dgemm_kernel(GemmDesc d, int tiles_m, int tiles_n)
{
    extern __shared__ double smem[];
    double *As = smem;
    double *Bs = smem + STAGES * TILE_ELEMS;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp >> 2, wn = warp & 3;          // 2 x 4 warps
    const int z = blockIdx.z, z1 = z / d.nb2, z2 = z % d.nb2;
    const double *A = d.A + z1 * d.sA1 + z2 * d.sA2;
    const double *B = d.B + z1 * d.sB1 + z2 * d.sB2;
    double *C = d.C + z1 * d.sC1 + z2 * d.sC2;
    // tile rasterisation: m fastest, so that concurrently running CTAs share the same B panel in L2
    const int t = blockIdx.x;
    const int tm = t % tiles_m, tn = t / tiles_m;
    const int m0 = tm * BM, n0 = tn * BN;

    double acc[8][4][2];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    const int nk = (d.K + BK - 1) / BK;
#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < nk) {
            load_tile<AKC>(As + s * TILE_ELEMS, A, d.lda, m0, s * BK, d.M, d.K, tid);
            load_tile<BKC>(Bs + s * TILE_ELEMS, B, d.ldb, n0, s * BK, d.N, d.K, tid);
        }
        cp_async_commit();
    }
    const int q = lane >> 2, r = lane & 3;
    for (int kt = 0; kt < nk; ++kt) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        {   // prefetch tile kt + STAGES - 1 into the slot freed by iteration kt - 1
            int kn = kt + STAGES - 1;
            if (kn < nk) {
                int s = kn % STAGES;
                load_tile<AKC>(As + s * TILE_ELEMS, A, d.lda, m0, kn * BK, d.M, d.K, tid);
                load_tile<BKC>(Bs + s * TILE_ELEMS, B, d.ldb, n0, kn * BK, d.N, d.K, tid);
            }
            cp_async_commit();
        }
        const double *as = As + (kt % STAGES) * TILE_ELEMS;
        const double *bs = Bs + (kt % STAGES) * TILE_ELEMS;
#pragma unroll
        for (int kk = 0; kk < BK; kk += 4) {
            double a[8], b[4];
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                int row = wm * 64 + i * 8 + q;
                a[i] = AKC ? as[row * PITCH_KC + kk + r] : as[(kk + r) * PITCH_MC + row];
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                int col = wn * 32 + j * 8 + q;
                b[j] = BKC ? bs[col * PITCH_KC + kk + r] : bs[(kk + r) * PITCH_MC + col];
            }
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
    }
    cp_async_wait<0>();
    // epilogue: thread holds C(row = q, col = 2r, 2r+1) of each 8x8 tile
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        int row = m0 + wm * 64 + i * 8 + q;
        if (row >= d.M) continue;
        const long long row_off = d.c_rpg > 0 ? (long long)(row / d.c_rpg) * d.c_gstride + (long long)(row % d.c_rpg) * d.ldc
                                              : (long long)row * d.ldc;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            int col = n0 + wn * 32 + j * 8 + 2 * r;
            double *c = C + row_off + col;
            if (col < d.N) c[0] = d.alpha * acc[i][j][0] + (d.beta != 0.0 ? d.beta * c[0] : 0.0);
            if (col + 1 < d.N) c[1] = d.alpha * acc[i][j][1] + (d.beta != 0.0 ? d.beta * c[1] : 0.0);
        }
    }
}

template <bool AKC, bool BKC>
cudaError_t launch(const GemmDesc &d, cudaStream_t st)
{
    static bool attr_set = false;
    size_t smem = (size_t)2 * STAGES * TILE_ELEMS * sizeof(double);
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(dgemm_kernel<AKC, BKC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    int tiles_m = (d.M + BM - 1) / BM, tiles_n = (d.N + BN - 1) / BN;
    dim3 grid(tiles_m * tiles_n, 1, d.nb1 * d.nb2);
    dgemm_kernel<AKC, BKC><<<grid, NTHREADS, smem, st>>>(d, tiles_m, tiles_n);
    return cudaGetLastError();
}

}  // namespace

cudaError_t risp_dgemm(const GemmDesc &d, cudaStream_t st)
{
    if (d.M <= 0 || d.N <= 0 || d.nb1 * d.nb2 <= 0) return cudaSuccess;
    if (d.a_kc) return d.b_kc ? launch<true, true>(d, st) : launch<true, false>(d, st);
    return d.b_kc ? launch<false, true>(d, st) : launch<false, false>(d, st);
}
