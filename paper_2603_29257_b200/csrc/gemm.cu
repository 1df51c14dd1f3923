// gemm.cu -- FP64 GEMM on the sm_100a tensor cores (DMMA.8x8x4 via mma.sync.m8n8k4.f64).
//
// Used for every dense contraction of the sigma-build: the AO<->MO transforms of the J path (Eq. 12, 17,
// PAPER.md:109, 123) and the exchange contractions M^P = X T_ab^P, K += T_ij^P M^P (Eq. 22-23).
// There is no tcgen05 path for FP64 on sm_100a; the native FP64 tensor instruction is the warp-level DMMA.
//
// This file holds the dispatcher and the cp.async kernel used when an operand cannot be described by a TMA tensor
// map (odd leading dimension or batch stride); the main kernel is the TMA/mbarrier pipeline of gemm_tma.cu.
// Tiling (template Cfg): CTA tile BM x BN x BK, WM x WN warps, warp tile (BM/WM) x (BN/WN) made of 8x8 DMMA tiles
// with register accumulators, operands staged in shared memory by a multi-stage cp.async pipeline (16-byte copies
// when the operand's alignment allows, 8-byte otherwise), padded pitches chosen so that the fragment loads (8-byte
// LDS) are bank-conflict free for both operand orientations.
#include "common.cuh"

namespace {

template <int BM_, int BN_, int BK_, int STAGES_, int WM_, int WN_, int MINB_>
struct Cfg {
    static constexpr int BM = BM_, BN = BN_, BK = BK_, STAGES = STAGES_, WM = WM_, WN = WN_, MINB = MINB_;
    static constexpr int NT = WM * WN * 32;
    static constexpr int MI = BM / WM / 8, NI = BN / WN / 8;     // 8x8 tiles per warp
    static constexpr int PITCH_K = BK + 4;                        // tile stored [mn][k]
    static constexpr int A_ELEMS = (BM * PITCH_K > BK * (BM + 4)) ? BM * PITCH_K : BK * (BM + 4);
    static constexpr int B_ELEMS = (BN * PITCH_K > BK * (BN + 4)) ? BN * PITCH_K : BK * (BN + 4);
    static constexpr size_t SMEM = (size_t)STAGES * (A_ELEMS + B_ELEMS) * sizeof(double);
};

__device__ __forceinline__ void cp_async8(double *smem_dst, const double *gsrc, bool pred)
{
    unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    int sz = pred ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(s), "l"(gsrc), "r"(sz));
}
__device__ __forceinline__ void cp_async16(double *smem_dst, const double *gsrc, int bytes)
{
    unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gsrc), "r"(bytes));
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

// load one ROWS x BK operand tile; KC: operand(mn,k) = src[mn*ld + k], else src[k*ld + mn].
// VEC: 16-byte copies (caller guarantees base and ld 16-byte aligned); zero fill outside [0,MN) x [0,K).
template <bool KC, int ROWS, int BK, int NT, bool VEC>
__device__ __forceinline__ void load_tile(double *dst, const double *src, long long ld, int mn0, int k0, int MN, int K, int tid)
{
    constexpr int PITCH_K = BK + 4, PITCH_M = ROWS + 4;
    if (VEC) {
        constexpr int ITER = (ROWS * BK / 2 + NT - 1) / NT;
#pragma unroll
        for (int i = 0; i < ITER; ++i) {
            int idx = tid + i * NT;
            if ((ROWS * BK / 2) % NT != 0 && idx >= ROWS * BK / 2) break;
            if (KC) {
                int k = (idx % (BK / 2)) * 2, r = idx / (BK / 2);
                int rem = (mn0 + r < MN) ? (K - (k0 + k)) : 0;
                int bytes = rem >= 2 ? 16 : (rem == 1 ? 8 : 0);
                const double *g = bytes ? src + (long long)(mn0 + r) * ld + (k0 + k) : src;
                cp_async16(dst + r * PITCH_K + k, g, bytes);
            } else {
                int r = (idx % (ROWS / 2)) * 2, k = idx / (ROWS / 2);
                int rem = (k0 + k < K) ? (MN - (mn0 + r)) : 0;
                int bytes = rem >= 2 ? 16 : (rem == 1 ? 8 : 0);
                const double *g = bytes ? src + (long long)(k0 + k) * ld + (mn0 + r) : src;
                cp_async16(dst + k * PITCH_M + r, g, bytes);
            }
        }
    } else {
        constexpr int ITER = (ROWS * BK + NT - 1) / NT;
#pragma unroll
        for (int i = 0; i < ITER; ++i) {
            int idx = tid + i * NT;
            if ((ROWS * BK) % NT != 0 && idx >= ROWS * BK) break;
            if (KC) {
                int k = idx % BK, r = idx / BK;
                bool ok = (mn0 + r < MN) && (k0 + k < K);
                const double *g = ok ? src + (long long)(mn0 + r) * ld + (k0 + k) : src;
                cp_async8(dst + r * PITCH_K + k, g, ok);
            } else {
                int r = idx % ROWS, k = idx / ROWS;
                bool ok = (mn0 + r < MN) && (k0 + k < K);
                const double *g = ok ? src + (long long)(k0 + k) * ld + (mn0 + r) : src;
                cp_async8(dst + k * PITCH_M + r, g, ok);
            }
        }
    }
}

template <class C, bool AKC, bool BKC, bool VECA, bool VECB>
__global__ void __launch_bounds__(C::NT, C::MINB) dgemm_kernel(GemmDesc d, int tiles_m, int tiles_n)
{
    constexpr int BM = C::BM, BN = C::BN, BK = C::BK, STAGES = C::STAGES, NT = C::NT, MI = C::MI, NI = C::NI;
    constexpr int PITCH_K = C::PITCH_K, PITCH_AM = BM + 4, PITCH_BM = BN + 4;
    extern __shared__ __align__(16) double smem[];
    double *As = smem;
    double *Bs = smem + STAGES * C::A_ELEMS;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp / C::WN, wn = warp % C::WN;
    const int z = blockIdx.z, z1 = z / d.nb2, z2 = z % d.nb2;
    const double *A = d.A + z1 * d.sA1 + z2 * d.sA2;
    const double *B = d.B + z1 * d.sB1 + z2 * d.sB2;
    double *Cp = d.C + z1 * d.sC1 + z2 * d.sC2;
    // tile rasterisation: m fastest, so that concurrently running CTAs share the same B panel in L2
    const int t = blockIdx.x;
    const int tm = t % tiles_m, tn = t / tiles_m;
    const int m0 = tm * BM, n0 = tn * BN;

    double acc[MI][NI][2];
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
        for (int j = 0; j < NI; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    const int nk = (d.K + BK - 1) / BK;
#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < nk) {
            load_tile<AKC, BM, BK, NT, VECA>(As + s * C::A_ELEMS, A, d.lda, m0, s * BK, d.M, d.K, tid);
            load_tile<BKC, BN, BK, NT, VECB>(Bs + s * C::B_ELEMS, B, d.ldb, n0, s * BK, d.N, d.K, tid);
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
                load_tile<AKC, BM, BK, NT, VECA>(As + s * C::A_ELEMS, A, d.lda, m0, kn * BK, d.M, d.K, tid);
                load_tile<BKC, BN, BK, NT, VECB>(Bs + s * C::B_ELEMS, B, d.ldb, n0, kn * BK, d.N, d.K, tid);
            }
            cp_async_commit();
        }
        const double *as = As + (kt % STAGES) * C::A_ELEMS;
        const double *bs = Bs + (kt % STAGES) * C::B_ELEMS;
#pragma unroll
        for (int kk = 0; kk < BK; kk += 4) {
            double a[MI], b[NI];
#pragma unroll
            for (int i = 0; i < MI; ++i) {
                int row = wm * (MI * 8) + i * 8 + q;
                a[i] = AKC ? as[row * PITCH_K + kk + r] : as[(kk + r) * PITCH_AM + row];
            }
#pragma unroll
            for (int j = 0; j < NI; ++j) {
                int col = wn * (NI * 8) + j * 8 + q;
                b[j] = BKC ? bs[col * PITCH_K + kk + r] : bs[(kk + r) * PITCH_BM + col];
            }
#pragma unroll
            for (int i = 0; i < MI; ++i)
#pragma unroll
                for (int j = 0; j < NI; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
    }
    cp_async_wait<0>();
    // epilogue: thread holds C(row = q, col = 2r, 2r+1) of each 8x8 tile
    const bool vecC = ((d.ldc & 1) == 0) && ((d.c_gstride & 1) == 0) && ((((size_t)Cp) & 15) == 0);
#pragma unroll
    for (int i = 0; i < MI; ++i) {
        int row = m0 + wm * (MI * 8) + i * 8 + q;
        if (row >= d.M) continue;
        const long long row_off = d.c_rpg > 0 ? (long long)(row / d.c_rpg) * d.c_gstride + (long long)(row % d.c_rpg) * d.ldc
                                              : (long long)row * d.ldc;
#pragma unroll
        for (int j = 0; j < NI; ++j) {
            int col = n0 + wn * (NI * 8) + j * 8 + 2 * r;
            risp_store_c_pair(d, Cp, row_off, col, acc[i][j][0], acc[i][j][1], vecC);
        }
    }
}

template <class C, bool AKC, bool BKC, bool VECA, bool VECB>
cudaError_t launch3(const GemmDesc &d, cudaStream_t st)
{
    static bool attr_set[64] = {};          // per device: the attribute belongs to the function as loaded on that device
    int dev = 0;
    cudaGetDevice(&dev);
    if (!attr_set[dev & 63]) {
        cudaError_t e = cudaFuncSetAttribute(dgemm_kernel<C, AKC, BKC, VECA, VECB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
        if (e != cudaSuccess) return e;
        attr_set[dev & 63] = true;
    }
    int tiles_m = (d.M + C::BM - 1) / C::BM, tiles_n = (d.N + C::BN - 1) / C::BN;
    dim3 grid(tiles_m * tiles_n, 1, d.nb1 * d.nb2);
    dgemm_kernel<C, AKC, BKC, VECA, VECB><<<grid, C::NT, C::SMEM, st>>>(d, tiles_m, tiles_n);
    return cudaGetLastError();
}

inline bool aligned16(const double *p, long long ld, long long s1, long long s2)
{
    return (((size_t)p) & 15) == 0 && (ld & 1) == 0 && (s1 & 1) == 0 && (s2 & 1) == 0;
}

template <class C, bool AKC, bool BKC>
cudaError_t launch2(const GemmDesc &d, cudaStream_t st)
{
    const bool va = aligned16(d.A, d.lda, d.sA1, d.sA2), vb = aligned16(d.B, d.ldb, d.sB1, d.sB2);
    if (va) return vb ? launch3<C, AKC, BKC, true, true>(d, st) : launch3<C, AKC, BKC, true, false>(d, st);
    return vb ? launch3<C, AKC, BKC, false, true>(d, st) : launch3<C, AKC, BKC, false, false>(d, st);
}

template <class C>
cudaError_t launch1(const GemmDesc &d, cudaStream_t st)
{
    if (d.a_kc) return d.b_kc ? launch2<C, true, true>(d, st) : launch2<C, true, false>(d, st);
    return d.b_kc ? launch2<C, false, true>(d, st) : launch2<C, false, false>(d, st);
}

using Cfg0 = Cfg<128, 128, 16, 4, 2, 4, 1>;    // 8 warps, 1 CTA/SM, warp tile 64x32

}  // namespace

cudaError_t risp_dgemm_tma(const GemmDesc &d, cudaStream_t st);   // gemm_tma.cu

cudaError_t risp_dgemm(const GemmDesc &d, cudaStream_t st)
{
    if (d.M <= 0 || d.N <= 0 || d.nb1 * d.nb2 <= 0) return cudaSuccess;
    if (d.variant != 0) {
        cudaError_t e = risp_dgemm_tma(d, st);
        if (e != cudaErrorNotSupported) return e;
    }
    return launch1<Cfg0>(d, st);
}
