// gemm_tma.cu -- FP64 tensor-core GEMM for sm_100a: TMA-fed, mbarrier-pipelined, persistent DMMA kernel.
//
// The dense contractions of the sigma-build (Eq. 12, 17, 22, 23) are FP64 and the only
// FP64 tensor instruction of sm_100a is the warp-level DMMA.8x8x4 (mma.sync.m8n8k4.f64); tcgen05 has no FP64 kind.
// What Blackwell adds for this kernel is the data path: operand tiles are brought into shared memory by TMA
// (cp.async.bulk.tensor, 128-byte swizzle, out-of-bounds zero fill) issued by ONE thread, completion is tracked by
// mbarriers, and the eight DMMA warps never meet at a CTA barrier: each waits on the "full" barrier of a stage and
// releases it through an "empty" barrier, so while one warp of a scheduler is between k tiles the other keeps the
// DMMA pipe busy.  One persistent CTA per SM walks its tiles with the load ring running ahead across tile boundaries
// (the next tile's operands arrive during the epilogue).
//
// Shared-memory layout and the k permutation.  A K-contiguous operand tile is a TMA box [128 rows][16 k] (128-byte
// rows), an MN-contiguous one is eight boxes [16 k][16 mn]; both are written with the 128-byte swizzle (16-byte chunk
// index ^= row index & 7).  A DMMA k-step needs, per lane (q = lane/4, r = lane%4), element (row q, k_r).  The GEMM is
// invariant under any permutation of k applied to both operands, so step s uses k_r = {0,3,12,15}[r] ^ {0,1,4,5}[s]:
// with these sets the 16 lanes of a half warp hit 16 distinct 8-byte words of a 128-byte line for BOTH operand
// orientations (bits (3,0) of k_r take all four values -> K-contiguous case; bits (2,1) too -> MN-contiguous case).
#include "common.cuh"
#include <cuda.h>

namespace {

constexpr int BM_MAX = 128, BN = 128, BK = 16, STAGES = 5, NWARPS = 8, NT = NWARPS * 32;
constexpr int TILE_BYTES = BM_MAX * BK * 8;                   // 16 KiB per operand per stage (A tiles of MI < 8 use a part of it)
constexpr size_t SMEM_BYTES = (size_t)STAGES * 2 * TILE_BYTES + 1024 /*alignment slack*/ + 2 * STAGES * 8;

int sm_count();
long long l2_bytes();

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_4d(unsigned dst, const CUtensorMap *tm, unsigned bar, int c0, int c1, int c2, int c3)
{
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
                 ::"r"(dst), "l"(tm), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}

__device__ __forceinline__ void dmma(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

// byte offset of element (mn, k) of a swizzled operand tile (mn tile-local, multiple-of-8 bases)
template <bool KC>
__device__ __forceinline__ int frag_off(int mn, int k)
{
    if (KC) return mn * 128 + ((((k >> 1) ^ mn) & 7) << 4) + ((k & 1) << 3);
    return (mn >> 4) * 2048 + k * 128 + (((((mn & 15) >> 1) ^ k) & 7) << 4) + ((mn & 1) << 3);
}

struct TmaArgs {
    int coff_a, coff_b;          // offset of the contiguous coordinate (always 0: TMA needs 16-byte aligned box starts)
    int za1, za2, zb1, zb2;      // 1: the operand moves with batch index z1 / z2; 0: shared by the batch
    int grp;                     // GRP kernels: row tiles per group (tile_coords)
};

// Tile number -> (batch z, row tile tm, column tile tn).  Plain order: tm fastest, then tn, then z -- the CTAs of a wave share
// one or two B panels in L2.  Grouped order (GRP; Eq. 22, where A = X' is shared by the whole batch and larger than L2): the
// row tiles are cut into groups of `grp`, and inside a group tm runs fastest, then tn, then z, so that the group's rows of A
// (sized by the host to a quarter of L2) stay resident while every B panel of the batch streams past them once per group.
// In the plain order each wave of 148 tiles touches all of A, and A is re-read from DRAM per column tile and batch entry
// (300 atoms: 202 GB read per launch against 3 GB of operands).
template <bool GRP>
__device__ __forceinline__ void tile_coords(int tile, int tiles_m, int tiles_n, int nbz, int grp, int &z, int &tm, int &tn)
{
    if (!GRP) {
        const int tiles_per_batch = tiles_m * tiles_n;
        z = tile / tiles_per_batch;
        const int tt = tile - z * tiles_per_batch;
        tn = tt / tiles_m;
        tm = tt - tn * tiles_m;
    } else {
        const int per_group = grp * tiles_n * nbz;               // tiles of a full group; only the last group can be shorter
        const int g = tile / per_group;
        const int rem = tile - g * per_group;
        const int gsz = min(grp, tiles_m - g * grp);
        const int r2 = rem / gsz;
        tm = g * grp + (rem - r2 * gsz);
        z = r2 / tiles_n;
        tn = r2 - z * tiles_n;
    }
}

// MI = 8x8 DMMA tiles per warp along m: CTA tile BM = 16 MI rows (128 ... 16), chosen per call (pick_mi).  The small values
// serve the skinny products of the Davidson loop (15 x dim Gram and Ritz updates), which are HBM-bound anyway.
template <bool AKC, bool BKC, int MI, bool GRP>
__global__ void __launch_bounds__(NT, 1) dgemm_tma_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                                                          GemmDesc d, TmaArgs ta, int tiles_m, int tiles_n)
{
    constexpr int BM = 16 * MI, WMROWS = 8 * MI;
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = (unsigned char *)(((size_t)smem_raw + 1023) & ~(size_t)1023);
    unsigned char *As = smem, *Bs = smem + STAGES * TILE_BYTES;
    unsigned long long *bars = (unsigned long long *)(smem + 2 * STAGES * TILE_BYTES);
    const unsigned full0 = smem_u32(bars), empty0 = smem_u32(bars + STAGES);
    const unsigned As_u = smem_u32(As), Bs_u = smem_u32(Bs);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp >> 2, wn = warp & 3;                  // 2 x 4 warps, warp tile (8 MI) x 32
    const int q = lane >> 2, r = lane & 3;

    if (tid == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, NWARPS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int nk = (d.K + BK - 1) / BK;
    const int nbz = d.nb1 * d.nb2;
    const int total_tiles = tiles_m * tiles_n * nbz;
    const int my_tiles = ((int)blockIdx.x < total_tiles) ? (total_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    const long long total_steps = (long long)my_tiles * nk;

    // producer state (warp 0, kept identically by all its lanes): next step to issue
    long long h = 0;
    int h_ti = 0, h_kt = 0, h_slot = 0;
    unsigned h_par = 1;                                        // parity to wait on the empty barrier (fresh barrier passes 1)
    // executed by all lanes of warp 0: lane 0 waits for the slot and arms the barrier, then the boxes of the stage are issued by
    // one lane each (an MN-contiguous operand is BM/16 or 8 boxes: issuing them from one thread costs that warp ~10 % of a k tile)
    int h_m0 = 0, h_n0 = 0, h_z1 = 0, h_z2 = 0;                // coordinates of the producer's tile, recomputed once per tile
    auto issue = [&]() {
        if (h_kt == 0) {
            int z, tm, tn;
            tile_coords<GRP>((int)blockIdx.x + h_ti * (int)gridDim.x, tiles_m, tiles_n, nbz, ta.grp, z, tm, tn);
            h_z1 = z / d.nb2; h_z2 = z - h_z1 * d.nb2;
            h_m0 = tm * BM; h_n0 = tn * BN;
        }
        const int z1 = h_z1, z2 = h_z2, m0 = h_m0, n0 = h_n0, k0 = h_kt * BK;
        const unsigned fb = full0 + 8 * h_slot;
        if (lane == 0) {
            mbar_wait(empty0 + 8 * h_slot, h_par);
            mbar_expect_tx(fb, (BM + BN) * BK * 8);
        }
        __syncwarp();
        const unsigned da = As_u + h_slot * TILE_BYTES, db = Bs_u + h_slot * TILE_BYTES;
        constexpr int NA = AKC ? 1 : BM / 16, NB = BKC ? 1 : BN / 16;
        if (lane < NA) {
            if (AKC) tma_load_4d(da, &tmA, fb, k0 + ta.coff_a, m0, z2 * ta.za2, z1 * ta.za1);
            else tma_load_4d(da + lane * 2048, &tmA, fb, m0 + lane * 16 + ta.coff_a, k0, z2 * ta.za2, z1 * ta.za1);
        } else if (lane < NA + NB) {
            const int b = lane - NA;
            if (BKC) tma_load_4d(db, &tmB, fb, k0 + ta.coff_b, n0, z2 * ta.zb2, z1 * ta.zb1);
            else tma_load_4d(db + b * 2048, &tmB, fb, n0 + b * 16 + ta.coff_b, k0, z2 * ta.zb2, z1 * ta.zb1);
        }
        ++h;
        if (++h_kt == nk) { h_kt = 0; ++h_ti; }
        if (++h_slot == STAGES) { h_slot = 0; h_par ^= 1; }
    };
    if (warp == 0) {
        for (int s = 0; s < STAGES - 2 && h < total_steps; ++s) issue();
    }

    // per-lane fragment offsets of the four k-steps (loop invariant)
    int offA[4], offB[4][2];
#pragma unroll
    for (int s = 0; s < 4; ++s) {
        const int kA = ((r == 0) ? 0 : (r == 1) ? 3 : (r == 2) ? 12 : 15) ^ ((s == 0) ? 0 : (s == 1) ? 1 : (s == 2) ? 4 : 5);
        offA[s] = frag_off<AKC>(wm * WMROWS + q, kA);
        offB[s][0] = frag_off<BKC>(wn * 32 + q, kA);
        offB[s][1] = frag_off<BKC>(wn * 32 + 8 + q, kA);
    }
    constexpr int A_ISTRIDE = AKC ? 8 * 128 : 0;              // KC: rows i*8 further are i*1024 bytes on
    int kstep[4];
#pragma unroll
    for (int s = 0; s < 4; ++s) kstep[s] = ((r == 0) ? 0 : (r == 1) ? 3 : (r == 2) ? 12 : 15) ^ ((s == 0) ? 0 : (s == 1) ? 1 : (s == 2) ? 4 : 5);
    auto offA_mc = [&](int s, int i) { return frag_off<false>(wm * WMROWS + i * 8 + q, kstep[s]); };
    int slot = 0;
    unsigned par = 0;
    const bool vecC = ((d.ldc & 1) == 0) && ((d.c_gstride & 1) == 0) && ((d.sC1 & 1) == 0) && ((d.sC2 & 1) == 0) && ((((size_t)d.C) & 15) == 0);

    for (int ti = 0; ti < my_tiles; ++ti) {
        double acc[MI][4][2];
#pragma unroll
        for (int i = 0; i < MI; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

        for (int kt = 0; kt < nk; ++kt) {
            if (warp == 0 && h < total_steps) issue();
            mbar_wait(full0 + 8 * slot, par);
            const unsigned char *as = As + slot * TILE_BYTES;
            const unsigned char *bs = Bs + slot * TILE_BYTES;
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                double a[MI], b[4];
#pragma unroll
                for (int i = 0; i < MI; ++i) {
                    const int off = AKC ? offA[s] + i * A_ISTRIDE : offA_mc(s, i);
                    a[i] = *reinterpret_cast<const double *>(as + off);
                }
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int off = BKC ? offB[s][0] + j * 8 * 128 : offB[s][j & 1] + (j >> 1) * 2048;
                    b[j] = *reinterpret_cast<const double *>(bs + off);
                }
#pragma unroll
                for (int i = 0; i < MI; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty0 + 8 * slot);
            if (++slot == STAGES) { slot = 0; par ^= 1; }
        }
        // epilogue: thread holds C(row = q, col = 2r, 2r+1) of each 8x8 tile
        int z, tm, tn;
        tile_coords<GRP>((int)blockIdx.x + ti * (int)gridDim.x, tiles_m, tiles_n, nbz, ta.grp, z, tm, tn);
        const int z1 = z / d.nb2, z2 = z % d.nb2;
        const int m0 = tm * BM, n0 = tn * BN;
        double *Cp = d.C + z1 * d.sC1 + z2 * d.sC2;
#pragma unroll
        for (int i = 0; i < MI; ++i) {
            const int row = m0 + wm * WMROWS + i * 8 + q;
            if (row >= d.M) continue;
            const long long row_off = d.c_rpg > 0 ? (long long)(row / d.c_rpg) * d.c_gstride + (long long)(row % d.c_rpg) * d.ldc
                                                  : (long long)row * d.ldc;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int col = n0 + wn * 32 + j * 8 + 2 * r;
                risp_store_c_pair(d, Cp, row_off, col, acc[i][j][0], acc[i][j][1], vecC);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------ host side
typedef CUresult (*EncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                             const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeFn get_encode()
{
    static EncodeFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) == cudaSuccess && qr == cudaDriverEntryPointSuccess)
            fn = (EncodeFn)p;
        else
            (void)cudaGetLastError();
    }
    return fn;
}

// operand(mn, k): KC -> p[mn*ld + k], else p[k*ld + mn]; batch strides s1 (index z1 < nb1), s2 (z2 < nb2)
bool make_map(EncodeFn enc, CUtensorMap *tm, const double *p, bool kc, int MN, int K, long long ld, long long s1, int nb1, long long s2, int nb2,
              int box_mn, int *coff, int *zm1, int *zm2)
{
    if ((ld & 1) || (s1 & 1) || (s2 & 1) || ld <= 0) return false;
    *coff = 0;
    if (((size_t)p) & 15) return false;   // a box that starts 8 bytes off a 16-byte boundary faults (measured): such operands use gemm.cu
    *zm1 = (s1 != 0 && nb1 > 1) ? 1 : 0;
    *zm2 = (s2 != 0 && nb2 > 1) ? 1 : 0;
    cuuint64_t dims[4], strides[3];
    cuuint32_t box[4], es[4] = {1, 1, 1, 1};
    dims[0] = (cuuint64_t)(kc ? K : MN) + *coff;
    dims[1] = (cuuint64_t)(kc ? MN : K);
    dims[2] = *zm2 ? nb2 : 1;
    dims[3] = *zm1 ? nb1 : 1;
    strides[0] = (cuuint64_t)ld * 8;
    strides[1] = *zm2 ? (cuuint64_t)s2 * 8 : strides[0] * dims[1];
    strides[2] = *zm1 ? (cuuint64_t)s1 * 8 : strides[1] * dims[2];
    if (s1 < 0 || s2 < 0 || strides[1] >= (1ull << 40) || strides[2] >= (1ull << 40)) return false;
    box[0] = 16; box[1] = kc ? box_mn : 16; box[2] = 1; box[3] = 1;
    CUresult rc = enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, (void *)p, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                      CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return rc == CUDA_SUCCESS;
}

template <bool AKC, bool BKC, int MI, bool GRP>
cudaError_t launch_mi(const CUtensorMap &ma, const CUtensorMap &mb, const GemmDesc &d, TmaArgs ta, cudaStream_t st)
{
    static bool attr[64] = {};              // per device
    int dev = 0;
    cudaGetDevice(&dev);
    if (!attr[dev & 63]) {
        cudaError_t e = cudaFuncSetAttribute(dgemm_tma_kernel<AKC, BKC, MI, GRP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES);
        if (e != cudaSuccess) return e;
        attr[dev & 63] = true;
    }
    const int sms = sm_count();
    constexpr int BM = 16 * MI;
    const int tiles_m = (d.M + BM - 1) / BM, tiles_n = (d.N + BN - 1) / BN;
    const long long total = (long long)tiles_m * tiles_n * d.nb1 * d.nb2;
    const int grid = (int)std::min<long long>(total, sms);
    if (GRP) {
        // rows of A kept resident per group: a quarter of L2 (the two halves of the L2 mirror each other's lines, B and C stream through)
        const long long row_tile_bytes = (long long)BM * d.K * 8;
        const int gmax = (int)std::max<long long>(8, l2_bytes() / 4 / row_tile_bytes);
        const int ngroups = (tiles_m + gmax - 1) / gmax;
        ta.grp = (tiles_m + ngroups - 1) / ngroups;
    }
    dgemm_tma_kernel<AKC, BKC, MI, GRP><<<grid, NT, SMEM_BYTES, st>>>(ma, mb, d, ta, tiles_m, tiles_n);
    return cudaGetLastError();
}

// Tile height BM = 16 mi for this call: minimise (waves over the SMs) x (rows per tile), i.e. both the padding of the last
// tile row (M = N_occK' = 423: 4 x 112 instead of 4 x 128) and the idle tail of the last wave (M = 4500, 6 column tiles:
// 47 x 6 tiles of 96 rows fill 1.9 waves, 36 x 6 tiles of 128 rows only 1.46); smaller tiles are charged 1.5 % per step.
int pick_mi(int M, long long col_tiles_x_batch, int sms)
{
    int best = 8;
    double best_cost = 1e300;
    for (int mi = 8; mi >= 1; --mi) {
        const int bm = 16 * mi;
        const long long tiles = (long long)((M + bm - 1) / bm) * col_tiles_x_batch;
        const long long waves = (tiles + sms - 1) / sms;
        const double cost = (double)waves * (bm + 12.0) * (1.0 + 0.015 * (8 - mi));   // + ~12 rows' worth of per-tile overhead
        if (cost < best_cost * 0.995) { best = mi; best_cost = cost; }
    }
    return best;
}

long long l2_bytes()
{
    static int l2[64] = {};                 // per device
    int dev = 0;
    cudaGetDevice(&dev);
    if (!l2[dev & 63]) cudaDeviceGetAttribute(&l2[dev & 63], cudaDevAttrL2CacheSize, dev);
    return l2[dev & 63];
}

int sm_count()
{
    static int sms[64] = {};                // per device
    int dev = 0;
    cudaGetDevice(&dev);
    if (!sms[dev & 63]) cudaDeviceGetAttribute(&sms[dev & 63], cudaDevAttrMultiProcessorCount, dev);
    return sms[dev & 63];
}

template <bool AKC, bool BKC, bool GRP = false>
cudaError_t launch(const CUtensorMap &ma, const CUtensorMap &mb, const GemmDesc &d, const TmaArgs &ta, int mi, cudaStream_t st)
{
    switch (mi) {
    case 7: return launch_mi<AKC, BKC, 7, GRP>(ma, mb, d, ta, st);
    case 6: return launch_mi<AKC, BKC, 6, GRP>(ma, mb, d, ta, st);
    case 5: return launch_mi<AKC, BKC, 5, GRP>(ma, mb, d, ta, st);
    case 4: return launch_mi<AKC, BKC, 4, GRP>(ma, mb, d, ta, st);
    case 3: return launch_mi<AKC, BKC, 3, GRP>(ma, mb, d, ta, st);
    case 2: return launch_mi<AKC, BKC, 2, GRP>(ma, mb, d, ta, st);
    case 1: return launch_mi<AKC, BKC, 1, GRP>(ma, mb, d, ta, st);
    default: return launch_mi<AKC, BKC, 8, GRP>(ma, mb, d, ta, st);
    }
}

}  // namespace

// Returns cudaErrorNotSupported when the operands cannot be described by TMA tensor maps (odd leading dimension or
// batch stride, K = 0, driver entry point missing); the caller then uses the cp.async kernel of gemm.cu.
cudaError_t risp_dgemm_tma(const GemmDesc &d, cudaStream_t st)
{
    if (d.K <= 0) return cudaErrorNotSupported;
    const int mi = pick_mi(d.M, (long long)((d.N + BN - 1) / BN) * d.nb1 * d.nb2, sm_count());
    if ((long long)((d.M + 16 * mi - 1) / (16 * mi)) * ((d.N + BN - 1) / BN) * d.nb1 * d.nb2 >= (1ll << 31)) return cudaErrorNotSupported;
    EncodeFn enc = get_encode();
    if (!enc) return cudaErrorNotSupported;
    CUtensorMap ma, mb;
    TmaArgs ta;
    if (!make_map(enc, &ma, d.A, d.a_kc, d.M, d.K, d.lda, d.sA1, d.nb1, d.sA2, d.nb2, 16 * mi, &ta.coff_a, &ta.za1, &ta.za2)) return cudaErrorNotSupported;
    if (!make_map(enc, &mb, d.B, d.b_kc, d.N, d.K, d.ldb, d.sB1, d.nb1, d.sB2, d.nb2, BN, &ta.coff_b, &ta.zb1, &ta.zb2)) return cudaErrorNotSupported;
    ta.grp = 0;
    // Eq. 22 shape: both operands K-contiguous, A shared by a batch of B's and too large to survive a sweep in L2
    const bool a_shared = ta.za1 == 0 && ta.za2 == 0 && (long long)d.nb1 * d.nb2 > 1;
    if (d.a_kc && d.b_kc && a_shared && mi >= 6 && (long long)d.M * d.K * 8 > l2_bytes() / 4)
        return mi == 6 ? launch_mi<true, true, 6, true>(ma, mb, d, ta, st) : mi == 7 ? launch_mi<true, true, 7, true>(ma, mb, d, ta, st)
                                                                                      : launch_mi<true, true, 8, true>(ma, mb, d, ta, st);
    if (d.a_kc) return d.b_kc ? launch<true, true>(ma, mb, d, ta, mi, st) : launch<true, false>(ma, mb, d, ta, mi, st);
    return d.b_kc ? launch<false, true>(ma, mb, d, ta, mi, st) : launch<false, false>(ma, mb, d, ta, mi, st);
}
