// gemm_tc.cu -- the single-precision mode of the K contractions (Eq. 22-23; "all quantities after the integral
// evaluation are kept in single precision") on the 5th-generation tensor cores of sm_100a.
//
// tcgen05 has no FP32 (or FP64) input kind, so an FP32 operand x is carried as three bfloat16 terms x = x1 + x2 + x3
// (x1 = bf16(x), x2 = bf16(x - x1), x3 = bf16(x - x1 - x2): 3 x 8 significand bits, the remainders are exact), and a product
// sum_k a_k b_k is formed from the six term products of weight >= 2^-16,
//     a1 b1 + (a1 b2 + a2 b1) + (a1 b3 + a2 b2 + a3 b1),
// each an exact bf16 x bf16 product accumulated in FP32 in tensor memory.  The dropped products are of relative size 2^-24, the
// unit roundoff of binary32: the result has the accuracy of an FP32 GEMM at one sixth of the bf16 tensor rate.
//
//   C^T-store GEMM:   acc(r, c) = sum_k A[r][k] B[c][k]        both operands K-contiguous, three planes each
//   out(r, c) at      z * sC + (r / rpg) * gstride + (r % rpg) + c * ldc      (the accumulator row index is the CONTIGUOUS output index)
//
// Single-CTA kernel (tcgemm_bf16x3_kernel): one persistent CTA per SM, 320 threads: warp 0 = TMA producer (one lane), warp 1 =
// tensor-memory allocation + MMA issue (one lane), warps 2-9 = epilogue (tcgen05.ld of the 128 x BN accumulator, one row and half the
// columns per thread, so that the 32 lanes of a warp write 32 consecutive output elements per column).  Operand tiles are TMA boxes
// [3 planes][rows][32 k] in the 64-byte swizzle, three stages; the accumulator is double-buffered in tensor memory (2 x 256 columns)
// so the register accumulation of one segment runs under the MMAs of the next.
// CTA-pair kernel (tcgemm2_bf16x3_kernel, what risp_matvec launches): the same roles in each CTA of a 2-CTA cluster, one
// tcgen05.mma.cta_group::2 stream issued by the leader for a 256 x BN tile; see the comment above it.
#include "common.cuh"
#include <cuda.h>
#include <cuda_bf16.h>
#include <algorithm>

namespace {

constexpr int BM = 128, BN_MAX = 256, NEPI = 8, NT = (2 + NEPI) * 32, SEG_K = 32;
// Shape of one kernel variant: BK k per stage (32: 64-byte swizzle rows, 64: 128-byte rows), column cap of the tile, stages
template <int BK_, int BNCAP_, int STAGES_>
struct TcShape {
    static constexpr int BK = BK_, BNCAP = BNCAP_, STAGES = STAGES_;
    static constexpr int A_PLANE = BM * BK * 2, B_PLANE_MAX = BNCAP * BK * 2, STAGE_BYTES = 3 * A_PLANE + 3 * B_PLANE_MAX;
    static constexpr size_t SMEM_BYTES = (size_t)STAGES * STAGE_BYTES + 1024 + 128;
};

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count)); }
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory"); }
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "TC_WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra TC_WAIT_DONE;\n"
        "bra TC_WAIT_LOOP;\n"
        "TC_WAIT_DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_4d(unsigned dst, const CUtensorMap *tm, unsigned bar, int c0, int c1, int c2, int c3)
{
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
                 ::"r"(dst), "l"(tm), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
// D[tmem] (+)= A[smem] B[smem]^T, bf16 inputs, FP32 accumulation
__device__ __forceinline__ void umma_bf16(unsigned tmem_d, unsigned long long adesc, unsigned long long bdesc, unsigned idesc, unsigned accumulate)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(unsigned bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_ld32(unsigned taddr, unsigned (&v)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,"
        "%27,%28,%29,%30,%31}, [%32];\n"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]), "=r"(v[10]),
          "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]),
          "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]),
          "=r"(v[31])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// shared-memory matrix descriptor of a K-contiguous operand plane [rows][32 bf16] in the 64-byte swizzle: 8-row groups are 512 B
// apart (SBO), the leading byte offset is unused for swizzled K-major layouts, version 1 (sm_100), layout type 4 = SWIZZLE_64B
template <int BK>
__device__ __forceinline__ unsigned long long smem_desc(unsigned addr)
{
    constexpr unsigned long long sbo = (8 * BK * 2) >> 4, lt = BK == 64 ? 2 : 4;       // 8 rows of BK bf16; SWIZZLE_128B = 2, SWIZZLE_64B = 4
    return (unsigned long long)((addr & 0x3FFFF) >> 4) | (1ull << 16) | (sbo << 32) | (1ull << 46) | (lt << 61);
}

struct TcArgs {
    int M, N, K, BN;
    int nb;                      // batch
    int za, zb;                  // 1: the operand moves with the batch index
    int out_kind;                // 0: FP64 (beta 0 / 1), 1: three bf16 planes
    void *C; long long ldc, sC, planeC; int rpg; long long gstride; int accumulate;
    int tiles_m, tiles_n;
    int seg_kb;                  // stages (of 32 k) per accumulation segment
    int gm;                      // row tiles per group of the tile order
};

// tile order inside one batch entry: groups of gm row tiles x all column tiles, m fastest inside a group, so that one wave of CTAs
// works on operands that stay in L2 (the same order as gemm_tma.cu)
__device__ __forceinline__ void tile_coords(int tt, int tiles_m, int tiles_n, int gm, int &tm, int &tn)
{
    const int per_group = gm * tiles_n;
    const int g = tt / per_group, r = tt - g * per_group;
    const int rows = min(gm, tiles_m - g * gm);
    tm = g * gm + r % rows;
    tn = r / rows;
}

__device__ __forceinline__ void split3(float v, __nv_bfloat16 &b1, __nv_bfloat16 &b2, __nv_bfloat16 &b3)
{
    b1 = __float2bfloat16_rn(v);
    const float r1 = v - __bfloat162float(b1);
    b2 = __float2bfloat16_rn(r1);
    b3 = __float2bfloat16_rn(r1 - __bfloat162float(b2));
}

// The tensor core adds every MMA result into the FP32 accumulator with truncation, and six MMAs per 16 k make that a bias that
// grows linearly with K (measured: 1e-5 relative at K = 1496, 2.3e-5 at K = 3392).  The K loop is therefore cut into segments of
// SEG_KB stages (32 k each): each segment is accumulated in tensor memory from zero and the eight epilogue warps add it, rounded to nearest, to FP32
// running sums they keep in registers (128 per thread: one accumulator row, half the columns) while the MMA warp fills the other
// accumulator buffer.  The result is written once per tile.
template <class S>
__global__ void __launch_bounds__(NT, 1) tcgemm_bf16x3_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, TcArgs g)
{
    constexpr int BK = S::BK, STAGES = S::STAGES, A_PLANE = S::A_PLANE, STAGE_BYTES = S::STAGE_BYTES;
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = (unsigned char *)(((size_t)smem_raw + 1023) & ~(size_t)1023);
    unsigned long long *bars = (unsigned long long *)(smem + STAGES * STAGE_BYTES);
    unsigned *tmem_slot = (unsigned *)(bars + 2 * STAGES + 4);
    const unsigned smem_u = smem_u32(smem);
    const unsigned full0 = smem_u32(bars), empty0 = smem_u32(bars + STAGES), tfull0 = smem_u32(bars + 2 * STAGES), tempty0 = smem_u32(bars + 2 * STAGES + 2);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(tfull0 + 8 * s, 1); mbar_init(tempty0 + 8 * s, NEPI); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(512) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const unsigned tmem_base = *tmem_slot;

    const int nk = (g.K + BK - 1) / BK;
    const int nseg = (nk + g.seg_kb - 1) / g.seg_kb;
    const int tiles_per_batch = g.tiles_m * g.tiles_n;
    const int total_tiles = tiles_per_batch * g.nb;
    const int b_plane = g.BN * BK * 2;
    const unsigned stage_tx = 3 * A_PLANE + 3 * b_plane;

    if (warp == 0) {
        if (lane == 0) {
            int slot = 0; unsigned par = 1;
            for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
                const int z = tile / tiles_per_batch, tt = tile % tiles_per_batch;
                int tm, tn;
                tile_coords(tt, g.tiles_m, g.tiles_n, g.gm, tm, tn);
                for (int kb = 0; kb < nk; ++kb) {
                    mbar_wait(empty0 + 8 * slot, par);
                    const unsigned fb = full0 + 8 * slot, dst = smem_u + slot * STAGE_BYTES;
                    mbar_expect_tx(fb, stage_tx);
                    tma_load_4d(dst, &tmA, fb, kb * BK, tm * BM, 0, g.za ? z : 0);
                    tma_load_4d(dst + 3 * A_PLANE, &tmB, fb, kb * BK, tn * g.BN, 0, g.zb ? z : 0);
                    if (++slot == STAGES) { slot = 0; par ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            // instruction descriptor: D = F32 (bits 4-5 = 1), A = B = BF16 (bits 7-9, 10-12 = 1), both K-major, N >> 3 at bit 17, M >> 4 at bit 24
            const unsigned idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((unsigned)(g.BN >> 3) << 17) | ((unsigned)(BM >> 4) << 24);
            int slot = 0; unsigned par = 0;
            int acc = 0; unsigned apar = 1;
            for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
                for (int kb0 = 0; kb0 < nk; kb0 += g.seg_kb) {
                    mbar_wait(tempty0 + 8 * acc, apar);
                    tc_fence_after();
                    const unsigned tacc = tmem_base + acc * BN_MAX;
                    const int kb1 = min(nk, kb0 + g.seg_kb);
                    for (int kb = kb0; kb < kb1; ++kb) {
                        mbar_wait(full0 + 8 * slot, par);
                        tc_fence_after();
                        const unsigned a0 = smem_u + slot * STAGE_BYTES, b0 = a0 + 3 * A_PLANE;
                        // Issue order inside a stage: the five small products of both 16-k steps first, the leading product a1 b1
                        // last.  Every MMA truncates the accumulator at its current magnitude; in a fresh segment the small terms
                        // therefore cost nothing and only the two leading MMAs per stage round at the size of the result.
                        unsigned long long ad[3][BK / 16], bd[3][BK / 16];
#pragma unroll
                        for (int ks = 0; ks < BK / 16; ++ks)
#pragma unroll
                            for (int p = 0; p < 3; ++p) {
                                ad[p][ks] = smem_desc<BK>(a0 + p * A_PLANE + ks * 32);
                                bd[p][ks] = smem_desc<BK>(b0 + p * b_plane + ks * 32);
                            }
                        constexpr int PA[6] = {2, 0, 1, 1, 0, 0}, PB[6] = {0, 2, 1, 0, 1, 0};
#pragma unroll
                        for (int t = 0; t < 6; ++t)
#pragma unroll
                            for (int ks = 0; ks < BK / 16; ++ks)
                                umma_bf16(tacc, ad[PA[t]][ks], bd[PB[t]][ks], idesc, (kb != kb0) || t != 0 || ks != 0);
                        umma_commit(empty0 + 8 * slot);
                        if (++slot == STAGES) { slot = 0; par ^= 1; }
                    }
                    umma_commit(tfull0 + 8 * acc);
                    if (++acc == 2) { acc = 0; apar ^= 1; }
                }
            }
        }
    } else {
        const int lg = warp & 3;                                 // the 32 tensor-memory lanes this warp may read
        const int half = (warp - 2) >> 2;                        // which 128 accumulator columns
        int acc = 0; unsigned apar = 0;
        for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
            const int z = tile / tiles_per_batch, tt = tile % tiles_per_batch;
            int tm, tn;
            tile_coords(tt, g.tiles_m, g.tiles_n, g.gm, tm, tn);
            float run[128];
#pragma unroll
            for (int c = 0; c < 128; ++c) run[c] = 0.f;
            const bool cols_used = half * 128 < g.BN;
            for (int sg = 0; sg < nseg; ++sg) {
                mbar_wait(tfull0 + 8 * acc, apar);
                tc_fence_after();
                if (cols_used) {
                    const unsigned taddr = tmem_base + ((unsigned)(lg * 32) << 16) + acc * BN_MAX + half * 128;
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        unsigned v[32];
                        tmem_ld32(taddr + q * 32, v);
#pragma unroll
                        for (int c = 0; c < 32; ++c) run[q * 32 + c] += __uint_as_float(v[c]);
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(tempty0 + 8 * acc);
                if (++acc == 2) { acc = 0; apar ^= 1; }
            }
            const int row = tm * BM + lg * 32 + lane;
            if (row < g.M && cols_used) {
                long long roff = (long long)z * g.sC;
                if (g.rpg > 0) roff += (long long)(row / g.rpg) * g.gstride + (row % g.rpg);
                else roff += row;
                const int colb = tn * g.BN + half * 128;
                const int ncol = min(128, min(g.BN - half * 128, g.N - colb));
                if (g.out_kind == 0) {
                    double *C = (double *)g.C + roff + (long long)colb * g.ldc;
#pragma unroll
                    for (int c = 0; c < 128; ++c)
                        if (c < ncol) {
                            double *p = C + (long long)c * g.ldc;
                            *p = g.accumulate ? *p + (double)run[c] : (double)run[c];
                        }
                } else {
                    __nv_bfloat16 *C = (__nv_bfloat16 *)g.C + roff + (long long)colb * g.ldc;
#pragma unroll
                    for (int c = 0; c < 128; ++c)
                        if (c < ncol) {
                            __nv_bfloat16 b1, b2, b3;
                            split3(run[c], b1, b2, b3);
                            __nv_bfloat16 *p = C + (long long)c * g.ldc;
                            p[0] = b1; p[g.planeC] = b2; p[2 * g.planeC] = b3;
                        }
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        __syncwarp();
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
    }
}

// ---------------------------------------------------------------------------------------------------------------------------
// CTA-pair variant (cta_group::2): the two CTAs of a cluster, on the two SMs of a TPC, work on one 256 x BN tile.  Each CTA loads
// its own 128 rows of A and HALF of the B rows (the tensor cores of the pair read both halves), so bytes and TMA requests per SM
// drop by a third against the single-CTA kernel and a stage is 48 KB: four stages.  The MMAs are issued by the leader CTA (rank 0)
// for the pair; each CTA's tensor memory holds the accumulator rows of its own A rows and is drained by its own epilogue warps.
//   full[s]   (leader's copy): 1 arrival (the leader's producer, which also posts the bytes of BOTH CTAs' loads); the TMA loads of
//             both CTAs complete on it
//   empty[s]  (each CTA): tcgen05.commit of the leader, multicast to both CTAs
//   tfull[a]  (each CTA): tcgen05.commit of the leader, multicast
//   tempty[a] (leader's copy): 2 x 8 arrivals, the epilogue warps of both CTAs
constexpr int STAGES2 = 4, BK2 = 32, A_PLANE2 = BM * BK2 * 2, BH_PLANE_MAX = (BN_MAX / 2) * BK2 * 2;
constexpr int STAGE2_BYTES = 3 * A_PLANE2 + 3 * BH_PLANE_MAX;                 // 48 KiB
constexpr size_t SMEM2_BYTES = (size_t)STAGES2 * STAGE2_BYTES + 1024 + 128;

// shared::cluster address of the leader CTA's copy of a shared-memory object
__device__ __forceinline__ unsigned leader_addr(unsigned addr)
{
    unsigned out;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(out) : "r"(addr), "r"(0));
    return out;
}
__device__ __forceinline__ void tma_load_4d_2sm(unsigned dst, const CUtensorMap *tm, unsigned bar_leader, int c0, int c1, int c2, int c3)
{
    asm volatile("cp.async.bulk.tensor.4d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
                 ::"r"(dst), "l"(tm), "r"(bar_leader), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void mbar_arrive_cluster(unsigned bar) { asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(bar) : "memory"); }
__device__ __forceinline__ void umma_bf16_2sm(unsigned tmem_d, unsigned long long adesc, unsigned long long bdesc, unsigned idesc, unsigned accumulate)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit_2sm(unsigned bar)
{
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar), "h"((unsigned short)3) : "memory");
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(NT, 1)
tcgemm2_bf16x3_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, TcArgs g)
{
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = (unsigned char *)(((size_t)smem_raw + 1023) & ~(size_t)1023);
    unsigned long long *bars = (unsigned long long *)(smem + STAGES2 * STAGE2_BYTES);
    unsigned *tmem_slot = (unsigned *)(bars + 2 * STAGES2 + 4);
    const unsigned smem_u = smem_u32(smem);
    const unsigned full0 = smem_u32(bars), empty0 = smem_u32(bars + STAGES2), tfull0 = smem_u32(bars + 2 * STAGES2), tempty0 = smem_u32(bars + 2 * STAGES2 + 2);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned rank;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
    const bool leader = rank == 0;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES2; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(tfull0 + 8 * s, 1); mbar_init(tempty0 + 8 * s, 2 * NEPI); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(512) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    cluster_sync_all();
    tc_fence_after();
    const unsigned tmem_base = *tmem_slot;

    const int nk = (g.K + BK2 - 1) / BK2;
    const int nseg = (nk + g.seg_kb - 1) / g.seg_kb;
    const int tiles_per_batch = g.tiles_m * g.tiles_n;          // tiles_m counts 256-row tiles here
    const int total_tiles = tiles_per_batch * g.nb;
    const int pair = blockIdx.x >> 1, npairs = gridDim.x >> 1;
    const int bh = g.BN >> 1;                                   // B rows held by one CTA
    const int bh_plane = bh * BK2 * 2;
    const unsigned stage_tx = 2 * (3 * A_PLANE2 + 3 * bh_plane);

    if (warp == 0) {
        if (lane == 0) {
            int slot = 0; unsigned par = 1;
            for (int tile = pair; tile < total_tiles; tile += npairs) {
                const int z = tile / tiles_per_batch, tt = tile % tiles_per_batch;
                int tm, tn;
                tile_coords(tt, g.tiles_m, g.tiles_n, g.gm, tm, tn);
                for (int kb = 0; kb < nk; ++kb) {
                    mbar_wait(empty0 + 8 * slot, par);
                    const unsigned fb = leader_addr(full0 + 8 * slot), dst = smem_u + slot * STAGE2_BYTES;
                    if (leader) mbar_expect_tx(full0 + 8 * slot, stage_tx);
                    tma_load_4d_2sm(dst, &tmA, fb, kb * BK2, tm * 256 + (int)rank * BM, 0, g.za ? z : 0);
                    tma_load_4d_2sm(dst + 3 * A_PLANE2, &tmB, fb, kb * BK2, tn * g.BN + (int)rank * bh, 0, g.zb ? z : 0);
                    if (++slot == STAGES2) { slot = 0; par ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        if (lane == 0 && leader) {
            // D = F32, A = B = BF16, both K-major, N >> 3 at bit 17, M = 256 >> 4 at bit 24
            const unsigned idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((unsigned)(g.BN >> 3) << 17) | ((unsigned)(256 >> 4) << 24);
            int slot = 0; unsigned par = 0;
            int acc = 0; unsigned apar = 1;
            for (int tile = pair; tile < total_tiles; tile += npairs) {
                for (int kb0 = 0; kb0 < nk; kb0 += g.seg_kb) {
                    mbar_wait(tempty0 + 8 * acc, apar);
                    tc_fence_after();
                    const unsigned tacc = tmem_base + acc * BN_MAX;
                    const int kb1 = min(nk, kb0 + g.seg_kb);
                    // A segment of up to STAGES2 / 2 stages is issued in two passes over its stages: the five small products of every
                    // stage first, into the fresh accumulator where their truncation costs nothing, then the leading products a1 b1.
                    // Only those (two per stage) truncate at the size of the result, however long the segment is; half of the ring
                    // stays free for the loads of the next segment.
                    const bool two_pass = 2 * g.seg_kb <= STAGES2;
                    constexpr int PA[6] = {2, 0, 1, 1, 0, 0}, PB[6] = {0, 2, 1, 0, 1, 0};
                    for (int pass = two_pass ? 0 : 2; pass < (two_pass ? 2 : 3); ++pass) {         // 0: small products, 1: leading products, 2: both
                        int sl = slot; unsigned pr = par;
                        for (int kb = kb0; kb < kb1; ++kb) {
                            if (pass != 1) { mbar_wait(full0 + 8 * sl, pr); tc_fence_after(); }
                            const unsigned a0 = smem_u + sl * STAGE2_BYTES, b0 = a0 + 3 * A_PLANE2;
                            unsigned long long ad[3][BK2 / 16], bd[3][BK2 / 16];
#pragma unroll
                            for (int ks = 0; ks < BK2 / 16; ++ks)
#pragma unroll
                                for (int p = 0; p < 3; ++p) {
                                    ad[p][ks] = smem_desc<BK2>(a0 + p * A_PLANE2 + ks * 32);
                                    bd[p][ks] = smem_desc<BK2>(b0 + p * bh_plane + ks * 32);
                                }
#pragma unroll
                            for (int t = 0; t < 6; ++t) {
                                if ((pass == 0 && t == 5) || (pass == 1 && t != 5)) continue;
#pragma unroll
                                for (int ks = 0; ks < BK2 / 16; ++ks)
                                    umma_bf16_2sm(tacc, ad[PA[t]][ks], bd[PB[t]][ks], idesc, (kb != kb0) || t != 0 || ks != 0);
                            }
                            if (pass != 0) umma_commit_2sm(empty0 + 8 * sl);
                            if (++sl == STAGES2) { sl = 0; pr ^= 1; }
                        }
                        if (pass != 0) { slot = sl; par = pr; }
                    }
                    umma_commit_2sm(tfull0 + 8 * acc);
                    if (++acc == 2) { acc = 0; apar ^= 1; }
                }
            }
        }
    } else {
        const int lg = warp & 3;
        const int half = (warp - 2) >> 2;
        int acc = 0; unsigned apar = 0;
        for (int tile = pair; tile < total_tiles; tile += npairs) {
            const int z = tile / tiles_per_batch, tt = tile % tiles_per_batch;
            int tm, tn;
            tile_coords(tt, g.tiles_m, g.tiles_n, g.gm, tm, tn);
            float run[128];
#pragma unroll
            for (int c = 0; c < 128; ++c) run[c] = 0.f;
            const bool cols_used = half * 128 < g.BN;
            for (int sg = 0; sg < nseg; ++sg) {
                mbar_wait(tfull0 + 8 * acc, apar);
                tc_fence_after();
                if (cols_used) {
                    const unsigned taddr = tmem_base + ((unsigned)(lg * 32) << 16) + acc * BN_MAX + half * 128;
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        unsigned v[32];
                        tmem_ld32(taddr + q * 32, v);
#pragma unroll
                        for (int c = 0; c < 32; ++c) run[q * 32 + c] += __uint_as_float(v[c]);
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(leader_addr(tempty0 + 8 * acc));
                if (++acc == 2) { acc = 0; apar ^= 1; }
            }
            const int row = tm * 256 + (int)rank * BM + lg * 32 + lane;
            if (row < g.M && cols_used) {
                long long roff = (long long)z * g.sC;
                if (g.rpg > 0) roff += (long long)(row / g.rpg) * g.gstride + (row % g.rpg);
                else roff += row;
                const int colb = tn * g.BN + half * 128;
                const int ncol = min(128, min(g.BN - half * 128, g.N - colb));
                if (g.out_kind == 0) {
                    double *C = (double *)g.C + roff + (long long)colb * g.ldc;
#pragma unroll
                    for (int c = 0; c < 128; ++c)
                        if (c < ncol) {
                            double *p = C + (long long)c * g.ldc;
                            *p = g.accumulate ? *p + (double)run[c] : (double)run[c];
                        }
                } else {
                    __nv_bfloat16 *C = (__nv_bfloat16 *)g.C + roff + (long long)colb * g.ldc;
#pragma unroll
                    for (int c = 0; c < 128; ++c)
                        if (c < ncol) {
                            __nv_bfloat16 b1, b2, b3;
                            split3(run[c], b1, b2, b3);
                            __nv_bfloat16 *p = C + (long long)c * g.ldc;
                            p[0] = b1; p[g.planeC] = b2; p[2 * g.planeC] = b3;
                        }
                }
            }
        }
    }
    __syncwarp();
    tc_fence_before();
    cluster_sync_all();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
    }
}

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
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) == cudaSuccess && qr == cudaDriverEntryPointSuccess) fn = (EncodeFn)p;
        else (void)cudaGetLastError();
    }
    return fn;
}

// planes [3][batch][rows][ld] of bf16, K contiguous; dims (k, row, plane, batch)
bool make_map(EncodeFn enc, CUtensorMap *tm, const __nv_bfloat16 *p, int rows, int K, long long ld, long long plane, long long sbatch, int nb, int box_rows, int BK)
{
    if ((ld & 7) || (plane & 7) || (sbatch & 7) || (((size_t)p) & 15) || ld <= 0) return false;
    cuuint64_t dims[4] = {(cuuint64_t)K, (cuuint64_t)rows, 3, (cuuint64_t)(sbatch ? nb : 1)};
    cuuint64_t strides[3] = {(cuuint64_t)ld * 2, (cuuint64_t)plane * 2, (cuuint64_t)(sbatch ? sbatch : plane * 3) * 2};
    cuuint32_t box[4] = {(cuuint32_t)BK, (cuuint32_t)box_rows, 3, 1}, es[4] = {1, 1, 1, 1};
    if (strides[1] >= (1ull << 40) || strides[2] >= (1ull << 40)) return false;
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, (void *)p, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, BK == 64 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B,
               CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// X (FP64) -> three bf16 planes, row by row: out[p*plane + r*ldo + c] for c < n (columns n .. ldo-1 are zeroed)
// (source row r lives at (r / rpg) * gstride + (r % rpg) * ldx when rpg > 0: the window rows of X[m][nocc][nvir])
__global__ void __launch_bounds__(256) split_rows_kernel(const double *__restrict__ X, long long ldx, long long rows, int n, __nv_bfloat16 *__restrict__ out,
                                                         long long ldo, long long plane, int rpg, long long gstride)
{
    for (long long r = blockIdx.x; r < rows; r += gridDim.x) {
        const double *x = X + (rpg > 0 ? (r / rpg) * gstride + (r % rpg) * ldx : r * ldx);
        __nv_bfloat16 *o = out + r * ldo;
        for (int c = threadIdx.x; c < ldo; c += blockDim.x) {
            const double v = c < n ? x[c] : 0.0;
            const __nv_bfloat16 b1 = __double2bfloat16(v);
            const double r1 = v - (double)__bfloat162float(b1);
            const __nv_bfloat16 b2 = __double2bfloat16(r1);
            const __nv_bfloat16 b3 = __double2bfloat16(r1 - (double)__bfloat162float(b2));
            o[c] = b1; o[plane + c] = b2; o[2 * plane + c] = b3;
        }
    }
}

// X^T (FP64 [rows][ldx], n columns) -> three bf16 planes out[p*plane + c*ldo + r], 32 x 32 tiles through shared memory; the padding
// columns r in [rows, ldo) of every output row are zeroed
__global__ void __launch_bounds__(256) split_transpose_kernel(const double *__restrict__ X, long long ldx, int rows, int n, __nv_bfloat16 *__restrict__ out,
                                                              long long ldo, long long plane)
{
    __shared__ double s[32][33];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int r0 = blockIdx.x * 32, c0 = blockIdx.y * 32;
    for (int rr = ty; rr < 32; rr += 8) {
        const int r = r0 + rr, c = c0 + tx;
        s[rr][tx] = (r < rows && c < n) ? X[(long long)r * ldx + c] : 0.0;
    }
    __syncthreads();
    for (int cc = ty; cc < 32; cc += 8) {
        const int c = c0 + cc, r = r0 + tx;
        if (c < n && r < ldo) {
            const double v = s[tx][cc];
            const __nv_bfloat16 b1 = __double2bfloat16(v);
            const double r1 = v - (double)__bfloat162float(b1);
            const __nv_bfloat16 b2 = __double2bfloat16(r1);
            __nv_bfloat16 *o = out + (long long)c * ldo + r;
            o[0] = b1; o[plane] = b2; o[2 * plane] = __double2bfloat16(r1 - (double)__bfloat162float(b2));
        }
    }
}

// full[p*p_stride + r*row_stride + c] = packed[p][max(r,c), min(r,c)] as three bf16 planes (the tiling of expand_sym_kernel)
__global__ void __launch_bounds__(256) expand_sym_bf3_kernel(const double *__restrict__ packed, long long tri, int n, __nv_bfloat16 *__restrict__ full,
                                                             long long row_stride, long long p_stride, long long plane)
{
    __shared__ double s[32][33];
    const int t = blockIdx.x, p = blockIdx.y;
    int tr = (int)((sqrt(8.0 * t + 1.0) - 1.0) * 0.5);
    while ((tr + 1) * (tr + 2) / 2 <= t) ++tr;
    while (tr * (tr + 1) / 2 > t) --tr;
    const int tc = t - tr * (tr + 1) / 2;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const double *pk = packed + (long long)p * tri;
    __nv_bfloat16 *out = full + (long long)p * p_stride;
    auto put = [&](long long idx, double v) {
        const __nv_bfloat16 b1 = __double2bfloat16(v);
        const double r1 = v - (double)__bfloat162float(b1);
        const __nv_bfloat16 b2 = __double2bfloat16(r1);
        out[idx] = b1; out[plane + idx] = b2; out[2 * plane + idx] = __double2bfloat16(r1 - (double)__bfloat162float(b2));
    };
    for (int rr = ty; rr < 32; rr += 8) {
        const int r = tr * 32 + rr, c = tc * 32 + tx;
        s[rr][tx] = (r < n && c <= r) ? pk[(long long)r * (r + 1) / 2 + c] : 0.0;
    }
    __syncthreads();
    for (int rr = ty; rr < 32; rr += 8) {
        const int r = tr * 32 + rr, c = tc * 32 + tx;
        if (r < n && c < n) put((long long)r * row_stride + c, (c <= r) ? s[rr][tx] : s[tx][rr]);
        if (tr != tc) {
            const int r2 = tc * 32 + rr, c2 = tr * 32 + tx;
            if (r2 < n && c2 < n) put((long long)r2 * row_stride + c2, s[tx][rr]);
        }
    }
}

}  // namespace

cudaError_t risp_split_rows_bf3(const double *X, long long ldx, long long rows, int n, void *out, long long ldo, long long plane, int rpg,
                                long long gstride, cudaStream_t st)
{
    if (rows <= 0 || ldo <= 0) return cudaSuccess;
    split_rows_kernel<<<(unsigned)std::min<long long>(rows, 148 * 32), 256, 0, st>>>(X, ldx, rows, n, (__nv_bfloat16 *)out, ldo, plane, rpg, gstride);
    return cudaGetLastError();
}

cudaError_t risp_split_transpose_bf3(const double *X, long long ldx, int rows, int n, void *out, long long ldo, long long plane, cudaStream_t st)
{
    if (rows <= 0 || n <= 0) return cudaSuccess;
    dim3 grid((unsigned)((ldo + 31) / 32), (unsigned)((n + 31) / 32));
    split_transpose_kernel<<<grid, 256, 0, st>>>(X, ldx, rows, n, (__nv_bfloat16 *)out, ldo, plane);
    return cudaGetLastError();
}

cudaError_t risp_expand_sym_bf3(const double *packed, long long tri, int n, int np, void *full, long long row_stride, long long p_stride, long long plane,
                                cudaStream_t st)
{
    if (n <= 0 || np <= 0) return cudaSuccess;
    const int nt = (n + 31) / 32;
    dim3 grid(nt * (nt + 1) / 2, np);
    expand_sym_bf3_kernel<<<grid, 256, 0, st>>>(packed, tri, n, (__nv_bfloat16 *)full, row_stride, p_stride, plane);
    return cudaGetLastError();
}

// Returns cudaErrorNotSupported when the operands cannot be described by tensor maps (leading dimensions / strides not multiples
// of 8 elements, misaligned base, driver entry point missing): there is no other FP32 path, the caller reports the error.
namespace {
template <class S>
cudaError_t launch_shape(const TcGemmDesc &d, cudaStream_t st)
{
    EncodeFn enc = get_encode();
    if (!enc) return cudaErrorNotSupported;
    static bool attr[64] = {};
    static int sms[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (!attr[dev & 63]) {
        cudaError_t e = cudaFuncSetAttribute(tcgemm_bf16x3_kernel<S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::SMEM_BYTES);
        if (e != cudaSuccess) return e;
        cudaDeviceGetAttribute(&sms[dev & 63], cudaDevAttrMultiProcessorCount, dev);
        attr[dev & 63] = true;
    }
    TcArgs g;
    // column tile: the fewest tiles of at most BNCAP columns, each a multiple of 16 (N = 423 -> 2 x 224 instead of 256 + 167)
    const int nt = (d.N + S::BNCAP - 1) / S::BNCAP;
    g.BN = std::min(S::BNCAP, (((d.N + nt - 1) / nt) + 15) & ~15);
    g.M = d.M; g.N = d.N; g.K = d.K; g.nb = d.nb; g.za = d.sA != 0; g.zb = d.sB != 0;
    g.out_kind = d.out_kind; g.C = d.C; g.ldc = d.ldc; g.sC = d.sC; g.planeC = d.planeC; g.rpg = d.rpg; g.gstride = d.gstride; g.accumulate = d.accumulate;
    g.seg_kb = d.seg_kb > 0 ? d.seg_kb : 1;
    g.tiles_m = (d.M + BM - 1) / BM; g.tiles_n = (d.N + g.BN - 1) / g.BN;
    const long long total = (long long)g.tiles_m * g.tiles_n * d.nb;
    if (total >= (1ll << 31)) return cudaErrorNotSupported;
    CUtensorMap ma, mb;
    if (!make_map(enc, &ma, (const __nv_bfloat16 *)d.A, d.M, d.K, d.lda, d.planeA, d.sA, d.nb, BM, S::BK)) return cudaErrorNotSupported;
    if (!make_map(enc, &mb, (const __nv_bfloat16 *)d.B, d.N, d.K, d.ldb, d.planeB, d.sB, d.nb, g.BN, S::BK)) return cudaErrorNotSupported;
    const int grid = (int)std::min<long long>(total, sms[dev & 63]);
    g.gm = std::max(1, std::min(g.tiles_m, (sms[dev & 63] + g.tiles_n - 1) / g.tiles_n));
    tcgemm_bf16x3_kernel<S><<<grid, NT, S::SMEM_BYTES, st>>>(ma, mb, g);
    return cudaGetLastError();
}
}  // namespace

namespace {
cudaError_t launch_pair(const TcGemmDesc &d, cudaStream_t st)
{
    EncodeFn enc = get_encode();
    if (!enc) return cudaErrorNotSupported;
    static bool attr[64] = {};
    static int sms[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (!attr[dev & 63]) {
        cudaError_t e = cudaFuncSetAttribute(tcgemm2_bf16x3_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM2_BYTES);
        if (e != cudaSuccess) return e;
        cudaDeviceGetAttribute(&sms[dev & 63], cudaDevAttrMultiProcessorCount, dev);
        attr[dev & 63] = true;
    }
    TcArgs g;
    const int nt = (d.N + BN_MAX - 1) / BN_MAX;
    g.BN = std::min(BN_MAX, (((d.N + nt - 1) / nt) + 15) & ~15);
    g.M = d.M; g.N = d.N; g.K = d.K; g.nb = d.nb; g.za = d.sA != 0; g.zb = d.sB != 0;
    g.out_kind = d.out_kind; g.C = d.C; g.ldc = d.ldc; g.sC = d.sC; g.planeC = d.planeC; g.rpg = d.rpg; g.gstride = d.gstride; g.accumulate = d.accumulate;
    g.seg_kb = d.seg_kb > 0 ? d.seg_kb : STAGES2 / 2;      // two stages (64 k), issued in two passes
    g.tiles_m = (d.M + 255) / 256; g.tiles_n = (d.N + g.BN - 1) / g.BN;
    const long long total = (long long)g.tiles_m * g.tiles_n * d.nb;
    if (total >= (1ll << 31)) return cudaErrorNotSupported;
    CUtensorMap ma, mb;
    if (!make_map(enc, &ma, (const __nv_bfloat16 *)d.A, d.M, d.K, d.lda, d.planeA, d.sA, d.nb, BM, BK2)) return cudaErrorNotSupported;
    if (!make_map(enc, &mb, (const __nv_bfloat16 *)d.B, d.N, d.K, d.ldb, d.planeB, d.sB, d.nb, g.BN / 2, BK2)) return cudaErrorNotSupported;
    const int pairs = (int)std::min<long long>(total, sms[dev & 63] / 2);
    g.gm = std::max(1, std::min(g.tiles_m, (sms[dev & 63] / 2 + g.tiles_n - 1) / g.tiles_n));
    tcgemm2_bf16x3_kernel<<<2 * pairs, NT, SMEM2_BYTES, st>>>(ma, mb, g);
    return cudaGetLastError();
}
}  // namespace

cudaError_t risp_tcgemm(const TcGemmDesc &d, cudaStream_t st)
{
    if (d.M <= 0 || d.N <= 0 || d.nb <= 0) return cudaSuccess;
    if (d.K <= 0) return cudaErrorNotSupported;
    if (d.shape == 2) return launch_pair(d, st);
    // Measured on the 300-atom system with the MMAs switched off, the operand traffic alone costs 44 ms of the 50 ms of the Eq. 22
    // launch of the single-CTA kernel: about half of it scales with the bytes (L2 -> SM), half with the number of TMA row requests.
    // The CTA pair (shape 2) moves a third fewer bytes per SM and is what risp_matvec uses: 44.9 / 14.7 ms for Eq. 22 / 23 against
    // 50.7 / 16.9 ms.  Its accumulator hand-over crosses the SM pair and costs ~3000 cycles per segment, which is why its segments
    // are two stages long and issued in two passes (at one stage per segment it is slower than the single-CTA kernel: 57 ms).
    if (d.shape == 1) return launch_shape<TcShape<64, 128, 2>>(d, st);
    return launch_shape<TcShape<32, 256, 3>>(d, st);
}

namespace {
__global__ void sum_planes_kernel(const __nv_bfloat16 *__restrict__ p, long long plane, long long n, double *__restrict__ out, int accumulate)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const double v = (double)__bfloat162float(p[i]) + (double)__bfloat162float(p[plane + i]) + (double)__bfloat162float(p[2 * plane + i]);
        out[i] = accumulate ? out[i] + v : v;
    }
}
}  // namespace

// include/risp_debug.h: C[z][c][r] (+)= sum_k A[z][r][k] B[z][c][k] through the single-precision tensor-core path, FP64 in and out
extern "C" int risp_debug_tcgemm(int32_t M, int32_t N, int32_t K, int32_t nbatch, const double *A_dev, const double *B_dev, double *C_dev,
                                 int32_t accumulate, int32_t via_planes, int32_t seg_kb, int32_t shape, void *cuda_stream)
{
    if (M <= 0 || N <= 0 || K <= 0 || nbatch <= 0 || !A_dev || !B_dev || !C_dev) return RISP_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long ldk = (K + 7) & ~7LL, ldm = (M + 7) & ~7LL;
    const long long planeA = (long long)nbatch * M * ldk, planeB = (long long)nbatch * N * ldk, planeC = (long long)nbatch * N * ldm;
    __nv_bfloat16 *a = nullptr, *b = nullptr, *c = nullptr;
    int rc = RISP_ECUDA;
    do {
        if (cudaMalloc((void **)&a, 3 * planeA * 2) != cudaSuccess || cudaMalloc((void **)&b, 3 * planeB * 2) != cudaSuccess) { rc = RISP_ENOMEM; break; }
        if (via_planes && cudaMalloc((void **)&c, 3 * planeC * 2) != cudaSuccess) { rc = RISP_ENOMEM; break; }
        if (risp_split_rows_bf3(A_dev, K, (long long)nbatch * M, K, a, ldk, planeA, 0, 0, st) != cudaSuccess) break;
        if (risp_split_rows_bf3(B_dev, K, (long long)nbatch * N, K, b, ldk, planeB, 0, 0, st) != cudaSuccess) break;
        TcGemmDesc d;
        d.M = M; d.N = N; d.K = K; d.nb = nbatch;
        d.A = a; d.lda = ldk; d.planeA = planeA; d.sA = (long long)M * ldk;
        d.B = b; d.ldb = ldk; d.planeB = planeB; d.sB = (long long)N * ldk;
        d.rpg = 0; d.gstride = 0; d.seg_kb = seg_kb; d.shape = shape;
        if (via_planes) {
            if (cudaMemsetAsync(c, 0, 3 * planeC * 2, st) != cudaSuccess) break;
            d.C = c; d.ldc = ldm; d.sC = (long long)N * ldm; d.planeC = planeC; d.out_kind = 1; d.accumulate = 0;
        } else {
            d.C = C_dev; d.ldc = M; d.sC = (long long)N * M; d.planeC = 0; d.out_kind = 0; d.accumulate = accumulate;
        }
        if (risp_tcgemm(d, st) != cudaSuccess) break;
        if (via_planes) {
            // planes are [z][c][ldm]; the FP64 result is [z][c][M]
            for (long long row = 0; row < (long long)nbatch * N; ++row) {
                sum_planes_kernel<<<(M + 255) / 256, 256, 0, st>>>(c + row * ldm, planeC, M, C_dev + row * M, accumulate);
            }
        }
        if (cudaStreamSynchronize(st) != cudaSuccess) break;
        rc = RISP_OK;
    } while (0);
    (void)cudaGetLastError();
    cudaFree(a); cudaFree(b); cudaFree(c);
    return rc;
}
