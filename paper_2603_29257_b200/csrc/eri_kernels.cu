// eri_kernels.cu -- kernels built on the integral engine of eri.cuh.
//
//   eri_fill      (mu nu|P) blocks written to a dense [P][mu][nu] buffer: K-tensor build (Eq. 20-21),
//                 the two-centre metrics (P|Q) (Eq. 3, 26) and the parity getter risp_eri3c_shell.
//   dens_to_e0    Eq. 14 prologue: symmetrised AO density block -> e0 space (adjoint HRR + spherical transform).
//   j_pass1       R_mQ = sum_z (Q|z) D_z^m        (Eq. 14), integrals generated on the fly.
//   j_pass2       U_z^m = sum_P (z|P) R~_mP       (Eq. 16), integrals regenerated.
//   e0_to_U       Eq. 16 epilogue: e0 space -> symmetric AO matrix U^m.
//
// Mapping (J passes): a warp generates the integrals of 32 (pair, aux-centre) tasks at once, one task per lane,
// and parks them in shared memory; then the lanes switch roles to the m trial vectors and contract the parked
// integrals with D (pass 1) or R~ (pass 2) -- each integral is generated once and used for all m vectors.
#include "ctx.h"

using namespace risp_eri;

namespace {

constexpr int MS = RISP_MS;  // padded trial-vector stride of the e0-space / aux-space arrays

// ------------------------------------------------------------------------------------------------- eri_fill
template <int LA, int LB, bool HASP, bool ERF>
__global__ void __launch_bounds__(128) eri_fill_kernel(const ShellPair *__restrict__ pairs, int npairs, const PrimPair *__restrict__ prims,
                                                       const AuxCentre *__restrict__ cen, int ncen, OpParams op,
                                                       const double *__restrict__ boys_tab, double *__restrict__ out,
                                                       long long stride_q, long long ld, int mirror)
{
    constexpr int NE = ne_of(LA, LB), NC = HASP ? 4 : 1;
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int pi = (int)(t / ncen), ci = (int)(t % ncen);
    if (pi >= npairs) return;
    const ShellPair sp = pairs[pi];
    const AuxCentre ax = cen[ci];
    double e0[NC][NE];
#pragma unroll
    for (int c = 0; c < NC; ++c)
#pragma unroll
        for (int e = 0; e < NE; ++e) e0[c][e] = 0.0;
    for (int k = 0; k < sp.npp; ++k) {
        const PrimPair pp = prims[sp.ppoff + k];
        eri_e0_prim<LA, LB, HASP, ERF>(pp, sp.Ax, sp.Ay, sp.Az, ax, op, boys_tab, [&](int e, int c, double v) { e0[c][e] += v; });
    }
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        int q = c == 0 ? ax.qs : (ax.qp < 0 ? -1 : ax.qp + c - 1);
        if (q < 0) continue;
        double blk[2 * LA + 1][2 * LB + 1];
        e0_to_sph<LA, LB>(e0[c], sp.ABx, sp.ABy, sp.ABz, blk);
        double *o = out + (long long)q * stride_q;
#pragma unroll
        for (int i = 0; i < 2 * LA + 1; ++i)
#pragma unroll
            for (int j = 0; j < 2 * LB + 1; ++j) {
                o[(long long)(sp.aoA + i) * ld + sp.aoB + j] = blk[i][j];
                if (mirror && sp.shA != sp.shB) o[(long long)(sp.aoB + j) * ld + sp.aoA + i] = blk[i][j];
            }
    }
}

// ------------------------------------------------------------------------------------------------- density -> e0
// D: rows [r0, ...) of the plain (unsymmetrised) AO density matrices of mj trial vectors (leading dimension ld, vector stride
// mstride).  Only sym(D) matters for a lower-triangular pair (reading G13): D-bar(A,B) = adjoint[D_AB + D_BA^T].
//   mode 0  all rows present (r0 = 0): both blocks read here, D-bar written.
//   mode 1  panel holds the rows of shell A:  D-bar += adjoint[D_AB]           (pairs [p0, p1) of the aoA-sorted list)
//   mode 2  panel holds the rows of shell B:  D-bar += adjoint[D_BA^T], A != B (pairs perm[p0 .. p1) of the aoB-sorted list)
// Modes 1 and 2 visit every pair once each over all panels; D-bar is zeroed before.
template <int LA, int LB>
__global__ void __launch_bounds__(128) dens_to_e0_kernel(const ShellPair *__restrict__ pairs, const int *__restrict__ perm, int p0, int p1,
                                                         long long e_off, int mj, int lane0, int m_total, int r0, long long ld, long long mstride, int mode,
                                                         const double *__restrict__ D, double *__restrict__ dbar)
{
    constexpr int NE = ne_of(LA, LB);
    const int mi = threadIdx.x;
    int pi = p0 + blockIdx.x * blockDim.y + threadIdx.y;
    if (pi >= p1) return;
    if (mi >= mj) {
        // dense mode overwrites D-bar lane by lane: the lanes beyond the batch are cleared here, so that neither pass ever works on
        // what an earlier, larger batch left there
        if (mode == 0 && lane0 + mi >= m_total && lane0 + mi < MS) {
            double *z = dbar + (e_off + (long long)pi * NE) * MS + lane0 + mi;
#pragma unroll
            for (int e = 0; e < NE; ++e) z[(long long)e * MS] = 0.0;
        }
        return;
    }
    if (mode == 2) pi = perm[pi];
    const ShellPair sp = pairs[pi];
    const bool diag = sp.shA == sp.shB;
    if (mode == 2 && diag) return;
    const double *Dm = D + (long long)mi * mstride;
    double d[2 * LA + 1][2 * LB + 1];
#pragma unroll
    for (int i = 0; i < 2 * LA + 1; ++i)
#pragma unroll
        for (int j = 0; j < 2 * LB + 1; ++j) {
            double v;
            if (mode == 2) v = Dm[(long long)(sp.aoB - r0 + j) * ld + sp.aoA + i];
            else {
                v = Dm[(long long)(sp.aoA - r0 + i) * ld + sp.aoB + j];
                if (mode == 0 && !diag) v += Dm[(long long)(sp.aoB + j) * ld + sp.aoA + i];
            }
            d[i][j] = v;
        }
    double out[NE];
    sph_to_e0_adjoint<LA, LB>(d, sp.ABx, sp.ABy, sp.ABz, out);
    double *dst = dbar + (e_off + (long long)pi * NE) * MS + lane0 + mi;
#pragma unroll
    for (int e = 0; e < NE; ++e) {
        if (mode == 0) dst[(long long)e * MS] = out[e];
        else dst[(long long)e * MS] += out[e];
    }
}

// U-bar -> rows [r0, ...) of the symmetric AO matrix U.
//   mode 0  dense (r0 = 0): the block and its transpose.   mode 1  block at the rows of shell A (aoA-sorted range).
//   mode 2  transposed block at the rows of shell B, A != B (aoB-sorted range through perm).
template <int LA, int LB>
__global__ void __launch_bounds__(128) e0_to_U_kernel(const ShellPair *__restrict__ pairs, const int *__restrict__ perm, int p0, int p1,
                                                      long long e_off, int mj, int lane0, int r0, long long ld, long long mstride, int mode,
                                                      const double *__restrict__ ubar, double *__restrict__ U)
{
    constexpr int NE = ne_of(LA, LB);
    const int mi = threadIdx.x;
    int pi = p0 + blockIdx.x * blockDim.y + threadIdx.y;
    if (pi >= p1 || mi >= mj) return;
    if (mode == 2) pi = perm[pi];
    const ShellPair sp = pairs[pi];
    const bool diag = sp.shA == sp.shB;
    if (mode == 2 && diag) return;
    double e0[NE];
#pragma unroll
    for (int e = 0; e < NE; ++e) e0[e] = ubar[(e_off + (long long)pi * NE + e) * MS + lane0 + mi];
    double blk[2 * LA + 1][2 * LB + 1];
    e0_to_sph<LA, LB>(e0, sp.ABx, sp.ABy, sp.ABz, blk);
    double *Um = U + (long long)mi * mstride;
#pragma unroll
    for (int i = 0; i < 2 * LA + 1; ++i)
#pragma unroll
        for (int j = 0; j < 2 * LB + 1; ++j) {
            if (mode != 2) Um[(long long)(sp.aoA - r0 + i) * ld + sp.aoB + j] = blk[i][j];
            if (mode == 2 || (mode == 0 && !diag)) Um[(long long)(sp.aoB - r0 + j) * ld + sp.aoA + i] = blk[i][j];
        }
}

// ------------------------------------------------------------------------------------------------- J passes
constexpr int JW = 4;   // warps per CTA

// Both passes have the same shape.  A warp step covers PW shell pairs x CW = 32 / PW aux centres, one (pair, centre) task per lane
// (lane = s * CW + a): every lane generates the NE x 4 contracted [e0|P) integrals of its task (s and the three p functions of the
// centre share one recursion) and parks them in shared memory as G[kappa = s NE + e][c CW + a] with row stride KS.  Then the
// warp contracts the parked block with the trial-vector operand ON THE FP64 TENSOR CORES (DMMA.8x8x4): the contraction is a
// dense [.. x ..] x [.. x 32 vectors] product, 2 m flops per integral, and as scalar FMAs with their shared-memory operand
// loads it used more issue slots than the integral generation itself.
//   pass 1 (Eq. 14):  R[(c, a)][m]     += sum_kappa G[kappa][(c, a)] Dbar[kappa][m]      A = G^T (rows (c,a)), B = Dbar rows
//   pass 2 (Eq. 16):  Ubar[kappa][m]   += sum_(c,a) G[kappa][(c, a)] R~[(a, c)][m]        A = G (rows kappa),   B = R~ by centre
// Fragment maps of mma.m8n8k4.f64: lane (q = lane / 4, r = lane % 4) holds A[q][r], B[r][q], C[q][2r], C[q][2r + 1].  The row
// strides are chosen so that the 32 lanes of an A-fragment load hit 32 different 8-byte words: pass 1 reads G[4t + r][8 mi + q]
// (KS = 40: r KS mod 32 = 0, 8, 16, 24), pass 2 reads G[8 mi + q][4t + r] (KS = 4 CW + 4: q KS mod 32 = 0, 4, ..., 28).
__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// Both passes are bound by FP64 arithmetic only if the global loads (primitive pairs, operands) are in flight early: at 8-16
// warps per SM nothing else hides their latency.  So the next primitive pair is fetched while the current one is processed.
// base = parking address of this lane's task: element (e, c) lives at base[e * KS + c * CW].
template <int LA, int LB, int KS, int CW>
__device__ __forceinline__ void park_integrals(double *__restrict__ base, bool valid, const ShellPair &sp, const PrimPair *__restrict__ prims,
                                               const AuxCentre &ax, const double *__restrict__ boys_tab)
{
    constexpr int NE = ne_of(LA, LB);
    constexpr bool REG = NE * 4 <= 36;          // small classes accumulate the contraction over primitives in registers
    if constexpr (REG) {
        double a[NE * 4];
#pragma unroll
        for (int k = 0; k < NE * 4; ++k) a[k] = 0.0;
        if (valid) {
            OpParams op{1.0, 0.0, 0.0};
            PrimPair pp = prims[sp.ppoff];
            for (int k = 0; k < sp.npp; ++k) {
                const PrimPair nxt = prims[sp.ppoff + min(k + 1, sp.npp - 1)];
                eri_e0_prim<LA, LB, true, false>(pp, sp.Ax, sp.Ay, sp.Az, ax, op, boys_tab, [&](int e, int c, double v) { a[e * 4 + c] += v; });
                pp = nxt;
            }
        }
#pragma unroll
        for (int e = 0; e < NE; ++e)
#pragma unroll
            for (int c = 0; c < 4; ++c) base[e * KS + c * CW] = a[e * 4 + c];
    } else {
#pragma unroll
        for (int e = 0; e < NE; ++e)
#pragma unroll
            for (int c = 0; c < 4; ++c) base[e * KS + c * CW] = 0.0;
        if (valid) {
            OpParams op{1.0, 0.0, 0.0};      // dp, dd: no prefetch, the recursion needs every register
            for (int k = 0; k < sp.npp; ++k) {
                const PrimPair pp = prims[sp.ppoff + k];
                eri_e0_prim<LA, LB, true, false>(pp, sp.Ax, sp.Ay, sp.Az, ax, op, boys_tab, [&](int e, int c, double v) { base[e * KS + c * CW] += v; });
            }
        }
    }
}

// R~ by centre: RtC[(centre*4 + comp)*MS + lane], zero where a centre has no s or no p function and for the padding centres up
// to a multiple of 32 -- pass 2 then reads its contraction operand without the (qs, qp) indirection
__global__ void rt_by_centre_kernel(const double *__restrict__ Rt, const AuxCentre *__restrict__ cen, int ncen, double *__restrict__ RtC)
{
    const int lane = threadIdx.x, k = blockIdx.x, ci = k >> 2, c = k & 3;
    int q = -1;
    if (ci < ncen) q = c == 0 ? cen[ci].qs : (cen[ci].qp < 0 ? -1 : cen[ci].qp + c - 1);
    RtC[(long long)k * MS + lane] = q >= 0 ? Rt[(long long)q * MS + lane] : 0.0;
}

template <int LA, int LB>
struct Pass2Cfg {
    static constexpr int NE = ne_of(LA, LB);
    // pairs per warp step: as many as keep the accumulator tile (8-row blocks of PW NE rows x 32 vectors) at <= 32 doubles per lane
    static constexpr int PW = NE <= 6 ? 4 : (NE <= 16 ? 2 : 1);
    static constexpr int CW = 32 / PW, KS = 4 * CW + 4, MROWS = PW * NE, M8 = (MROWS + 7) / 8 * 8, MT = M8 / 8;
    static constexpr size_t SMEM_PER_WARP = (size_t)M8 * KS * sizeof(double);
};

// pass 2: a warp owns PW pairs and walks over all aux centres, CW per step.  ubar[(e_off + pair*NE + e)*MS + m]
template <int LA, int LB>
__global__ void __launch_bounds__(32 * JW) j_pass2_kernel(const ShellPair *__restrict__ pairs, int npairs, const PrimPair *__restrict__ prims,
                                                          const AuxCentre *__restrict__ cen, int ncen, const double *__restrict__ boys_tab,
                                                          const double *__restrict__ RtC, long long e_off, double *__restrict__ ubar, int njn)
{
    using C = Pass2Cfg<LA, LB>;
    constexpr int NE = C::NE, PW = C::PW, CW = C::CW, KS = C::KS, MROWS = C::MROWS, M8 = C::M8, MT = C::MT;
    extern __shared__ double smem[];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    double *g = smem + (size_t)w * M8 * KS;
    const int pg = (blockIdx.x * JW + w) * PW;
    if (pg >= npairs) return;
    const int s = lane / CW, a = lane % CW, q = lane >> 2, r = lane & 3;
    const bool pvalid = pg + s < npairs;
    const ShellPair sp = pairs[min(pg + s, npairs - 1)];
    for (int i = MROWS * KS + lane; i < M8 * KS; i += 32) g[i] = 0.0;      // padding rows of the last 8-row block
    double acc[MT][4][2];
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    AuxCentre ax = cen[min(a, ncen - 1)];
    double *base = g + (size_t)s * NE * KS + a;
    for (int c0 = 0; c0 < ncen; c0 += CW) {
        const bool valid = pvalid && c0 + a < ncen;
        const AuxCentre ax_next = cen[min(c0 + CW + a, ncen - 1)];
        park_integrals<LA, LB, KS, CW>(base, valid, sp, prims, ax, boys_tab);
        ax = ax_next;
        __syncwarp();
#pragma unroll 4
        for (int t = 0; t < CW; ++t) {              // K = 4 CW = (c, a) in steps of 4
            const int kk = 4 * t + r, c = kk / CW, aa = kk % CW;
            const double *rc = RtC + ((long long)(c0 + aa) * 4 + c) * MS + q;      // padding centres carry zero integrals and zero R~
            double bf[4], af[MT];
#pragma unroll
            for (int j = 0; j < 4; ++j) bf[j] = j < njn ? rc[8 * j] : 0.0;
#pragma unroll
            for (int i = 0; i < MT; ++i) af[i] = g[(8 * i + q) * KS + kk];
#pragma unroll
            for (int i = 0; i < MT; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
        __syncwarp();
    }
#pragma unroll
    for (int i = 0; i < MT; ++i) {
        const int row = 8 * i + q;
        if (row < MROWS && pg + row / NE < npairs) {
            double *dst = ubar + (e_off + (long long)pg * NE + row) * MS + 2 * r;
#pragma unroll
            for (int j = 0; j < 4; ++j) *reinterpret_cast<double2 *>(dst + 8 * j) = make_double2(acc[i][j][0], acc[i][j][1]);
        }
    }
}

// pass 1: CTA = (pair chunk, 8 aux centres); warp step = 4 pairs x 8 centres.
// Rpart[((chunk_global * ncen_pad + centre) * 4 + comp) * MS + mi]
constexpr int P1_KS = 40;
template <int LA, int LB>
__global__ void __launch_bounds__(32 * JW) j_pass1_kernel(const ShellPair *__restrict__ pairs, int npairs, int chunk, int chunk_base,
                                                          const PrimPair *__restrict__ prims, const AuxCentre *__restrict__ cen, int ncen,
                                                          int ncen_pad, const double *__restrict__ boys_tab, const double *__restrict__ dbar,
                                                          long long e_off, double *__restrict__ Rpart, int njn)
{
    // SKEW: with an even NE the four pair slots of a step would start 0 mod 16 doubles apart and their parking stores would
    // collide four ways; 8 doubles of skew per slot bring the stores to the two-wavefront optimum (the fragment loads then
    // collide two ways only in the k-steps that straddle two slots)
    constexpr int NE = ne_of(LA, LB), KS = P1_KS, KROWS = 4 * NE, SKEW = (NE % 2 == 0) ? 8 : 0, WARP_DOUBLES = KROWS * KS + 4 * SKEW;
    extern __shared__ double smem[];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    double *g = smem + (size_t)w * WARP_DOUBLES;
    const int p_begin = blockIdx.x * chunk, p_end = min(npairs, p_begin + chunk);
    const int slot = lane >> 3, a = lane & 7, q = lane >> 2, r = lane & 3;
    const int ci = blockIdx.y * 8 + a;
    const bool cvalid = ci < ncen;
    const AuxCentre ax = cen[cvalid ? ci : 0];
    double acc[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    constexpr bool LEAN = NE > 10;          // dp, dd: the recursion already spills; no shell-pair prefetch
    ShellPair sp = pairs[min(p_begin + w * 4 + slot, p_end - 1)];
    double *base = g + (size_t)slot * (NE * KS + SKEW) + a;
    constexpr bool PRE = NE <= 4;           // ss, ps: the operand fragments of the whole step are fetched before the integrals are generated
    for (int pg = p_begin + w * 4; pg < p_end; pg += JW * 4) {
        const int pi = pg + slot;
        const bool valid = cvalid && pi < p_end;
        if constexpr (LEAN) sp = pairs[min(pi, p_end - 1)];
        ShellPair sp_next;
        if constexpr (!LEAN) sp_next = pairs[min(pi + JW * 4, p_end - 1)];
        const double *db = dbar + (e_off + (long long)pg * NE) * MS + q;
        double bpre[PRE ? NE : 1][4];
        if constexpr (PRE) {
#pragma unroll
            for (int t = 0; t < NE; ++t) {
                const int kk = 4 * t + r;
                const bool kv = pg + kk / NE < p_end;
#pragma unroll
                for (int j = 0; j < 4; ++j) bpre[t][j] = (kv && j < njn) ? db[(long long)kk * MS + 8 * j] : 0.0;
            }
        }
        park_integrals<LA, LB, KS, 8>(base, valid, sp, prims, ax, boys_tab);
        if constexpr (!LEAN) sp = sp_next;
        __syncwarp();
#pragma unroll(PRE ? NE : 4)
        for (int t = 0; t < NE; ++t) {              // K = 4 NE = (pair, e) in steps of 4
            const int kk = 4 * t + r;
            const bool kv = pg + kk / NE < p_end;   // rows of pairs beyond the chunk: parked zeros, operand not read
            double bf[4], af[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                if constexpr (PRE) bf[j] = bpre[t][j];
                else bf[j] = (kv && j < njn) ? db[(long long)kk * MS + 8 * j] : 0.0;
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) af[i] = g[kk * KS + (kk / NE) * SKEW + 8 * i + q];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
        __syncwarp();
    }
    // cross-warp reduction (fixed order -> deterministic) in a dedicated region after the parking area: red[w][k = a*4 + c][m];
    // this lane holds, for component c = i, centre a = q and vectors m = 8j + 2r, 8j + 2r + 1
    __syncthreads();
    double *red = smem + (size_t)JW * WARP_DOUBLES;   // [JW][32][32]
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
            *reinterpret_cast<double2 *>(&red[(w * 32 + q * 4 + i) * 32 + 8 * j + 2 * r]) = make_double2(acc[i][j][0], acc[i][j][1]);
    __syncthreads();
    for (int k = w; k < 32; k += JW) {
        double s = 0.0;
#pragma unroll
        for (int ww = 0; ww < JW; ++ww) s += red[(ww * 32 + k) * 32 + lane];
        const int aa = k >> 2, c = k & 3;
        const int cc = blockIdx.y * 8 + aa;
        if (cc < ncen) Rpart[(((long long)(chunk_base + blockIdx.x) * ncen_pad + cc) * 4 + c) * MS + lane] = s;
    }
}

// R[q][lane] = sum over pair chunks of the pass-1 partials, fixed order: warp w of 8 takes chunks w, w+8, ... into four
// interleaved partial sums (independent loads in flight), then the 8 warps' sums are added in order
__global__ void __launch_bounds__(256) j_reduce_R_kernel(const double *__restrict__ Rpart, int nchunks, const AuxCentre *__restrict__ cen, int ncen,
                                                         int ncen_pad, double *__restrict__ R)
{
    __shared__ double part[8][32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, k = blockIdx.x;          // k = centre*4 + comp
    const int ci = k >> 2, c = k & 3;
    const int q = c == 0 ? cen[ci].qs : (cen[ci].qp < 0 ? -1 : cen[ci].qp + c - 1);
    if (q < 0) return;
    const long long stride = (long long)ncen_pad * 4 * MS;
    const double *src = Rpart + ((long long)ci * 4 + c) * MS + lane;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
    int ch = w;
    for (; ch + 24 < nchunks; ch += 32) {
        s0 += src[(long long)ch * stride];
        s1 += src[(long long)(ch + 8) * stride];
        s2 += src[(long long)(ch + 16) * stride];
        s3 += src[(long long)(ch + 24) * stride];
    }
    for (; ch < nchunks; ch += 8) s0 += src[(long long)ch * stride];
    part[w][lane] = (s0 + s1) + (s2 + s3);
    __syncthreads();
    if (w == 0) {
        double s = 0.0;
#pragma unroll
        for (int ww = 0; ww < 8; ++ww) s += part[ww][lane];
        R[(long long)q * MS + lane] = s;
    }
}

template <class F>
inline void dispatch_class(int la, int lb, F &&f)
{
    if (la == 0) f(std::integral_constant<int, 0>{}, std::integral_constant<int, 0>{});
    else if (la == 1 && lb == 0) f(std::integral_constant<int, 1>{}, std::integral_constant<int, 0>{});
    else if (la == 1) f(std::integral_constant<int, 1>{}, std::integral_constant<int, 1>{});
    else if (lb == 0) f(std::integral_constant<int, 2>{}, std::integral_constant<int, 0>{});
    else if (lb == 1) f(std::integral_constant<int, 2>{}, std::integral_constant<int, 1>{});
    else f(std::integral_constant<int, 2>{}, std::integral_constant<int, 2>{});
}

template <class K>
cudaError_t ensure_smem(K kernel, size_t bytes)
{
    if (bytes <= 48 * 1024) return cudaSuccess;
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);      // per device, cheap: set on every launch
}

}  // namespace

// ===================================================================================================== host wrappers
cudaError_t risp_eri_fill(int la, int lb, bool hasp, bool erf_op, const ShellPair *pairs, int npairs, const PrimPair *prims,
                          const AuxCentre *cen, int ncen, OpParams op, const double *boys_tab, double *out, long long stride_q,
                          long long ld, int mirror, cudaStream_t st)
{
    if (npairs <= 0 || ncen <= 0) return cudaSuccess;
    long long total = (long long)npairs * ncen;
    unsigned grid = (unsigned)((total + 127) / 128);
    dispatch_class(la, lb, [&](auto LA, auto LB) {
        constexpr int A = decltype(LA)::value, B = decltype(LB)::value;
        if (hasp) {
            if (erf_op) eri_fill_kernel<A, B, true, true><<<grid, 128, 0, st>>>(pairs, npairs, prims, cen, ncen, op, boys_tab, out, stride_q, ld, mirror);
            else eri_fill_kernel<A, B, true, false><<<grid, 128, 0, st>>>(pairs, npairs, prims, cen, ncen, op, boys_tab, out, stride_q, ld, mirror);
        } else {
            if (erf_op) eri_fill_kernel<A, B, false, true><<<grid, 128, 0, st>>>(pairs, npairs, prims, cen, ncen, op, boys_tab, out, stride_q, ld, mirror);
            else eri_fill_kernel<A, B, false, false><<<grid, 128, 0, st>>>(pairs, npairs, prims, cen, ncen, op, boys_tab, out, stride_q, ld, mirror);
        }
    });
    return cudaGetLastError();
}

cudaError_t risp_dens_to_e0(const PairClass &pc, int p0, int p1, int mj, int lane0, int m_total, int r0, long long ld, long long mstride, int mode,
                            const double *D, double *dbar, cudaStream_t st)
{
    if (p1 <= p0) return cudaSuccess;
    dim3 block(32, 4), grid((p1 - p0 + 3) / 4);
    dispatch_class(pc.la, pc.lb, [&](auto LA, auto LB) {
        dens_to_e0_kernel<decltype(LA)::value, decltype(LB)::value><<<grid, block, 0, st>>>(pc.d_pairs, pc.d_permB, p0, p1, pc.e_off, mj, lane0, m_total, r0,
                                                                                            ld, mstride, mode, D, dbar);
    });
    return cudaGetLastError();
}

cudaError_t risp_e0_to_U(const PairClass &pc, int p0, int p1, int mj, int lane0, int r0, long long ld, long long mstride, int mode,
                         const double *ubar, double *U, cudaStream_t st)
{
    if (p1 <= p0) return cudaSuccess;
    dim3 block(32, 4), grid((p1 - p0 + 3) / 4);
    dispatch_class(pc.la, pc.lb, [&](auto LA, auto LB) {
        e0_to_U_kernel<decltype(LA)::value, decltype(LB)::value><<<grid, block, 0, st>>>(pc.d_pairs, pc.d_permB, p0, p1, pc.e_off, mj, lane0, r0, ld,
                                                                                         mstride, mode, ubar, U);
    });
    return cudaGetLastError();
}

cudaError_t risp_j_pass1(const PairClass &pc, const PrimPair *prims, const AuxCentre *cen, int ncen, int ncen_pad, const double *boys_tab,
                         const double *dbar, double *Rpart, int m, cudaStream_t st)
{
    if (pc.npairs <= 0) return cudaSuccess;
    cudaError_t err = cudaSuccess;
    dispatch_class(pc.la, pc.lb, [&](auto LA, auto LB) {
        constexpr int A = decltype(LA)::value, B = decltype(LB)::value;
        size_t smem = ((size_t)JW * (4 * ne_of(A, B) * P1_KS + 32) + (size_t)JW * 32 * 32) * sizeof(double);
        err = ensure_smem(j_pass1_kernel<A, B>, smem);
        if (err != cudaSuccess) return;
        dim3 grid(pc.nchunks, (ncen + 7) / 8);
        j_pass1_kernel<A, B><<<grid, 32 * JW, smem, st>>>(pc.d_pairs, pc.npairs, pc.chunk, pc.chunk_base, prims, cen, ncen, ncen_pad, boys_tab,
                                                          dbar, pc.e_off, Rpart, (m + 7) / 8);
    });
    return err != cudaSuccess ? err : cudaGetLastError();
}

cudaError_t risp_j_reduce_R(const double *Rpart, int nchunks, const AuxCentre *cen, int ncen, int ncen_pad, double *R, cudaStream_t st)
{
    j_reduce_R_kernel<<<ncen * 4, 256, 0, st>>>(Rpart, nchunks, cen, ncen, ncen_pad, R);
    return cudaGetLastError();
}

cudaError_t risp_rt_by_centre(const double *Rt, const AuxCentre *cen, int ncen, double *RtC, cudaStream_t st)
{
    const int ncen32 = (ncen + 31) / 32 * 32;
    rt_by_centre_kernel<<<ncen32 * 4, 32, 0, st>>>(Rt, cen, ncen, RtC);
    return cudaGetLastError();
}

cudaError_t risp_j_pass2(const PairClass &pc, const PrimPair *prims, const AuxCentre *cen, int ncen, const double *boys_tab, const double *Rt,
                         double *ubar, int m, cudaStream_t st)
{
    if (pc.npairs <= 0) return cudaSuccess;
    cudaError_t err = cudaSuccess;
    dispatch_class(pc.la, pc.lb, [&](auto LA, auto LB) {
        constexpr int A = decltype(LA)::value, B = decltype(LB)::value;
        using C = Pass2Cfg<A, B>;
        size_t smem = (size_t)JW * C::SMEM_PER_WARP;
        err = ensure_smem(j_pass2_kernel<A, B>, smem);
        if (err != cudaSuccess) return;
        const int per_cta = JW * C::PW;
        j_pass2_kernel<A, B><<<(pc.npairs + per_cta - 1) / per_cta, 32 * JW, smem, st>>>(pc.d_pairs, pc.npairs, prims, cen, ncen, boys_tab, Rt, pc.e_off,
                                                                                         ubar, (m + 7) / 8);
    });
    return err != cudaSuccess ? err : cudaGetLastError();
}
