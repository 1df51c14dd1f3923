// ctx.h -- the library context and the internal interfaces between the .cu files.
#pragma once
#include "common.cuh"
#include "eri.cuh"
#include <type_traits>

#define RISP_MS 32   // padded trial-vector stride of R, R~, D-bar, U-bar (one lane per trial vector)
#define RISP_NEV 16

// Temporaries of one call: everything allocated through it is released when it goes out of scope (any early return included).
struct DevScratch {
    std::vector<void *> v;
    template <class T>
    cudaError_t alloc(T *&p, size_t count)
    {
        p = nullptr;
        if (count == 0) return cudaSuccess;
        cudaError_t e = cudaMalloc((void **)&p, count * sizeof(T));
        if (e == cudaSuccess) v.push_back(p);
        return e;
    }
    template <class T>
    void release(T *&p)
    {
        for (auto &q : v) if (q == (void *)p) { cudaFree(q); q = nullptr; }
        p = nullptr;
    }
    ~DevScratch() { for (void *q : v) if (q) cudaFree(q); }
};

struct PairClass {                 // kept shell pairs of one (la >= lb) class, sorted by the first AO of shell A
    int la, lb, npairs;
    risp_eri::ShellPair *d_pairs;  // device
    long long e_off;               // first e0 row of this class in D-bar / U-bar
    int chunk, nchunks, chunk_base; // pass-1 pair chunking (chunk_base: global index of the class's first chunk)
    std::vector<int> h_aoA;        // host copy of sp.aoA (ascending): row panels of the J transforms are pair ranges
    int *d_permB = nullptr;        // pair indices sorted by sp.aoB (device), and the sorted aoB values (host)
    std::vector<int> h_aoB;
};

// Plan of one risp_matvec (sizes depend on m and on what the HBM budget leaves after the K tensors).
struct MatvecPlan {
    int mj = 0;                    // trial vectors per sub-batch of the AO<->MO transforms of the J path
    int prow = 0;                  // AO rows per panel of D / U (prow >= nao: one dense panel)
    int pc = 0;                    // K auxiliary functions per chunk of the exchange contraction
    std::vector<int> panel_r0;     // panel boundaries (AO rows, even, shell aligned), size npanel + 1
    size_t arena_bytes = 0;
};

struct risp_ctx {
    std::string err;
    int device = 0;
    // ---- dimensions
    int natm = 0, nshl = 0, nao = 0, nocc = 0, nvir = 0, nmo = 0;
    int ldao = 0, ldocc = 0, ldvir = 0;          // even leading dimensions (TMA needs 16-byte strides)
    int nauxJ = 0, nauxK = 0, ncenJ = 0, ncenK = 0, ncenJ_pad = 0;
    int noccK = 0, nvirK = 0, occK0 = 0, virK0 = 0, no_p = 0, nv_p = 0;
    double alpha = 0, beta = 0, omega = 0;
    bool has_K = false;
    long long n_shell_pairs = 0, n_shell_pairs_kept = 0, n_ao_pairs_kept = 0, e_rows = 0;
    int total_chunks = 0;
    size_t hbm_budget = 0, host_budget = 0;
    int max_batch = RISP_MS, flags = 0;
    int tc_shape22 = -1, tc_shape23 = -1, tc_seg22 = 0, tc_seg23 = 0;   // tile shape / stages per segment of the Eq. 22 / 23 launches of gemm_tc.cu (-1 / 0: default)
    int precision = 0;                                          // RISP_PRECISION_*
    int shard_rank = 0, shard_count = 1, nauxK_global = 0;      // P-sharded sigma-build: this context holds 1 / shard_count of the pairs and K slices
    // ---- host copies needed after setup (getters, solver)
    std::vector<double> h_xyz, h_prim_exp, h_prim_d /* coef*radial norm, shell-normalised */, h_eps;
    std::vector<int> h_shl_atom, h_shl_l, h_shl_nprim, h_shl_poff, h_shl_ao;
    std::vector<int> h_aux_atom, h_aux_l, h_aux_fn /* first J function of each aux shell */, h_aux_fnK /* first K function or -1 */;
    std::vector<double> h_aux_exp;
    std::vector<long long> h_kept_pairs;   // (shl_i, shl_j) of every kept pair
    std::vector<int> h_even_shell_ao;      // AO offsets of shell starts that are even (candidate panel boundaries), ascending
    // ---- device data built by setup
    double *d_Cocc = nullptr;     // [nao][ldocc]
    double *d_CoccT = nullptr;    // [nocc][ldao]: C_occ^T, so that the back-transform Z = C_occ^T U reads a K-contiguous operand (one TMA box per stage)
    double *d_Cvir = nullptr;     // [nao][ldvir]
    double *d_eps = nullptr;      // [nmo]
    double *d_boys = nullptr;     // Boys table
    void *d_oneel_shl = nullptr;  // shell table of the one-electron kernel (properties.cu), uploaded on first use
    double *d_prim_exp = nullptr, *d_prim_d = nullptr;
    PairClass cls[6];
    risp_eri::PrimPair *d_prims = nullptr;
    risp_eri::AuxCentre *d_cenJ = nullptr, *d_cenK = nullptr;
    double *d_MJ = nullptr, *d_LinvJ = nullptr;     // (P|Q)_J and the inverse of its Cholesky factor, [nauxJ][nauxJ]
    double *d_MK = nullptr, *d_MKinv = nullptr;     // (P|J^|Q)_K and its inverse, [nauxK][nauxK]
    // K tensors (Eq. 20-21), symmetric in (ij) / (ab): stored as packed lower triangles, P-major.  Slices P < nK_dev live
    // in HBM, the rest in pinned host memory and are streamed per matvec on the side stream.
    long long tri_o = 0, tri_v = 0;
    int nK_dev = 0;
    double *d_TijP = nullptr, *d_TabP = nullptr;    // [nK_dev][tri_o], [nK_dev][tri_v]
    double *d_LinvK = nullptr;    // L_K^-1 of the K metric (RISP_FLAG_TDDFT only)
    double *d_Tov = nullptr;      // full TDDFT only (RISP_FLAG_TDDFT): L_K^-1 (ia|J^|Q) over the window, [nauxK][noccK][nv_p] (T_ia^P')
    double *h_TijP = nullptr, *h_TabP = nullptr;    // pinned [nauxK - nK_dev][tri]
    // ---- matvec work space (sized for m_cap vectors)
    int m_cap = 0;
    MatvecPlan plan;
    int force_mj = 0, force_prow = 0, force_pc = 0; // debug overrides (risp_debug_force_plan)
    double *w_arena = nullptr;    // J phase: Y [mj][nocc][ldao], D/U panel [mj][prow][ldao];  K phase: X', K', M, expanded T chunk
    double *w_dbar = nullptr;     // [e_rows][MS]     e0-space density, reused for U-bar
    double *w_Rpart = nullptr, *w_R = nullptr, *w_Rt = nullptr, *w_Rtmp = nullptr, *w_RtC = nullptr;
    double *w_J = nullptr;        // [m][nocc][nvir], only with RISP_FLAG_KEEP_STAGES
    double *w_stage[2] = {nullptr, nullptr};      // packed host-resident T chunks in flight
    double *w_Xin = nullptr, *w_Sout = nullptr;   // staging for risp_matvec_host
    // RISP_PRECISION_FP32_JK: bf16 x 3 planes of the MO coefficients (matvec.cu, built at the first sigma-build in that mode):
    // C_vir [nao][nvir_q], C_occ [nao][nocc_q], C_occ^T [nocc][nao_q], C_vir^T [nvir][nao_q]; rows padded to 8 elements
    unsigned short *q_C = nullptr;
    int q_C_failed = 0;
    int xin_cap = 0;
    size_t w_bytes = 0, setup_bytes = 0;
    int last_m = 0;
    cudaEvent_t ev[RISP_NEV];
    cudaEvent_t evStage[2], evStageFree[2];
    bool ev_ok = false;
    risp_timings tim;
    cudaStream_t side = nullptr;  // side stream: host-resident K chunks, Davidson subspace copies
    cudaStream_t cls_st[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // the six pair classes of a J step run concurrently
    cudaEvent_t evFork = nullptr, evJoin[6];
};

// ---- eri_kernels.cu
cudaError_t risp_eri_fill(int la, int lb, bool hasp, bool erf_op, const risp_eri::ShellPair *pairs, int npairs, const risp_eri::PrimPair *prims,
                          const risp_eri::AuxCentre *cen, int ncen, risp_eri::OpParams op, const double *boys_tab, double *out,
                          long long stride_q, long long ld, int mirror, cudaStream_t st);
// D rows [r0, ...) (leading dimension ld, vector stride mstride) -> e0 space, lanes [lane0, lane0 + mj).  mode 0: dense, pairs
// [p0, p1) of the aoA-sorted list; mode 1: += from the rows of shell A; mode 2: += from the rows of shell B, [p0, p1) of the aoB-sorted list
// (mode 0 also zeroes the lanes >= m_total, so that the unused lanes of the passes never carry stale data)
cudaError_t risp_dens_to_e0(const PairClass &pc, int p0, int p1, int mj, int lane0, int m_total, int r0, long long ld, long long mstride, int mode,
                            const double *D, double *dbar, cudaStream_t st);
// e0 space -> U rows [r0, ...), same modes (0: block and mirror image; 1: block at the rows of A; 2: transposed block at the rows of B)
cudaError_t risp_e0_to_U(const PairClass &pc, int p0, int p1, int mj, int lane0, int r0, long long ld, long long mstride, int mode,
                         const double *ubar, double *U, cudaStream_t st);
cudaError_t risp_j_pass1(const PairClass &pc, const risp_eri::PrimPair *prims, const risp_eri::AuxCentre *cen, int ncen, int ncen_pad,
                         const double *boys_tab, const double *dbar, double *Rpart, int m, cudaStream_t st);
cudaError_t risp_j_reduce_R(const double *Rpart, int nchunks, const risp_eri::AuxCentre *cen, int ncen, int ncen_pad, double *R, cudaStream_t st);
// R~ [nauxJ][MS] -> by centre [ceil32(ncen)*4][MS] (zero padded); pass 2 takes the by-centre array
cudaError_t risp_rt_by_centre(const double *Rt, const risp_eri::AuxCentre *cen, int ncen, double *RtC, cudaStream_t st);
cudaError_t risp_j_pass2(const PairClass &pc, const risp_eri::PrimPair *prims, const risp_eri::AuxCentre *cen, int ncen, const double *boys_tab,
                         const double *Rt, double *ubar, int m, cudaStream_t st);

// ---- linalg.cu: Cholesky A = L L^T (lower, in place; upper triangle zeroed) and Linv = L^-1, both [n][n] row-major on the device.
// *info_host = 0 on success, k+1 if the k-th pivot is not positive.
cudaError_t risp_cholesky_inverse(double *A, double *Linv, int n, int *info_host, cudaStream_t st);
cudaError_t risp_metric_solve32(const double *Linv, int n, const double *R, double *tmp, double *Rt, cudaStream_t st);

// ---- elementwise.cu
cudaError_t risp_gather_window(const double *X, double *Xk, int m, int nocc, int nvir, int o0, int no, int v0, int nv, int ldk, cudaStream_t st);
cudaError_t risp_diag_sigma(const double *X, const double *eps, double *sigma, int m, int nocc, int nvir, cudaStream_t st);
cudaError_t risp_sub_window(const double *Kk, double *sigma, int m, int nocc, int nvir, int o0, int no, int v0, int nv, int ldk, cudaStream_t st);
cudaError_t risp_axpy_window(const double *Kk, double scale, double *sigma, int m, int nocc, int nvir, int o0, int no, int v0, int nv, int ldk, cudaStream_t st);
cudaError_t risp_scatter_window(const double *Kk, double *Kfull, int m, int nocc, int nvir, int o0, int no, int v0, int nv, int ldk, cudaStream_t st);
// packed lower triangle [n(n+1)/2] <-> full symmetric [n][ld]; batched over np slices
cudaError_t risp_pack_sym(const double *full, long long full_stride, int ld, int n, int np, double *packed, long long tri, cudaStream_t st);
cudaError_t risp_expand_sym(const double *packed, long long tri, int n, int np, double *full, long long row_stride, long long p_stride,
                            cudaStream_t st);

// ---- setup.cu / matvec.cu / solve.cu internals
int risp_ensure_workspace(risp_ctx *ctx, int m);
size_t risp_plan_workspace(const risp_ctx *ctx, int m, size_t avail, MatvecPlan &plan, bool spilled);
// sigma = A X (TDA).  With sigma_minus != nullptr (full TDDFT, needs d_Tov): sigma = (A+B) X, sigma_minus = (A-B) X (Eq. 2).
// phase 0: the whole sigma-build.  Sharded contexts: phase 1 = up to the partial R_mQ of pass 1 (Eq. 14), phase 2 = from the metric
// solve on (the caller has summed R over the shards in between).
int risp_matvec_impl(risp_ctx *ctx, int m, const double *X, double *sigma, cudaStream_t st, double *sigma_minus = nullptr, int phase = 0);
int risp_build_pair(risp_ctx *ctx, int shA, int shB, risp_eri::ShellPair &sp, std::vector<risp_eri::PrimPair> &pp, double prim_tol);
void risp_free_workspace(risp_ctx *ctx);
int risp_rows_gram(risp_ctx *ctx, const double *A, int na, const double *B, int nb, long long dim, long long slice, double *dPart, double *dSmall,
                   std::vector<double> &out, cudaStream_t st);
int risp_rows_lincomb(risp_ctx *ctx, const double *coef_host, int nc, int na, const double *A, double *C, long long dim, double alpha, double beta,
                      double *dCoef, cudaStream_t st);
