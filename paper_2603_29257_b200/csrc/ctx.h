// ctx.h -- the library context and the internal interfaces between the .cu files.
#pragma once
#include "common.cuh"
#include "eri.cuh"
#include <type_traits>

#define RISP_MS 32   // padded trial-vector stride of R, R~, D-bar, U-bar (one lane per trial vector)

struct PairClass {                 // kept shell pairs of one (la >= lb) class, sorted together
    int la, lb, npairs;
    risp_eri::ShellPair *d_pairs;  // device
    long long e_off;               // first e0 row of this class in D-bar / U-bar
    int chunk, nchunks, chunk_base; // pass-1 pair chunking (chunk_base: global index of the class's first chunk)
};

struct DevBuf {                    // grow-only device scratch buffer
    void *p = nullptr; size_t cap = 0;
};

struct risp_ctx {
    std::string err;
    int device = 0;
    // ---- dimensions
    int natm = 0, nshl = 0, nao = 0, nocc = 0, nvir = 0, nmo = 0;
    int nauxJ = 0, nauxK = 0, ncenJ = 0, ncenK = 0, ncenJ_pad = 0;
    int noccK = 0, nvirK = 0, occK0 = 0, virK0 = 0;
    double alpha = 0, beta = 0, omega = 0;
    bool has_K = false;
    long long n_shell_pairs = 0, n_shell_pairs_kept = 0, n_ao_pairs_kept = 0, e_rows = 0;
    int total_chunks = 0;
    size_t hbm_budget = 0, host_budget = 0;
    // ---- host copies needed after setup (getters, solver)
    std::vector<double> h_xyz, h_prim_exp, h_prim_d /* coef*radial norm, shell-normalised */, h_eps;
    std::vector<int> h_shl_atom, h_shl_l, h_shl_nprim, h_shl_poff, h_shl_ao;
    std::vector<int> h_aux_atom, h_aux_l, h_aux_fn /* first J function of each aux shell */, h_aux_fnK /* first K function or -1 */;
    std::vector<double> h_aux_exp;
    std::vector<long long> h_kept_pairs;   // (shl_i, shl_j) of every kept pair
    // ---- device data built by setup
    double *d_C = nullptr;        // [nao][nmo]
    double *d_eps = nullptr;      // [nmo]
    double *d_boys = nullptr;     // Boys table
    PairClass cls[6];
    risp_eri::PrimPair *d_prims = nullptr;
    risp_eri::AuxCentre *d_cenJ = nullptr, *d_cenK = nullptr;
    double *d_MJ = nullptr, *d_LinvJ = nullptr;     // (P|Q)_J and the inverse of its Cholesky factor, [nauxJ][nauxJ]
    double *d_MK = nullptr, *d_MKinv = nullptr;     // (P|J^|Q)_K and its inverse, [nauxK][nauxK]
    double *d_Tij = nullptr;      // [noccK][nauxK][noccK]   T_ij^P of Eq. 20 stored i-major: Tij[i][P][j]
    double *d_Tab = nullptr;      // [nauxK][nvirK][nvirK]   T_ab^P of Eq. 21, P-major
    int aux_chunk = 0;            // K aux functions per matvec chunk
    // ---- matvec work space (sized for m_cap vectors)
    int m_cap = 0;
    double *w_Y = nullptr;        // [m][nocc][nao]   (X C_vir^T, later C_occ^T U)
    double *w_D = nullptr;        // [m][nao][nao]    AO density, reused for U
    double *w_dbar = nullptr;     // [e_rows][MS]     e0-space density, reused for U-bar
    double *w_Rpart = nullptr, *w_R = nullptr, *w_Rt = nullptr, *w_Rtmp = nullptr;
    double *w_J = nullptr;        // [m][nocc][nvir]
    double *w_Xk = nullptr, *w_Kk = nullptr;  // [m][noccK][nvirK]
    double *w_M = nullptr;        // [m][aux_chunk][noccK][nvirK]
    double *w_Xin = nullptr, *w_Sout = nullptr;   // staging for risp_matvec_host
    size_t w_bytes = 0, setup_bytes = 0;
    int last_m = 0;
    cudaEvent_t ev[12];
    bool ev_ok = false;
    risp_timings tim;
    cudaStream_t side = nullptr;  // side stream of the Davidson subspace copies
};

// ---- eri_kernels.cu
cudaError_t risp_eri_fill(int la, int lb, bool hasp, bool erf_op, const risp_eri::ShellPair *pairs, int npairs, const risp_eri::PrimPair *prims,
                          const risp_eri::AuxCentre *cen, int ncen, risp_eri::OpParams op, const double *boys_tab, double *out,
                          long long stride_q, long long ld, int mirror, cudaStream_t st);
cudaError_t risp_dens_to_e0(const PairClass &pc, int m, int nao, const double *D, double *dbar, cudaStream_t st);
cudaError_t risp_e0_to_U(const PairClass &pc, int m, int nao, const double *ubar, double *U, cudaStream_t st);
cudaError_t risp_j_pass1(const PairClass &pc, const risp_eri::PrimPair *prims, const risp_eri::AuxCentre *cen, int ncen, int ncen_pad,
                         const double *boys_tab, const double *dbar, double *Rpart, cudaStream_t st);
cudaError_t risp_j_reduce_R(const double *Rpart, int nchunks, const risp_eri::AuxCentre *cen, int ncen, int ncen_pad, double *R, cudaStream_t st);
cudaError_t risp_j_pass2(const PairClass &pc, const risp_eri::PrimPair *prims, const risp_eri::AuxCentre *cen, int ncen, const double *boys_tab,
                         const double *Rt, double *ubar, cudaStream_t st);

// ---- linalg.cu: Cholesky A = L L^T (lower, in place; upper triangle zeroed) and Linv = L^-1, both [n][n] row-major on the device.
// *info_host = 0 on success, k+1 if the k-th pivot is not positive.
cudaError_t risp_cholesky_inverse(double *A, double *Linv, int n, int *info_host, cudaStream_t st);

// ---- elementwise.cu
cudaError_t risp_gather_window(const double *X, double *Xk, int m, int nocc, int nvir, int o0, int no, int v0, int nv, cudaStream_t st);
cudaError_t risp_assemble_sigma(const double *X, const double *J, const double *Kk, const double *eps, double *sigma, int m, int nocc, int nvir,
                                int o0, int no, int v0, int nv, int has_K, cudaStream_t st);
cudaError_t risp_scatter_window(const double *Kk, double *Kfull, int m, int nocc, int nvir, int o0, int no, int v0, int nv, cudaStream_t st);

// ---- setup.cu / matvec.cu / solve.cu internals
int risp_ensure_workspace(risp_ctx *ctx, int m);
int risp_matvec_impl(risp_ctx *ctx, int m, const double *X, double *sigma, cudaStream_t st);
int risp_build_pair(risp_ctx *ctx, int shA, int shB, risp_eri::ShellPair &sp, std::vector<risp_eri::PrimPair> &pp, double prim_tol);
