/*
 * risp.h -- C ABI of the B200-native TDA-risp sigma-build library (librisp.so).
 *
 * Method: arxiv/paper_2603_29257 ("GPU Accelerated Minimal Auxiliary Basis Approach TDDFT
 * for Large Organic Molecules").  Citations are PAPER.md:<line> of /root/reference/PAPER.md.
 *
 * The library computes, entirely in CUDA kernels for sm_100a and in FP64,
 *
 *     sigma_m = A X_m ,   A[ia,jb] = d_ij d_ab (e_a - e_i) + 2 (ia|jb) - (ij|J^|ab)        (Eq. 9-10)
 *
 * with (ia|jb) by RI in the Coulomb metric over an s+p auxiliary basis, evaluated AO-direct with the
 * three-centre integrals regenerated on the fly (Eq. 11-17), and (ij|J^|ab) by RI over the
 * K auxiliary subset with stored T_ij^P, T_ab^P tensors restricted to the energy window
 * (Eq. 18-26); J^ = (alpha + beta erf(omega r12))/r12 (Eq. 25).  risp_tda_solve runs a
 * Davidson loop whose subspace lives in pinned host memory.
 *
 * Conventions
 *   - every call returns RISP_OK (0) or a negative RISP_E* code; nothing throws across the ABI;
 *     risp_last_error() gives a text for the last failure on that context.
 *   - units: bohr and Hartree; only `cutoff_ev` is in eV (1 Ha = 27.211386245988 eV).
 *   - AO order inside a shell: s; p = (x, y, z); d = (xy, yz, z2, xz, x2-y2); unit-normalised real solid
 *     harmonics; a contracted shell is sum_k c_k N(a_k,l) r^l exp(-a_k r^2) Y_lm, rescaled by the library to
 *     unit norm (so `prim_coef` multiplies *unit-normalised primitives* and its overall scale is irrelevant).
 *   - auxiliary functions (Eq. 4): unit-normalised primitive Cartesian Gaussians, l = 0 (one
 *     function) or l = 1 (x, y, z).  Function index = running index over `aux_*` shells in the given order.
 *     The caller supplies the exponents theta/R_A^2 and omits hydrogens.
 *   - pointers in risp_system are HOST pointers, read during risp_setup only and never retained.
 *   - one context per host thread at a time; no global state.  Test and tuning exports are declared in risp_debug.h.
 */
#ifndef RISP_H
#define RISP_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RISP_OK 0
#define RISP_EINVAL (-1)   /* bad argument (NULL, negative size, l out of range, overlapping X/sigma, ...) */
#define RISP_ENOMEM (-2)   /* device or pinned-host allocation failed */
#define RISP_ECUDA (-3)    /* a CUDA call or kernel failed; see risp_last_error */
#define RISP_ENOTPD (-4)   /* an auxiliary metric (P|Q) is not positive definite */
#define RISP_ENOTCONV (-5) /* risp_tda_solve hit max_iter; outputs are still filled with the last Ritz pairs */

typedef struct risp_ctx risp_ctx; /* opaque; owns every device and pinned allocation it makes */

/* The problem, as the paper states it: a converged closed-shell SCF (geometry, AO basis, MO coefficients,
 * orbital energies) plus the method parameters (aux exponents, Eq. 4; the K operator, Eq. 25;
 * the exchange-space cutoff). */
typedef struct {
    int32_t natm;
    const double *xyz_bohr;     /* [natm][3] */
    const int32_t *Z;           /* [natm] nuclear charges (reporting only) */
    int32_t nshl;               /* AO shells */
    const int32_t *shl_atom;    /* [nshl] */
    const int32_t *shl_l;       /* [nshl] 0, 1 or 2 */
    const int32_t *shl_nprim;   /* [nshl] >= 1 */
    const int32_t *shl_poff;    /* [nshl] offset of the shell's first primitive in prim_exp / prim_coef */
    const double *prim_exp;
    const double *prim_coef;
    int32_t naux;               /* auxiliary shells (all of them enter J) */
    const int32_t *aux_atom;    /* [naux] */
    const int32_t *aux_l;       /* [naux] 0 or 1 */
    const double *aux_exp;      /* [naux] */
    const uint8_t *aux_in_K;    /* [naux] 1: shell also belongs to the K auxiliary set (paper: the s shells) */
    int32_t nao, nocc, nvir;    /* nao = sum (2l+1); nocc + nvir <= nao */
    const double *C;            /* [nao][nocc+nvir] row-major, occupied columns first */
    const double *eps;          /* [nocc+nvir] Hartree, ascending within occ and within vir */
    double alpha, beta, omega;  /* K operator (alpha + beta erf(omega r))/r; global hybrid: alpha = a_x, beta = 0 */
    double cutoff_ev;           /* keep occ with eps > -cutoff and vir with eps < +cutoff;
                                   <= 0 or +inf: no truncation */
} risp_system;

typedef struct {
    double screen_tol;          /* shell-pair screening threshold tau (0 -> default 1e-13; < 0 -> keep every pair) */
    size_t hbm_budget_bytes;    /* device memory the library may use (0 -> 85 % of what is free at setup); K-tensor slices that do
                                   not fit are kept in pinned host memory and streamed per matvec */
    size_t host_budget_bytes;   /* pinned-host budget of the part of the Davidson subspace that does not fit in HBM; 0 -> half of the
                                   physical host memory */
    int32_t device;             /* CUDA device ordinal */
    int32_t flags;              /* RISP_FLAG_* */
    int32_t max_batch;          /* largest m the caller will pass to risp_matvec (0 -> 32); HBM is reserved for its X, sigma
                                   and work space before the K tensors are placed */
    int32_t reserved;
    int32_t shard_rank, shard_count; /* P-sharded sigma-build over several GPUs: shard_count > 1 makes this context
                                   hold every shard_count-th kept shell pair and the K-tensor slices of every shard_count-th
                                   auxiliary centre, all in HBM; see risp_matvec_shard_begin / _end.  0 or 1: not sharded */
} risp_options;

#define RISP_FLAG_KEEP_STAGES 1   /* keep J_mia of the last risp_matvec for risp_get_stage (costs one more [m][nocc][nvir] buffer) */
#define RISP_FLAG_SPILL_HALF 2    /* testing: place the upper half of the K-tensor slices in pinned host memory regardless of the budget */
#define RISP_FLAG_TDDFT 8         /* also build T_ia^P' over the exchange window, kept whole in HBM: enables risp_matvec_tddft
                                     and risp_tddft_solve (full TDDFT-risp, Eq. 1-2) */
#define RISP_FLAG_SMALL_KBUILD 4  /* testing: build the K tensors in runs of at most 5 auxiliary functions (the large-system code path) */

typedef struct {
    double tol;                 /* residual 2-norm threshold (0 -> 1e-5) */
    int32_t max_iter;           /* 0 -> 100 */
    int32_t n_guess;            /* initial unit vectors on the smallest e_a - e_i (0 -> 2*nroots) */
    int32_t max_sub;            /* restart when the subspace would exceed this (0 -> 20*nroots) */
    int32_t flags;              /* RISP_SOLVE_* */
    int32_t max_block;          /* trial vectors per sigma-build inside the solver (0 -> min(32, max_batch of risp_setup, n_guess)); the
                                   solver holds two blocks of this many vectors on the device, everything else of the subspace is
                                   cached in what HBM is left or streamed from pinned host memory */
    int32_t max_seconds;        /* wall-clock guard: no new iteration starts after this many seconds (0 -> none); the call then returns
                                   RISP_ENOTCONV with the current Ritz values, residual norms and vectors */
    size_t device_budget_bytes; /* device memory the solver may allocate (0 -> what is free after the matvec work space); if two
                                   blocks and the streaming buffers do not fit: RISP_ENOMEM, nothing stays allocated */
} risp_solve_options;

#define RISP_SOLVE_NO_CACHE 1        /* every pass over V, W streams from pinned host memory (no device cache) */
#define RISP_SOLVE_TINY_CACHE 2      /* testing: cache only nroots + 2 vectors, the rest is streamed */
#define RISP_SOLVE_PERTURBED_GUESS 4 /* guess = unit vectors + seeded dense noise (relative norm 0.3), orthonormalised: a second,
                                        different start to check that no lower root was missed */
#define RISP_SOLVE_HOST_FP32 8       /* host-resident part of V, W stored in single precision (the paper's storage precision,
                                        PAPER.md:201); every product still accumulates in FP64.  Trial vectors are rounded to
                                        FP32-representable values before their sigma-build, so V is stored exactly */

#define RISP_SOLVE_X_OUT_HOST 16      /* X_out is a HOST pointer: the Ritz vectors are written there chunk by chunk (3000 atoms: 15 vectors
                                        are 16 GB, more than is left on the device beside the K tensors) */

#define RISP_SOLVE_LOG_STDERR 32     /* one line per iteration on stderr (iteration, subspace size, unconverged roots, largest residual, seconds):
                                        a long solve leaves its history behind even if the job is cut short */

#define RISP_MAX_ROOTS 64
typedef struct {
    int32_t iterations, restarts, n_sigma, converged;
    double resid[RISP_MAX_ROOTS];        /* final residual norms */
    double sec_total, sec_matvec, sec_subspace; /* wall seconds: whole call, sigma-builds, subspace algebra (incl. streaming) */
    double bytes_h2d, bytes_d2h;         /* subspace traffic over the host link */
    int32_t subspace_max;                /* largest subspace held */
    int32_t cached_vectors;              /* leading vectors of V and of W kept in HBM as well */
    double sec_alloc;                    /* wall seconds spent allocating the pinned subspace and the device buffers */
    int32_t block;                       /* trial vectors per sigma-build the solver used */
    int32_t capacity;                    /* subspace vectors the device cache and the pinned-host budget hold together */
    double bytes_host_subspace;          /* pinned host bytes reserved for V and W */
} risp_solve_info;

typedef struct {
    int32_t nao, nocc, nvir, nauxJ, nauxK; /* function counts */
    int32_t noccK, nvirK, occK_first, virK_first; /* window: occupied [occK_first, occK_first+noccK), virtual likewise
                                                     (indices within occ / within vir) */
    int64_t n_shell_pairs, n_shell_pairs_kept, n_ao_pairs_kept;
    int64_t bytes_Tij, bytes_Tab, bytes_device_total; /* K tensors as stored (packed lower triangles), all device allocations */
    int32_t aux_chunk;                   /* K auxiliary functions per chunk in the matvec */
    int32_t nauxK_device;                /* K-tensor slices resident in HBM; the other nauxK - nauxK_device live in pinned host memory */
    int64_t bytes_T_host;                /* pinned host bytes of the spilled slices */
    int32_t j_sub_batch, j_panels;       /* J transforms: trial vectors per sub-batch, AO row panels per sub-batch (1 = dense) */
    int64_t pairs_per_class[6];          /* kept shell pairs by angular-momentum class (l_a >= l_b): ss, ps, pp, ds, dp, dd */
    int64_t n_aux_centres;               /* auxiliary centres of the J set (an s and a p shell of one atom share a centre, Eq. 4) */
} risp_dims;

/* per-phase device seconds of the last risp_matvec (CUDA events; valid after the stream was synchronised) */
typedef struct {
    double total, j_transform_in, j_pass1, j_solve, j_pass2, j_transform_out, k_gather;
    double k_gemm1, k_gemm2;     /* the FIRST aux chunk's M^P = X' T_ab^P launch (Eq. 22) and K' += T_ij^P M^P launch (Eq. 23) */
    double k_total, assemble;    /* all chunks of the K contraction (expansion of the packed slices included); sigma -= K' */
    int32_t kernel_launches;     /* kernels launched by the last risp_matvec */
    int32_t first_chunk_naux;    /* K aux functions in the first chunk (work of the two timed launches) */
} risp_timings;

/* Build everything that does not depend on X: screened shell-pair list, metrics (P|Q)_J, (P|J^|Q)_K and their
 * Cholesky factors, the window, and the tensors T_ij^P (Eq. 20), T_ab^P (Eq. 21).  Synchronous. */
int risp_setup(const risp_system *sys, const risp_options *opt, risp_ctx **out);

/* sigma = A X for a batch of m trial vectors.  X_dev, sigma_dev: DEVICE pointers, [m][nocc][nvir] row-major,
 * sigma overwritten, X not modified, the two must not overlap.  Asynchronous on `cuda_stream` (a cudaStream_t;
 * NULL = default stream).  Any m >= 1 is accepted: the call works through sub-batches of at most 32 vectors (one lane per
 * trial vector in the integral passes); the work space grows to min(m, 32) vectors if `max_batch` of risp_setup was smaller
 * (RISP_ENOMEM if that no longer fits beside the K tensors).  risp_get_timings / risp_get_stage refer to the last sub-batch. */
int risp_matvec(risp_ctx *ctx, int32_t m, const double *X_dev, double *sigma_dev, void *cuda_stream);

/* Precision of the exchange contractions Eq. 22-23 of every following sigma-build of this context
 * (risp_matvec, risp_matvec_host, risp_matvec_shard_*, risp_tda_solve):
 *   RISP_PRECISION_FP64    (default) FP64 DMMA GEMMs; sigma within 1e-10 of the FP64 oracle;
 *   RISP_PRECISION_FP32_K  the paper's own precision for everything after the integrals: X', T_ij, T_ab and M^P are
 *                          carried as three bf16 terms each (24 significand bits), the products run on the tcgen05 tensor cores with
 *                          FP32 accumulation in tensor memory, the aux chunks are summed in FP64.  The K term then carries a
 *                          relative error of order 1e-7 (DESIGN.md "FP32 mode" derives the bound; oracle/risp_fp32.py is the
 *                          plain binary32 contraction it is compared with).  Diagonal, J term and the Davidson algebra stay FP64;
 *                          the K tensors stay stored in FP64.  risp_matvec_tddft returns RISP_EINVAL in this mode.
 *   RISP_PRECISION_FP32_JK RISP_PRECISION_FP32_K, and the four dense AO<->MO transforms of the Coulomb term (Eq. 12, 17;
 *                          PAPER.md:109, 123) through the same tensor-core GEMM (X, C_occ, C_vir, U and the half-transformed
 *                          intermediates as three bf16 terms); integrals, both ERI passes, the metric solve, the diagonal and the
 *                          Davidson algebra stay FP64.  The rounding of the density enters R~ = (P|Q)^-1 R, so J carries a relative
 *                          error of up to (2 cond(P|Q) + 2) x 1e-6 (measured 1e-5 at cond 9e4).  Used for
 *                          unsharded TDA sigma-builds whose J work space holds all AO rows of a sub-batch at once; with row
 *                          panels (3000 atoms on one GPU) and in the sharded sigma-build the transforms stay FP64 (slower,
 *                          more accurate).
 * Returns RISP_OK or RISP_EINVAL (unknown mode, or a single-precision mode on a device without tcgen05). */
#define RISP_PRECISION_FP64 0
#define RISP_PRECISION_FP32_K 1
#define RISP_PRECISION_FP32_JK 2
int risp_set_precision(risp_ctx *ctx, int32_t mode);

/* Full TDDFT-risp (Eq. 1-2; XC kernel dropped): for m trial vectors
 *     sigma_plus  = (A+B) X = Delta X + 4 J X - K1 X - K2 X,        sigma_minus = (A-B) X = Delta X - K1 X + K2 X,
 * J = (ia|jb)_RI-J, K1 = (ij|J^|ab)_RI-K, K2 = (ib|J^|ja)_RI-K, the two exchange terms restricted to the exchange window
 * (reading G25: Eq. 2a's "2(ia|jb)" is read as 4(ia|jb), consistent with Eq. 10 and Eq. 2b).  Needs RISP_FLAG_TDDFT at
 * setup.  All three buffers DEVICE [m][nocc][nvir], pairwise disjoint; asynchronous on cuda_stream. */
int risp_matvec_tddft(risp_ctx *ctx, int32_t m, const double *X_dev, double *sigma_plus_dev, double *sigma_minus_dev, void *cuda_stream);

/* P-sharded sigma-build, one context per GPU (set up with shard_rank / shard_count; X replicated on every rank):
 *     risp_matvec_shard_begin   D (Eq. 12) and pass 1 (Eq. 14) over this rank's shell pairs -> R_partial_dev [nauxJ][32] (DEVICE,
 *                               trial vector fastest, zero beyond m);
 *     -- the caller sums R_partial over the ranks (one all-reduce of nauxJ * 32 doubles, < 2 MB) --
 *     risp_matvec_shard_end     R~ (Eq. 15), pass 2 (Eq. 16) and the back-transform (Eq. 17) on this rank's pairs, Eq. 22-23 over this
 *                               rank's K slices, the diagonal on rank 0 -> sigma_partial_dev [m][nocc][nvir];
 *     -- the caller sums sigma_partial over the ranks (all-reduce or reduce-scatter of m * nocc * nvir doubles) --
 * m <= 32 per call.  Both calls are asynchronous on cuda_stream; the sum of the partial results equals risp_matvec of an
 * unsharded context up to the order of the floating-point sums. */
int risp_matvec_shard_begin(risp_ctx *ctx, int32_t m, const double *X_dev, double *R_partial_dev, void *cuda_stream);
int risp_matvec_shard_end(risp_ctx *ctx, int32_t m, const double *X_dev, const double *R_dev, double *sigma_partial_dev, void *cuda_stream);

/* Same with HOST buffers: copies X in, runs risp_matvec, copies sigma out, synchronises. */
int risp_matvec_host(risp_ctx *ctx, int32_t m, const double *X_host, double *sigma_host);

/* Lowest `nroots` eigenpairs of A by a Davidson iteration whose subspace (V, W = A V) lives in pinned host
 * memory and is streamed through the device on a side stream.  omega_hartree: HOST [nroots]
 * ascending.  X_out: DEVICE [nroots][nocc][nvir] (HOST with RISP_SOLVE_X_OUT_HOST) or NULL.  info may be NULL. */
int risp_tda_solve(risp_ctx *ctx, int32_t nroots, const risp_solve_options *opt, double *omega_hartree, double *X_out,
                   risp_solve_info *info);

/* Transition properties of n TDA states (Eq. 5-8; TDA: Y = 0):
 *     mu_0n = scale sum_ia r_ia X_nia (Eq. 7),   m_0n = scale sum_ia (r x nabla)_ia X_nia (Eq. 8),
 *     f_0n = 2/3 Omega_n mu_0n . mu_0n (Eq. 5),  R_0n = 1/2 mu_0n . m_0n (Eq. 6),    atomic units, dipole-length form.
 * X_dev: DEVICE [n][nocc][nvir] (e.g. X_out of risp_tda_solve, <X|X> = 1); omega_hartree: HOST [n] (needed for f_out only);
 * origin_bohr: HOST [3] gauge origin of r and r x nabla, NULL = (0,0,0); scale: factor on both moments, <= 0 selects sqrt(2), the
 * closed-shell singlet factor for unit-normalised X (the paper prints none: DESIGN.md reading G24).  Outputs are HOST arrays,
 * mu_out[n][3], m_out[n][3], f_out[n], R_out[n]; any of them may be NULL.  Synchronous; allocates and frees its own scratch
 * (one AO matrix, one half-transformed matrix, six [nocc][nvir] blocks). */
int risp_transition_properties(risp_ctx *ctx, int32_t n, const double *X_dev, const double *omega_hartree, const double *origin_bohr,
                               double scale, double *mu_out, double *m_out, double *f_out, double *R_out);

/* Lowest `nroots` (<= 32) excitation energies of full TDDFT-risp, the symplectic problem Eq. 1, by a Davidson
 * iteration that projects A+B and A-B into one orthonormal trial space (reading G26).  Needs
 * RISP_FLAG_TDDFT at setup; the subspace (b, (A+B) b, (A-B) b) is device resident and the iteration restarts from {X+Y, X-Y} when
 * it is full.  omega_hartree: HOST [nroots] ascending; X_out, Y_out: DEVICE [nroots][nocc][nvir] or NULL, normalised to
 * <X|X> - <Y|Y> = 1.  Options as risp_tda_solve (tol on max(|r1|, |r2|), max_iter, n_guess, max_sub, device_budget_bytes);
 * RISP_ENOTPD if the projected A-B is not positive definite. */
int risp_tddft_solve(risp_ctx *ctx, int32_t nroots, const risp_solve_options *opt, double *omega_hartree, double *X_out, double *Y_out,
                     risp_solve_info *info);

/* The single-precision-mode GEMM on its own, for callers that must not allocate (CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc):
 *     C[c][r] (+)= sum_k A[r][k] B[c][k]        A_dev [M][K], B_dev [N][K], C_dev [N][M], contiguous DEVICE FP64,
 * the arithmetic of RISP_PRECISION_FP32_K (operands as three bf16 terms, FP32 accumulation on the tcgen05 tensor cores, result
 * added to C in FP64 when accumulate != 0).  It calls no cudaMalloc / cudaFree and no allocating library routine: the bf16
 * operand planes, 6 (M + N) ceil8(K) bytes, live in ONE static device array of RISP_STATIC_SCRATCH_BYTES that every GPU which
 * loads the library holds until exit.  Larger problems are rejected with RISP_EINVAL (text from risp_static_last_error()).
 * Works on the CURRENT device, which cuda_stream must belong to; asynchronous on that stream.  All calls share the array: calls
 * that overlap on the GPU (different streams, or host threads without ordering) race on it; calls on one stream do not.  Nothing
 * in it has to be cleared between calls (every element a call reads it has written itself).  Needs no risp_ctx.
 * Returns RISP_OK, RISP_EINVAL or RISP_ECUDA. */
#define RISP_STATIC_SCRATCH_BYTES (16u << 20)
int risp_tcgemm_static(int32_t M, int32_t N, int32_t K, const double *A_dev, const double *B_dev, double *C_dev, int32_t accumulate,
                       void *cuda_stream);
const char *risp_static_last_error(void); /* text of the calling thread's last risp_tcgemm_static failure ("" if none) */

void risp_destroy(risp_ctx *ctx);
const char *risp_last_error(const risp_ctx *ctx); /* static text if ctx == NULL */

/* ---- debug / parity getters (not timed) ---- */
int risp_get_dims(const risp_ctx *ctx, risp_dims *out);
int risp_get_timings(const risp_ctx *ctx, risp_timings *out);

/* (shell_i shell_j | aux shell k) block, out_host[(2li+1)][(2lj+1)][nk] (nk = 1 or 3), computed by the same device
 * integral code as the hot path.  op = 0: Coulomb 1/r (J); op = 1: the K operator of risp_system. */
int risp_eri3c_shell(risp_ctx *ctx, int32_t shl_i, int32_t shl_j, int32_t aux_k, int32_t op, double *out_host);

/* Intermediate of the LAST risp_matvec / setup, copied to out_host (HOST).  `which`: */
#define RISP_STAGE_R 1       /* R_mQ (Eq. 14):  out[nauxJ][m]                                   sel ignored */
#define RISP_STAGE_RTILDE 2  /* R~_mP (Eq. 15): out[nauxJ][m]                                                */
#define RISP_STAGE_J 3       /* J_mia (Eq. 17): out[m][nocc][nvir]            needs RISP_FLAG_KEEP_STAGES            */
#define RISP_STAGE_K 4       /* K_mia (Eq. 23) scattered to the full space: out[m][nocc][nvir]               */
#define RISP_STAGE_TIJ 5     /* T_ij^P for the K-aux functions P in sel: out[nsel][noccK][noccK]             */
#define RISP_STAGE_TAB 6     /* T_ab^P:                                  out[nsel][nvirK][nvirK]             */
#define RISP_STAGE_PAIRS 7   /* kept shell pairs as (shl_i, shl_j) int64 pairs: out = int64[n_kept][2]       */
#define RISP_STAGE_METRIC_J 8 /* (P|Q)_J: out[nauxJ][nauxJ] */
#define RISP_STAGE_METRIC_K 9 /* (P|J^|Q)_K: out[nauxK][nauxK] */
#define RISP_STAGE_U 10      /* U^m (Eq. 16), dense AO matrix of vector sel[0]: out[nao][nao] */
int risp_get_stage(risp_ctx *ctx, int32_t which, const int64_t *sel, int64_t nsel, void *out_host);

#ifdef __cplusplus
}
#endif
#endif /* RISP_H */
