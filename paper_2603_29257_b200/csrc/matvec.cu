// matvec.cu -- risp_matvec: sigma = A X for a batch of m trial vectors (Eq. 10).
//
//   sigma = (eps_a - eps_i) X                                                                         (diagonal)
//   J (Eq. 11-17), per sub-batch of mj vectors and per panel of AO rows:
//       Y = X C_vir^T ; D = C_occ Y (Eq. 12) ; D -> e0 space on the kept pairs (a pair takes D_AB from the panel that holds
//       the rows of shell A and D_BA^T from the one that holds the rows of B) ;
//     then once for all m vectors: pass 1 (Eq. 14) ; R~ = L^-T L^-1 R (Eq. 15) ; pass 2 (Eq. 16) ;
//     then per sub-batch / panel: e0 space -> U ; Z = C_occ^T U ; sigma += 2 Z C_vir (Eq. 17)
//   K (Eq. 18-23):  X' = X[window] ; per aux chunk (from HBM, or from pinned host memory through the
//       side stream): expand the packed slices ; M^P = X' T_ab^P (Eq. 22) ; K' += T_ij^P M^P (Eq. 23) ; sigma[window] -= K'
//
// One arena serves the J phase (Y, D/U panel) and then the K phase (X', K', M, expanded T chunk); its size, the sub-batch
// mj, the panel height and the aux chunk follow from what the HBM budget leaves after the K tensors (risp_plan_workspace).
#include "ctx.h"
#include <algorithm>

void risp_free_workspace(risp_ctx *ctx)
{
    double **bufs[] = {&ctx->w_arena, &ctx->w_dbar, &ctx->w_Rpart, &ctx->w_R, &ctx->w_Rt, &ctx->w_Rtmp, &ctx->w_RtC, &ctx->w_J,
                       &ctx->w_stage[0], &ctx->w_stage[1]};
    for (auto b : bufs) { if (*b) cudaFree(*b); *b = nullptr; }
    ctx->m_cap = 0; ctx->w_bytes = 0;
}

static size_t fixed_ws_bytes(const risp_ctx *ctx)
{
    return ((size_t)ctx->e_rows * RISP_MS + (size_t)ctx->total_chunks * ctx->ncenJ_pad * 4 * RISP_MS + 3 * (size_t)ctx->nauxJ * RISP_MS) * sizeof(double);
}

// Choose (mj, panels, pc) for m vectors within `avail` bytes; returns the bytes needed (arena + staging), 0 if even the
// smallest plan does not fit.
size_t risp_plan_workspace(const risp_ctx *ctx, int m, size_t avail, MatvecPlan &pl, bool spilled)
{
    const size_t nao = ctx->nao, nocc = ctx->nocc, ldao = ctx->ldao, no = ctx->noccK, nv = ctx->nvirK, no_p = ctx->no_p, nv_p = ctx->nv_p;
    const int nK = ctx->nauxK;
    const size_t GiB = (size_t)1 << 30;
    const size_t stage_per_fn = spilled ? 2 * (size_t)(ctx->tri_o + ctx->tri_v) * 8 : 0;
    const size_t soft = (spilled ? 12 : 32) * GiB;      // arena target: every GiB of it is a GiB of K tensor streamed from the host when HBM is short
    auto kneed = [&](size_t pc) { return (2 * (size_t)m * no * nv_p + (size_t)m * pc * no_p * nv_p + pc * nv * nv_p + no * pc * no_p) * 8 + pc * stage_per_fn; };
    auto jneed = [&](size_t mj, size_t prow) { return (mj * nocc * ldao + mj * prow * ldao) * 8; };
    // ---- K chunk
    size_t karena = 0;
    pl.pc = 1;
    if (ctx->has_K) {
        const size_t klimit = std::min(avail, std::max(kneed(std::min(2, nK)), std::min(avail / 2, soft)));
        if (kneed(1) > avail) return 0;
        int pc = 1;
        while (pc < nK && kneed(pc + 1) <= klimit) ++pc;
        if (ctx->force_pc > 0) pc = std::min(ctx->force_pc, nK);
        pl.pc = pc;
        karena = kneed(pc) - pc * stage_per_fn;
    }
    // ---- J sub-batch and panels
    const size_t jlimit = std::min(avail, std::max(karena, std::min(avail / 2, soft)));
    int mj = m;
    size_t prow = nao;
    if (jneed(m, nao) > jlimit) {
        bool ok = false;
        for (int div = 1; div <= m && !ok; ++div) {
            mj = (m + div - 1) / div;
            const size_t yb = (size_t)mj * nocc * ldao * 8;
            if (yb > jlimit / 2 && mj > 1) continue;
            if (yb >= jlimit) break;
            prow = (jlimit - yb) / ((size_t)mj * ldao * 8);
            if (prow >= std::min<size_t>(nao, 256) || mj == 1) ok = prow >= 32;
        }
        if (!ok) return 0;
        prow = std::min(prow, nao);
    }
    if (ctx->force_mj > 0) mj = std::min(ctx->force_mj, m);
    if (ctx->force_prow > 0) prow = std::min<size_t>(ctx->force_prow, nao);
    // RISP_PRECISION_FP32_JK: bf16 x 3 planes of X, Y^T / Z and U behind the FP64 D / U block (risp_matvec_impl), all AO rows at once;
    // the largest sub-batch whose planes fit is taken, and without room for a single vector the J transforms stay FP64
    auto j32need = [&](size_t mj_) {
        const size_t nvir_q = ((size_t)ctx->nvir + 7) & ~(size_t)7, nocc_q = (nocc + 7) & ~(size_t)7, nao_q = (nao + 7) & ~(size_t)7;
        return jneed(mj_, nao) + 6 * mj_ * (nocc * nvir_q + std::max(nao * nocc_q, nocc * nao_q) + nao * nao_q) + 64;
    };
    bool jk = false;
    if (ctx->precision == RISP_PRECISION_FP32_JK && ctx->force_prow <= 0) {
        const int mtop = ctx->force_mj > 0 ? std::min(ctx->force_mj, m) : m;
        for (int div = 1; div <= mtop && !jk; ++div) {
            const int mj2 = (mtop + div - 1) / div;
            if (j32need(mj2) <= std::max(jlimit, karena)) { mj = mj2; prow = nao; jk = true; }
        }
    }
    // panel boundaries: even, shell-aligned AO offsets (TMA coordinates of the MN-contiguous operand must be 16-byte aligned)
    pl.panel_r0.clear();
    pl.panel_r0.push_back(0);
    size_t prow_max = 0;
    if (prow >= nao) { pl.panel_r0.push_back((int)nao); prow_max = nao; }
    else {
        const std::vector<int> &ev = ctx->h_even_shell_ao;
        int cur = 0;
        while (cur < (int)nao) {
            // largest candidate <= cur + prow, but at least the next candidate after cur
            auto it = std::upper_bound(ev.begin(), ev.end(), cur + (int)prow);
            int nxt = (it == ev.begin()) ? (int)nao : *(it - 1);
            if (nxt <= cur) nxt = (it == ev.end()) ? (int)nao : *it;
            if (cur + (int)prow >= (int)nao) nxt = (int)nao;
            prow_max = std::max<size_t>(prow_max, nxt - cur);
            pl.panel_r0.push_back(nxt);
            cur = nxt;
        }
    }
    pl.mj = mj; pl.prow = (int)prow_max;
    pl.arena_bytes = std::max(karena, jneed(mj, prow_max));
    if (jk) pl.arena_bytes = std::max(pl.arena_bytes, j32need(mj));
    return pl.arena_bytes + (ctx->has_K ? pl.pc * stage_per_fn : 0);
}

int risp_ensure_workspace(risp_ctx *ctx, int m)
{
    if (m <= ctx->m_cap) return RISP_OK;
    risp_free_workspace(ctx);
    size_t free_b = 0, total_b = 0;
    RISP_CUDA_TRY(cudaMemGetInfo(&free_b, &total_b));
    const size_t fixed = fixed_ws_bytes(ctx) + ((ctx->flags & RISP_FLAG_KEEP_STAGES) ? (size_t)m * ctx->nocc * ctx->nvir * 8 : 0);
    size_t avail = ctx->hbm_budget > ctx->setup_bytes + fixed ? ctx->hbm_budget - ctx->setup_bytes - fixed : 0;
    avail = std::min(avail, free_b > fixed + ((size_t)256 << 20) ? free_b - fixed - ((size_t)256 << 20) : 0);
    const bool spilled = ctx->has_K && ctx->nK_dev < ctx->nauxK;
    size_t need = risp_plan_workspace(ctx, m, avail, ctx->plan, spilled);
    if (need == 0) { risp_set_error(ctx, "risp_matvec: the HBM budget leaves no room for the work space of this batch size"); return RISP_ENOMEM; }
    auto A = [&](double *&p, size_t bytes) -> int {
        if (bytes == 0) { p = nullptr; return RISP_OK; }
        RISP_CUDA_TRY(cudaMalloc((void **)&p, bytes));
        ctx->w_bytes += bytes;
        return RISP_OK;
    };
    int rc;
    if ((rc = A(ctx->w_arena, ctx->plan.arena_bytes))) return rc;
    if ((rc = A(ctx->w_dbar, (size_t)ctx->e_rows * RISP_MS * 8))) return rc;
    if ((rc = A(ctx->w_Rpart, (size_t)ctx->total_chunks * ctx->ncenJ_pad * 4 * RISP_MS * 8))) return rc;
    if ((rc = A(ctx->w_R, (size_t)ctx->nauxJ * RISP_MS * 8))) return rc;
    if ((rc = A(ctx->w_Rt, (size_t)ctx->nauxJ * RISP_MS * 8))) return rc;
    if ((rc = A(ctx->w_Rtmp, (size_t)ctx->nauxJ * RISP_MS * 8))) return rc;
    if ((rc = A(ctx->w_RtC, (size_t)((ctx->ncenJ + 31) / 32 * 32) * 4 * RISP_MS * 8))) return rc;
    if (ctx->flags & RISP_FLAG_KEEP_STAGES) { if ((rc = A(ctx->w_J, (size_t)m * ctx->nocc * ctx->nvir * 8))) return rc; }
    if (spilled)
        for (int b = 0; b < 2; ++b)
            if ((rc = A(ctx->w_stage[b], (size_t)ctx->plan.pc * (ctx->tri_o + ctx->tri_v) * 8))) return rc;
    RISP_CUDA_TRY(cudaMemset(ctx->w_Rpart, 0, (size_t)ctx->total_chunks * ctx->ncenJ_pad * 4 * RISP_MS * sizeof(double)));
    RISP_CUDA_TRY(cudaMemset(ctx->w_dbar, 0, (size_t)ctx->e_rows * RISP_MS * sizeof(double)));
    RISP_CUDA_TRY(cudaMemset(ctx->w_R, 0, (size_t)ctx->nauxJ * RISP_MS * sizeof(double)));
    ctx->m_cap = m;
    return RISP_OK;
}

// index range of an ascending list of first-AO offsets (shell A of the aoA-sorted pairs, or shell B of the aoB-sorted index)
// that falls into AO rows [r0, r1)
static void panel_pairs(const std::vector<int> &ao, int r0, int r1, int &p0, int &p1)
{
    p0 = (int)(std::lower_bound(ao.begin(), ao.end(), r0) - ao.begin());
    p1 = (int)(std::lower_bound(ao.begin(), ao.end(), r1) - ao.begin());
}

// The six pair classes of one J step touch disjoint rows of D-bar / U-bar / R partials and disjoint AO blocks, so their kernels
// run concurrently on six internal streams between a fork and a join on the caller's stream (the small classes -- a few dozen
// CTAs at 100 atoms -- would otherwise each leave most of the 148 SMs idle).
static int fork_classes(risp_ctx *ctx, cudaStream_t st)
{
    RISP_CUDA_TRY(cudaEventRecord(ctx->evFork, st));
    for (int c = 0; c < 6; ++c) RISP_CUDA_TRY(cudaStreamWaitEvent(ctx->cls_st[c], ctx->evFork, 0));
    return RISP_OK;
}
static int join_classes(risp_ctx *ctx, cudaStream_t st)
{
    for (int c = 0; c < 6; ++c) {
        RISP_CUDA_TRY(cudaEventRecord(ctx->evJoin[c], ctx->cls_st[c]));
        RISP_CUDA_TRY(cudaStreamWaitEvent(st, ctx->evJoin[c], 0));
    }
    return RISP_OK;
}

int risp_matvec_impl(risp_ctx *ctx, int m, const double *X, double *sigma, cudaStream_t st, double *sigma_minus, int phase)
{
    const bool tddft = sigma_minus != nullptr;
    if (tddft && ctx->has_K && !ctx->d_Tov) { risp_set_error(ctx, "risp_matvec_tddft: the context was set up without RISP_FLAG_TDDFT"); return RISP_EINVAL; }
    const int nao = ctx->nao, nocc = ctx->nocc, nvir = ctx->nvir, nJ = ctx->nauxJ;
    const int no = ctx->noccK, nv = ctx->nvirK, nK = ctx->nauxK, no_p = ctx->no_p, nv_p = ctx->nv_p;
    const long long ldao = ctx->ldao, ldocc = ctx->ldocc, ldvir = ctx->ldvir;
    const MatvecPlan &pl = ctx->plan;
    const int npanel = (int)pl.panel_r0.size() - 1;
    const bool dense = npanel == 1;
    int launches = 0, rc;
    cudaEvent_t *ev = ctx->ev;
    double *wY = ctx->w_arena;                                   // [mj][nocc][ldao]   (J-phase views of the arena)
    double *wD = wY + (size_t)pl.mj * nocc * ldao;               // [mj][prow][ldao]
    // RISP_PRECISION_FP32_JK: the four AO<->MO GEMMs on the tcgen05 path (gemm_tc.cu).  bf16 x 3 planes behind wD:
    //   qX [mq nocc][nvir_q]   qH [mq][nao][nocc_q] (Y^T), later [mq][nocc][nao_q] (Z)   qU [mq][nao][nao_q],   mq = vectors per sub-batch
    const long long nvir_q = (nvir + 7) & ~7, nocc_q = (nocc + 7) & ~7, nao_q = (nao + 7) & ~7, mq = std::min(pl.mj, m);
    const long long plX = mq * nocc * nvir_q, plH = mq * std::max((long long)nao * nocc_q, (long long)nocc * nao_q), plU = mq * nao * nao_q;
    const long long plCv = (long long)nao * nvir_q, plCo = (long long)nao * nocc_q, plCoT = (long long)nocc * nao_q, plCvT = (long long)nvir * nao_q;
    unsigned short *qX = (unsigned short *)(((size_t)(wD + (size_t)pl.mj * nao * ldao) + 15) & ~(size_t)15), *qH = qX + 3 * plX, *qU = qH + 3 * plH;
    bool f32j = ctx->precision == RISP_PRECISION_FP32_JK && phase == 0 && !tddft && dense && !ctx->q_C_failed &&
                (size_t)((char *)(qU + 3 * plU) - (char *)ctx->w_arena) <= ctx->plan.arena_bytes;
    if (f32j && !ctx->q_C) {
        // the MO coefficients as bf16 x 3 planes, once per context; if they do not fit the transforms stay FP64
        const size_t bytes = (size_t)6 * (plCv + plCo + plCoT + plCvT) + 64;
        if (cudaMalloc((void **)&ctx->q_C, bytes) != cudaSuccess) { (void)cudaGetLastError(); ctx->q_C = nullptr; ctx->q_C_failed = 1; f32j = false; }
        else {
            unsigned short *c = ctx->q_C;
            RISP_CUDA_TRY(risp_split_rows_bf3(ctx->d_Cvir, ldvir, nao, nvir, c, nvir_q, plCv, 0, 0, st)); c += 3 * plCv;
            RISP_CUDA_TRY(risp_split_rows_bf3(ctx->d_Cocc, ldocc, nao, nocc, c, nocc_q, plCo, 0, 0, st)); c += 3 * plCo;
            RISP_CUDA_TRY(risp_split_rows_bf3(ctx->d_CoccT, ldao, nocc, nao, c, nao_q, plCoT, 0, 0, st)); c += 3 * plCoT;
            RISP_CUDA_TRY(risp_split_transpose_bf3(ctx->d_Cvir, ldvir, nao, nvir, c, nao_q, plCvT, st));
        }
    }
    const unsigned short *qCv = ctx->q_C, *qCo = qCv + 3 * plCv, *qCoT = qCo + 3 * plCo, *qCvT = qCoT + 3 * plCoT;
    if (phase == 2) goto after_pass1;
    RISP_CUDA_TRY(cudaEventRecord(ev[0], st));
    if (phase == 1) goto density;
    // ---------------- diagonal (Eq. 10); in a sharded sigma-build rank 0 carries it
    if (ctx->shard_rank == 0) { RISP_CUDA_TRY(risp_diag_sigma(X, ctx->d_eps, sigma, m, nocc, nvir, st)); ++launches; }
    else RISP_CUDA_TRY(cudaMemsetAsync(sigma, 0, (size_t)m * nocc * nvir * sizeof(double), st));
    if (tddft) { RISP_CUDA_TRY(risp_diag_sigma(X, ctx->d_eps, sigma_minus, m, nocc, nvir, st)); ++launches; }
density:
    // ---------------- J: AO transition density (Eq. 12) on the kept pairs, in e0 space
    if (!dense) RISP_CUDA_TRY(cudaMemsetAsync(ctx->w_dbar, 0, (size_t)ctx->e_rows * RISP_MS * sizeof(double), st));   // panels accumulate
    for (int l0 = 0; l0 < m; l0 += pl.mj) {
        const int mj = std::min(pl.mj, m - l0);
        const double *Xb = X + (size_t)l0 * nocc * nvir;
        if (f32j) {
            // Y^T[mi][nu][i] = sum_a X[(mi, i)][a] C_vir[nu][a] (rows split by trial vector), then D[mi][mu][nu] = sum_i Y^T[mi][nu][i] C_occ[mu][i]
            RISP_CUDA_TRY(risp_split_rows_bf3(Xb, nvir, (long long)mj * nocc, nvir, qX, nvir_q, plX, 0, 0, st)); ++launches;
            TcGemmDesc d;
            d.M = mj * nocc; d.N = nao; d.K = nvir; d.nb = 1;
            d.A = qX; d.lda = nvir_q; d.planeA = plX; d.sA = 0;
            d.B = qCv; d.ldb = nvir_q; d.planeB = plCv; d.sB = 0;
            d.C = qH; d.ldc = nocc_q; d.sC = 0; d.planeC = plH; d.out_kind = 1; d.rpg = nocc; d.gstride = (long long)nao * nocc_q; d.accumulate = 0; d.shape = 2;
            RISP_CUDA_TRY(risp_tcgemm(d, st)); ++launches;
            TcGemmDesc e;
            e.M = nao; e.N = nao; e.K = nocc; e.nb = mj;
            e.A = qH; e.lda = nocc_q; e.planeA = plH; e.sA = (long long)nao * nocc_q;
            e.B = qCo; e.ldb = nocc_q; e.planeB = plCo; e.sB = 0;
            e.C = wD; e.ldc = ldao; e.sC = (long long)nao * ldao; e.planeC = 0; e.out_kind = 0; e.rpg = 0; e.gstride = 0; e.accumulate = 0; e.shape = 2;
            RISP_CUDA_TRY(risp_tcgemm(e, st)); ++launches;
        } else {
            GemmDesc d = gemm_desc(mj * nocc, nao, nvir, Xb, nvir, true, ctx->d_Cvir, ldvir, true, wY, ldao);
            RISP_CUDA_TRY(risp_dgemm(d, st)); ++launches;
        }
        for (int p = 0; p < npanel; ++p) {
            const int r0 = pl.panel_r0[p], r1 = pl.panel_r0[p + 1], pr = r1 - r0;
            const long long mstride = (long long)pr * ldao;
            if (!f32j) {
                // D[mu in panel][nu] = sum_i C_occ[mu][i] Y[i][nu]
                GemmDesc e = gemm_desc(pr, nao, nocc, ctx->d_Cocc + (size_t)r0 * ldocc, ldocc, true, wY, ldao, false, wD, ldao);
                e.nb1 = mj; e.sB1 = (long long)nocc * ldao; e.sC1 = mstride;
                RISP_CUDA_TRY(risp_dgemm(e, st)); ++launches;
            }
            if ((rc = fork_classes(ctx, st))) return rc;
            for (int c = 0; c < 6; ++c) {
                const PairClass &pc = ctx->cls[c];
                int p0, p1;
                panel_pairs(pc.h_aoA, r0, r1, p0, p1);
                if (p1 > p0) { RISP_CUDA_TRY(risp_dens_to_e0(pc, p0, p1, mj, l0, m, r0, ldao, mstride, dense ? 0 : 1, wD, ctx->w_dbar, ctx->cls_st[c])); ++launches; }
                if (!dense) {      // the lower-triangular pair also takes D_BA^T (reading G13), found in the panel that holds the rows of B
                    panel_pairs(pc.h_aoB, r0, r1, p0, p1);
                    if (p1 > p0) { RISP_CUDA_TRY(risp_dens_to_e0(pc, p0, p1, mj, l0, m, r0, ldao, mstride, 2, wD, ctx->w_dbar, ctx->cls_st[c])); ++launches; }
                }
            }
            if ((rc = join_classes(ctx, st))) return rc;
        }
    }
    RISP_CUDA_TRY(cudaEventRecord(ev[1], st));
    // ---------------- pass 1: R_mQ (Eq. 14)
    if ((rc = fork_classes(ctx, st))) return rc;
    for (int c = 5; c >= 0; --c)          // heaviest recursion first
        if (ctx->cls[c].npairs) {
            RISP_CUDA_TRY(risp_j_pass1(ctx->cls[c], ctx->d_prims, ctx->d_cenJ, ctx->ncenJ, ctx->ncenJ_pad, ctx->d_boys, ctx->w_dbar, ctx->w_Rpart, m, ctx->cls_st[c]));
            ++launches;
        }
    if ((rc = join_classes(ctx, st))) return rc;
    RISP_CUDA_TRY(risp_j_reduce_R(ctx->w_Rpart, ctx->total_chunks, ctx->d_cenJ, ctx->ncenJ, ctx->ncenJ_pad, ctx->w_R, st)); ++launches;
    RISP_CUDA_TRY(cudaEventRecord(ev[2], st));
    if (phase == 1) { ctx->last_m = m; return RISP_OK; }
after_pass1:
    if (phase == 2) {      // the diagonal of the second half of a sharded sigma-build
        if (ctx->shard_rank == 0) { RISP_CUDA_TRY(risp_diag_sigma(X, ctx->d_eps, sigma, m, nocc, nvir, st)); ++launches; }
        else RISP_CUDA_TRY(cudaMemsetAsync(sigma, 0, (size_t)m * nocc * nvir * sizeof(double), st));
    }
    // ---------------- R~ = (P|Q)^-1 R = L^-T (L^-1 R)  (Eq. 15)
    RISP_CUDA_TRY(risp_metric_solve32(ctx->d_LinvJ, nJ, ctx->w_R, ctx->w_Rtmp, ctx->w_Rt, st)); launches += 2;
    RISP_CUDA_TRY(risp_rt_by_centre(ctx->w_Rt, ctx->d_cenJ, ctx->ncenJ, ctx->w_RtC, st)); ++launches;
    RISP_CUDA_TRY(cudaEventRecord(ev[3], st));
    // ---------------- pass 2: U (Eq. 16), into the e0 buffer
    if ((rc = fork_classes(ctx, st))) return rc;
    for (int c = 5; c >= 0; --c)
        if (ctx->cls[c].npairs) {
            RISP_CUDA_TRY(risp_j_pass2(ctx->cls[c], ctx->d_prims, ctx->d_cenJ, ctx->ncenJ, ctx->d_boys, ctx->w_RtC, ctx->w_dbar, m, ctx->cls_st[c]));
            ++launches;
        }
    if ((rc = join_classes(ctx, st))) return rc;
    RISP_CUDA_TRY(cudaEventRecord(ev[4], st));
    // ---------------- back-transform (Eq. 17), sigma += 2 J
    for (int l0 = 0; l0 < m; l0 += pl.mj) {
        const int mj = std::min(pl.mj, m - l0);
        for (int p = 0; p < npanel; ++p) {
            const int r0 = pl.panel_r0[p], r1 = pl.panel_r0[p + 1], pr = r1 - r0;
            const long long mstride = (long long)pr * ldao;
            RISP_CUDA_TRY(cudaMemsetAsync(wD, 0, (size_t)mj * mstride * sizeof(double), st));
            if ((rc = fork_classes(ctx, st))) return rc;
            for (int c = 0; c < 6; ++c) {
                const PairClass &pc = ctx->cls[c];
                int p0, p1;
                panel_pairs(pc.h_aoA, r0, r1, p0, p1);
                if (p1 > p0) { RISP_CUDA_TRY(risp_e0_to_U(pc, p0, p1, mj, l0, r0, ldao, mstride, dense ? 0 : 1, ctx->w_dbar, wD, ctx->cls_st[c])); ++launches; }
                if (!dense) {      // complete rows of the symmetric U: the transposed blocks of the pairs whose shell B lies in the panel
                    panel_pairs(pc.h_aoB, r0, r1, p0, p1);
                    if (p1 > p0) { RISP_CUDA_TRY(risp_e0_to_U(pc, p0, p1, mj, l0, r0, ldao, mstride, 2, ctx->w_dbar, wD, ctx->cls_st[c])); ++launches; }
                }
            }
            if ((rc = join_classes(ctx, st))) return rc;
            if (f32j) continue;
            // Z[i][nu] (+)= sum_{mu in panel} C_occ[mu][i] U[mu][nu]
            GemmDesc d = gemm_desc(nocc, nao, pr, ctx->d_CoccT + r0, ldao, true, wD, ldao, false, wY, ldao, 1.0, p == 0 ? 0.0 : 1.0);
            d.nb1 = mj; d.sB1 = mstride; d.sC1 = (long long)nocc * ldao;
            RISP_CUDA_TRY(risp_dgemm(d, st)); ++launches;
        }
        double *Sb = sigma + (size_t)l0 * nocc * nvir;
        if (f32j) {
            // U is symmetric: Z[mi][i][nu] = sum_mu U[mi][nu][mu] C_occ^T[i][mu], then J[(mi, i)][a] = sum_nu C_vir^T[a][nu] Z[(mi, i)][nu];
            // J lands in the (free) Y region or in the stage buffer, sigma += 2 J
            RISP_CUDA_TRY(risp_split_rows_bf3(wD, ldao, (long long)mj * nao, nao, qU, nao_q, plU, 0, 0, st)); ++launches;
            TcGemmDesc d;
            d.M = nao; d.N = nocc; d.K = nao; d.nb = mj;
            d.A = qU; d.lda = nao_q; d.planeA = plU; d.sA = (long long)nao * nao_q;
            d.B = qCoT; d.ldb = nao_q; d.planeB = plCoT; d.sB = 0;
            d.C = qH; d.ldc = nao_q; d.sC = (long long)nocc * nao_q; d.planeC = plH; d.out_kind = 1; d.rpg = 0; d.gstride = 0; d.accumulate = 0; d.shape = 2;
            RISP_CUDA_TRY(risp_tcgemm(d, st)); ++launches;
            double *Jb = ctx->w_J ? ctx->w_J + (size_t)l0 * nocc * nvir : wY;
            TcGemmDesc e;
            e.M = nvir; e.N = mj * nocc; e.K = nao; e.nb = 1;
            e.A = qCvT; e.lda = nao_q; e.planeA = plCvT; e.sA = 0;
            e.B = qH; e.ldb = nao_q; e.planeB = plH; e.sB = 0;
            e.C = Jb; e.ldc = nvir; e.sC = 0; e.planeC = 0; e.out_kind = 0; e.rpg = 0; e.gstride = 0; e.accumulate = 0; e.shape = 2;
            RISP_CUDA_TRY(risp_tcgemm(e, st)); ++launches;
            RISP_CUDA_TRY(risp_axpy_window(Jb, 2.0, Sb, mj, nocc, nvir, 0, nocc, 0, nvir, nvir, st)); ++launches;
            continue;
        }
        if (ctx->w_J) {
            GemmDesc e = gemm_desc(mj * nocc, nvir, nao, wY, ldao, true, ctx->d_Cvir, ldvir, false, ctx->w_J + (size_t)l0 * nocc * nvir, nvir);
            RISP_CUDA_TRY(risp_dgemm(e, st)); ++launches;
        }
        // the Coulomb term enters A with 2 (ia|jb) (Eq. 10) and A+B with 4 (ia|jb) (Eq. 2a, reading G25); A-B has none
        GemmDesc e = gemm_desc(mj * nocc, nvir, nao, wY, ldao, true, ctx->d_Cvir, ldvir, false, Sb, nvir, tddft ? 4.0 : 2.0, 1.0);
        RISP_CUDA_TRY(risp_dgemm(e, st)); ++launches;
    }
    RISP_CUDA_TRY(cudaEventRecord(ev[5], st));
    // ---------------- K (Eq. 22-23)
    if (ctx->has_K) {
        const bool f32 = ctx->precision != RISP_PRECISION_FP64;
        if (f32 && tddft) { risp_set_error(ctx, "risp_matvec_tddft: the single-precision mode covers the TDA sigma-build only"); return RISP_EINVAL; }
        int pc = pl.pc;
        double *wXk = ctx->w_arena;                                  // [m][no][nv_p]
        double *wKk = wXk + (size_t)m * no * nv_p;                   // [m][no][nv_p]
        double *wM = wKk + (size_t)m * no * nv_p;                    // [m][pc][no_p][nv_p]
        double *wTab = wM + (size_t)m * pc * no_p * nv_p;            // [pc][nv][nv_p]
        double *wTij = wTab + (size_t)pc * nv * nv_p;                // [no][pc][no_p]
        // single-precision mode (gemm_tc.cu): every operand is three bf16 planes with rows padded to 8 elements;
        // K' stays FP64 (the chunks are summed in FP64), X' FP64 is not needed
        const long long nv_q = (nv + 7) & ~7, no_q = (no + 7) & ~7;
        long long ldK = 0, plX = 0, plM = 0, plTab = 0, plTij = 0;
        unsigned short *qX = nullptr, *qM = nullptr, *qTab = nullptr, *qTij = nullptr;      // bf16 bit patterns
        if (f32) {
            auto need = [&](long long c) {
                return 8 * (size_t)m * no * nv_p + 6 * ((size_t)m * no * nv_q + (size_t)m * nv * c * no_q + (size_t)c * nv * nv_q + (size_t)no * c * no_q) + 64;
            };
            while (pc > 1 && need(pc) > ctx->plan.arena_bytes) --pc;
            if (need(pc) > ctx->plan.arena_bytes) { risp_set_error(ctx, "risp_matvec: work space too small for the single-precision K contractions"); return RISP_ENOMEM; }
            ldK = (long long)pc * no_q;
            plX = (long long)m * no * nv_q; plM = (long long)m * nv * ldK; plTab = (long long)pc * nv * nv_q; plTij = (long long)no * ldK;
            wKk = ctx->w_arena;
            qX = (unsigned short *)(((size_t)(wKk + (size_t)m * no * nv_p) + 15) & ~(size_t)15);
            qM = qX + 3 * plX; qTab = qM + 3 * plM; qTij = qTab + 3 * plTab;
            if (no_q != no) {       // the padding columns j of (P, j) enter Eq. 23 as 0 * M: both must be finite, T_ij's must be zero
                RISP_CUDA_TRY(cudaMemsetAsync(qM, 0, (size_t)3 * plM * 2, st));
                RISP_CUDA_TRY(cudaMemsetAsync(qTij, 0, (size_t)3 * plTij * 2, st));
            }
            RISP_CUDA_TRY(risp_split_rows_bf3(X + (size_t)ctx->occK0 * nvir + ctx->virK0, nvir, (long long)m * no, nv, qX, nv_q, plX, no,
                                              (long long)nocc * nvir, st)); ++launches;
        } else
        if (nv_p != nv) {   // padding columns of X' must not carry NaNs of the J phase into the TMA boxes (they are never read
                            // as operands -- K = nv bounds the boxes -- but keep the buffers clean anyway)
            RISP_CUDA_TRY(cudaMemsetAsync(wXk, 0, (size_t)m * no * nv_p * sizeof(double), st));
        }
        if (!f32) { RISP_CUDA_TRY(risp_gather_window(X, wXk, m, nocc, nvir, ctx->occK0, no, ctx->virK0, nv, nv_p, st)); ++launches; }
        if (!f32 && no_p != no) {
            // the contraction index (P, j) of Eq. 23 runs over no_p per P: the padding row of M and the padding column of T_ij are zero
            RISP_CUDA_TRY(cudaMemset2DAsync(wM + (size_t)no * nv_p, (size_t)no_p * nv_p * 8, 0, (size_t)nv_p * 8, (size_t)m * pc, st));
            RISP_CUDA_TRY(cudaMemset2DAsync(wTij + no, (size_t)no_p * 8, 0, 8, (size_t)no * pc, st));
        }
        RISP_CUDA_TRY(cudaEventRecord(ev[6], st));
        // chunk list: [p0, p0+np) never straddles the device / host boundary
        struct Chunk { int p0, np; bool host; };
        std::vector<Chunk> chunks;
        for (int p0 = 0; p0 < nK;) {
            const bool host = p0 >= ctx->nK_dev;
            const int lim = host ? nK : ctx->nK_dev;
            const int np = std::min(pc, lim - p0);
            chunks.push_back({p0, np, host});
            p0 += np;
        }
        const size_t stage_tab_off = (size_t)pc * ctx->tri_o;        // staging buffer: [pc][tri_o] then [pc][tri_v]
        auto prefetch = [&](int ci, int buf) -> int {
            const Chunk &c = chunks[ci];
            const size_t h0 = (size_t)(c.p0 - ctx->nK_dev);
            RISP_CUDA_TRY(cudaStreamWaitEvent(ctx->side, ctx->evStageFree[buf], 0));
            RISP_CUDA_TRY(cudaMemcpyAsync(ctx->w_stage[buf], ctx->h_TijP + h0 * ctx->tri_o, (size_t)c.np * ctx->tri_o * 8, cudaMemcpyHostToDevice, ctx->side));
            RISP_CUDA_TRY(cudaMemcpyAsync(ctx->w_stage[buf] + stage_tab_off, ctx->h_TabP + h0 * ctx->tri_v, (size_t)c.np * ctx->tri_v * 8,
                                          cudaMemcpyHostToDevice, ctx->side));
            RISP_CUDA_TRY(cudaEventRecord(ctx->evStage[buf], ctx->side));
            return RISP_OK;
        };
        int first_host = -1;
        for (size_t i = 0; i < chunks.size(); ++i) if (chunks[i].host) { first_host = (int)i; break; }
        int nhost_seen = 0;
        if (first_host >= 0 && (rc = prefetch(first_host, 0))) return rc;
        for (size_t ci = 0; ci < chunks.size(); ++ci) {
            const Chunk &c = chunks[ci];
            const double *pij, *pab;
            int buf = -1;
            if (c.host) {
                buf = nhost_seen & 1;
                if (ci + 1 < chunks.size() && (rc = prefetch((int)ci + 1, buf ^ 1))) return rc;   // every later chunk is host resident too
                RISP_CUDA_TRY(cudaStreamWaitEvent(st, ctx->evStage[buf], 0));
                pij = ctx->w_stage[buf]; pab = ctx->w_stage[buf] + stage_tab_off;
                ++nhost_seen;
            } else {
                pij = ctx->d_TijP + (size_t)c.p0 * ctx->tri_o; pab = ctx->d_TabP + (size_t)c.p0 * ctx->tri_v;
            }
            if (f32) {
                // packed lower triangles -> bf16 planes of T_ab [P][a][b] and T_ij [i][(P, j)]
                RISP_CUDA_TRY(risp_expand_sym_bf3(pab, ctx->tri_v, nv, c.np, qTab, nv_q, (long long)nv * nv_q, plTab, st)); ++launches;
                RISP_CUDA_TRY(risp_expand_sym_bf3(pij, ctx->tri_o, no, c.np, qTij, ldK, no_q, plTij, st)); ++launches;
                if (c.host) RISP_CUDA_TRY(cudaEventRecord(ctx->evStageFree[buf], st));
                if (ci == 0) RISP_CUDA_TRY(cudaEventRecord(ev[11], st));
                // Eq. 22, stored transposed: Mt[mi][a][(P, j)] = sum_b X'[(mi, j)][b] T_ab^P[a][b]
                TcGemmDesc d;
                d.M = m * no; d.N = nv; d.K = nv; d.nb = c.np;
                d.A = qX; d.lda = nv_q; d.planeA = plX; d.sA = 0;
                d.B = qTab; d.ldb = nv_q; d.planeB = plTab; d.sB = (long long)nv * nv_q;
                d.C = qM; d.ldc = ldK; d.sC = no_q; d.planeC = plM; d.out_kind = 1; d.rpg = no; d.gstride = (long long)nv * ldK; d.accumulate = 0; d.seg_kb = ctx->tc_seg22; d.shape = ctx->tc_shape22 >= 0 ? ctx->tc_shape22 : 2;
                RISP_CUDA_TRY(risp_tcgemm(d, st)); ++launches;
                if (ci == 0) RISP_CUDA_TRY(cudaEventRecord(ev[9], st));
                // Eq. 23, stored transposed: K'[mi][i][a] (+)= sum_{(P, j)} Mt[mi][a][(P, j)] T_ij[i][(P, j)]
                TcGemmDesc e;
                e.M = nv; e.N = no; e.K = (int)(c.np * no_q); e.nb = m;
                e.A = qM; e.lda = ldK; e.planeA = plM; e.sA = (long long)nv * ldK;
                e.B = qTij; e.ldb = ldK; e.planeB = plTij; e.sB = 0;
                e.C = wKk; e.ldc = nv_p; e.sC = (long long)no * nv_p; e.planeC = 0; e.out_kind = 0; e.rpg = 0; e.gstride = 0; e.accumulate = ci != 0; e.seg_kb = ctx->tc_seg23; e.shape = ctx->tc_shape23 >= 0 ? ctx->tc_shape23 : 2;
                RISP_CUDA_TRY(risp_tcgemm(e, st)); ++launches;
                if (ci == 0) { RISP_CUDA_TRY(cudaEventRecord(ev[10], st)); ctx->tim.first_chunk_naux = c.np; }
                continue;
            }
            // packed lower triangles -> T_ab [P][a][b] and T_ij [i][(P, j)]
            RISP_CUDA_TRY(risp_expand_sym(pab, ctx->tri_v, nv, c.np, wTab, nv_p, (long long)nv * nv_p, st)); ++launches;
            RISP_CUDA_TRY(risp_expand_sym(pij, ctx->tri_o, no, c.np, wTij, (long long)pc * no_p, no_p, st)); ++launches;
            if (c.host) RISP_CUDA_TRY(cudaEventRecord(ctx->evStageFree[buf], st));
            if (ci == 0) RISP_CUDA_TRY(cudaEventRecord(ev[11], st));
            // M[mi][P][j][a] = sum_b X'[mi][j][b] T_ab^P[a][b]; rows (mi,j) of one P are split by mi
            GemmDesc d = gemm_desc(m * no, nv, nv, wXk, nv_p, true, wTab, nv_p, true, wM, nv_p);
            d.nb1 = c.np; d.sB1 = (long long)nv * nv_p; d.sC1 = (long long)no_p * nv_p;
            d.c_rpg = no; d.c_gstride = (long long)pc * no_p * nv_p;
            RISP_CUDA_TRY(risp_dgemm(d, st)); ++launches;
            if (ci == 0) RISP_CUDA_TRY(cudaEventRecord(ev[9], st));
            // K'[mi][i][a] (+)= sum_{(P,j)} T_ij[i][(P,j)] M[mi][(P,j)][a]
            GemmDesc e = gemm_desc(no, nv, c.np * no_p, wTij, (long long)pc * no_p, true, wM, nv_p, false, wKk, nv_p, 1.0, ci == 0 ? 0.0 : 1.0);
            e.nb1 = m; e.sB1 = (long long)pc * no_p * nv_p; e.sC1 = (long long)no * nv_p;
            RISP_CUDA_TRY(risp_dgemm(e, st)); ++launches;
            if (ci == 0) { RISP_CUDA_TRY(cudaEventRecord(ev[10], st)); ctx->tim.first_chunk_naux = c.np; }
        }
        RISP_CUDA_TRY(cudaEventRecord(ev[7], st));
        RISP_CUDA_TRY(risp_sub_window(wKk, sigma, m, nocc, nvir, ctx->occK0, no, ctx->virK0, nv, nv_p, st)); ++launches;
        if (tddft) {
            RISP_CUDA_TRY(risp_sub_window(wKk, sigma_minus, m, nocc, nvir, ctx->occK0, no, ctx->virK0, nv, nv_p, st)); ++launches;
            // ---------------- (ib|ja) term of full TDDFT (Eq. 2): K2_mia = sum_P sum_j (sum_b T_ib^P X'_mjb) T_ja^P with the whitened
            //                  T^P = L_K^-1 (ov|J^|Q).  Contracting b first costs 4 m N_auxK o'^2 v' flops (o' < v').
            const long long ldw_max = (long long)((ctx->plan.arena_bytes / 8 - 2 * (size_t)m * no * nv_p) / ((size_t)m * no)) & ~1LL;
            const int pc2 = (int)std::min<long long>(nK, ldw_max / std::max(no, 1));
            if (pc2 < 1) { risp_set_error(ctx, "risp_matvec_tddft: work space too small for the (ib|ja) contraction"); return RISP_ENOMEM; }
            const long long ldw = ((long long)pc2 * no + 1) & ~1LL;
            double *wW = wKk + (size_t)m * no * nv_p;                   // [m][no][ldw]: W_m[i][(P, j)] = sum_b T_ib^P X'_mjb
            for (int p0 = 0; p0 < nK; p0 += pc2) {
                const int np = std::min(pc2, nK - p0);
                const double *Tp = ctx->d_Tov + (size_t)p0 * no * nv_p;
                GemmDesc d = gemm_desc(no, no, nv, Tp, nv_p, true, wXk, nv_p, true, wW, ldw);
                d.nb1 = np; d.sA1 = (long long)no * nv_p; d.sB1 = 0; d.sC1 = no;
                d.nb2 = m; d.sA2 = 0; d.sB2 = (long long)no * nv_p; d.sC2 = (long long)no * ldw;
                RISP_CUDA_TRY(risp_dgemm(d, st)); ++launches;
                GemmDesc e = gemm_desc(no, nv, np * no, wW, ldw, true, Tp, nv_p, false, wKk, nv_p, 1.0, p0 == 0 ? 0.0 : 1.0);
                e.nb1 = m; e.sA1 = (long long)no * ldw; e.sB1 = 0; e.sC1 = (long long)no * nv_p;
                RISP_CUDA_TRY(risp_dgemm(e, st)); ++launches;
            }
            RISP_CUDA_TRY(risp_axpy_window(wKk, -1.0, sigma, m, nocc, nvir, ctx->occK0, no, ctx->virK0, nv, nv_p, st)); ++launches;
            RISP_CUDA_TRY(risp_axpy_window(wKk, 1.0, sigma_minus, m, nocc, nvir, ctx->occK0, no, ctx->virK0, nv, nv_p, st)); ++launches;
        }
    } else {
        RISP_CUDA_TRY(cudaEventRecord(ev[6], st));
        RISP_CUDA_TRY(cudaEventRecord(ev[7], st));
    }
    RISP_CUDA_TRY(cudaEventRecord(ev[8], st));
    ctx->tim.kernel_launches = launches;
    ctx->last_m = m;
    return RISP_OK;
}

// m > 32 is worked through in sub-batches of 32 (one lane per trial vector in the integral passes)
extern "C" int risp_matvec(risp_ctx *ctx, int32_t m, const double *X_dev, double *sigma_dev, void *cuda_stream)
{
    if (!ctx) return RISP_EINVAL;
    if (m <= 0 || !X_dev || !sigma_dev) { risp_set_error(ctx, "risp_matvec: need m >= 1 and non-NULL device pointers"); return RISP_EINVAL; }
    const size_t vec = (size_t)ctx->nocc * ctx->nvir, bytes = (size_t)m * vec * sizeof(double);
    const char *x = (const char *)X_dev, *s = (const char *)sigma_dev;
    if (x < s + bytes && s < x + bytes) { risp_set_error(ctx, "risp_matvec: X and sigma overlap"); return RISP_EINVAL; }
    RISP_CUDA_TRY(cudaSetDevice(ctx->device));
    int rc = risp_ensure_workspace(ctx, std::min<int>(m, RISP_MS));
    if (rc) return rc;
    for (int m0 = 0; m0 < m; m0 += RISP_MS)
        if ((rc = risp_matvec_impl(ctx, std::min<int>(RISP_MS, m - m0), X_dev + (size_t)m0 * vec, sigma_dev + (size_t)m0 * vec, (cudaStream_t)cuda_stream))) return rc;
    return RISP_OK;
}

extern "C" int risp_matvec_host(risp_ctx *ctx, int32_t m, const double *X_host, double *sigma_host)
{
    if (!ctx) return RISP_EINVAL;
    if (m <= 0 || !X_host || !sigma_host) { risp_set_error(ctx, "risp_matvec_host: need m >= 1 and non-NULL host pointers"); return RISP_EINVAL; }
    RISP_CUDA_TRY(cudaSetDevice(ctx->device));
    const size_t vec = (size_t)ctx->nocc * ctx->nvir;
    const int mb = std::min<int>(m, RISP_MS);
    if (mb > ctx->xin_cap) {
        // the staging copies of X and sigma are the caller's share of HBM in this entry point: allocate them before the work space is planned
        risp_free_workspace(ctx);
        if (ctx->w_Xin) { cudaFree(ctx->w_Xin); ctx->w_Xin = nullptr; }
        if (ctx->w_Sout) { cudaFree(ctx->w_Sout); ctx->w_Sout = nullptr; }
        ctx->xin_cap = 0;
        RISP_CUDA_TRY(cudaMalloc((void **)&ctx->w_Xin, (size_t)mb * vec * sizeof(double)));
        RISP_CUDA_TRY(cudaMalloc((void **)&ctx->w_Sout, (size_t)mb * vec * sizeof(double)));
        ctx->xin_cap = mb;
    }
    int rc = risp_ensure_workspace(ctx, mb);
    if (rc) return rc;
    for (int m0 = 0; m0 < m; m0 += RISP_MS) {
        const int mc = std::min<int>(RISP_MS, m - m0);
        const size_t bytes = (size_t)mc * vec * sizeof(double);
        RISP_CUDA_TRY(cudaMemcpyAsync(ctx->w_Xin, X_host + (size_t)m0 * vec, bytes, cudaMemcpyHostToDevice, 0));
        if ((rc = risp_matvec_impl(ctx, mc, ctx->w_Xin, ctx->w_Sout, 0))) return rc;
        RISP_CUDA_TRY(cudaMemcpyAsync(sigma_host + (size_t)m0 * vec, ctx->w_Sout, bytes, cudaMemcpyDeviceToHost, 0));
    }
    RISP_CUDA_TRY(cudaStreamSynchronize(0));
    return RISP_OK;
}

// P-sharded sigma-build: first half -- this rank's pairs contribute to R_mQ (Eq. 14)
extern "C" int risp_matvec_shard_begin(risp_ctx *ctx, int32_t m, const double *X_dev, double *R_partial_dev, void *cuda_stream)
{
    if (!ctx) return RISP_EINVAL;
    if (m <= 0 || m > RISP_MS || !X_dev || !R_partial_dev) { risp_set_error(ctx, "risp_matvec_shard_begin: need 1 <= m <= 32 and non-NULL device pointers"); return RISP_EINVAL; }
    RISP_CUDA_TRY(cudaSetDevice(ctx->device));
    int rc = risp_ensure_workspace(ctx, m);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = risp_matvec_impl(ctx, m, X_dev, nullptr, st, nullptr, 1))) return rc;
    RISP_CUDA_TRY(cudaMemcpyAsync(R_partial_dev, ctx->w_R, (size_t)ctx->nauxJ * RISP_MS * sizeof(double), cudaMemcpyDeviceToDevice, st));
    return RISP_OK;
}

// second half: R_dev holds the sum of all shards' partial R; returns this rank's share of sigma (rank 0 carries the diagonal)
extern "C" int risp_matvec_shard_end(risp_ctx *ctx, int32_t m, const double *X_dev, const double *R_dev, double *sigma_partial_dev, void *cuda_stream)
{
    if (!ctx) return RISP_EINVAL;
    if (m <= 0 || m > RISP_MS || !X_dev || !R_dev || !sigma_partial_dev) { risp_set_error(ctx, "risp_matvec_shard_end: need 1 <= m <= 32 and non-NULL device pointers"); return RISP_EINVAL; }
    if (m != ctx->last_m || m > ctx->m_cap) { risp_set_error(ctx, "risp_matvec_shard_end: no matching risp_matvec_shard_begin"); return RISP_EINVAL; }
    RISP_CUDA_TRY(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    RISP_CUDA_TRY(cudaMemcpyAsync(ctx->w_R, R_dev, (size_t)ctx->nauxJ * RISP_MS * sizeof(double), cudaMemcpyDeviceToDevice, st));
    return risp_matvec_impl(ctx, m, X_dev, sigma_partial_dev, st, nullptr, 2);
}

// (A+B) X and (A-B) X of full TDDFT-risp (Eq. 2) for m trial vectors; same conventions as risp_matvec
extern "C" int risp_matvec_tddft(risp_ctx *ctx, int32_t m, const double *X_dev, double *sigma_plus_dev, double *sigma_minus_dev, void *cuda_stream)
{
    if (!ctx) return RISP_EINVAL;
    if (m <= 0 || !X_dev || !sigma_plus_dev || !sigma_minus_dev) { risp_set_error(ctx, "risp_matvec_tddft: need m >= 1 and non-NULL device pointers"); return RISP_EINVAL; }
    const size_t vec = (size_t)ctx->nocc * ctx->nvir, bytes = (size_t)m * vec * sizeof(double);
    const char *x = (const char *)X_dev, *a = (const char *)sigma_plus_dev, *b = (const char *)sigma_minus_dev;
    if ((x < a + bytes && a < x + bytes) || (x < b + bytes && b < x + bytes) || (a < b + bytes && b < a + bytes)) {
        risp_set_error(ctx, "risp_matvec_tddft: X, sigma_plus and sigma_minus overlap"); return RISP_EINVAL;
    }
    if (!(ctx->flags & RISP_FLAG_TDDFT)) { risp_set_error(ctx, "risp_matvec_tddft: the context was set up without RISP_FLAG_TDDFT"); return RISP_EINVAL; }
    RISP_CUDA_TRY(cudaSetDevice(ctx->device));
    int rc = risp_ensure_workspace(ctx, std::min<int>(m, RISP_MS));
    if (rc) return rc;
    for (int m0 = 0; m0 < m; m0 += RISP_MS)
        if ((rc = risp_matvec_impl(ctx, std::min<int>(RISP_MS, m - m0), X_dev + (size_t)m0 * vec, sigma_plus_dev + (size_t)m0 * vec, (cudaStream_t)cuda_stream,
                                   sigma_minus_dev + (size_t)m0 * vec))) return rc;
    return RISP_OK;
}

// Testing: override the work-space plan of the next risp_matvec (0 = automatic).
extern "C" int risp_debug_force_plan(risp_ctx *ctx, int mj, int prow, int pc)
{
    if (!ctx) return RISP_EINVAL;
    cudaSetDevice(ctx->device);
    cudaDeviceSynchronize();
    risp_free_workspace(ctx);
    ctx->force_mj = mj; ctx->force_prow = prow; ctx->force_pc = pc;
    return RISP_OK;
}
