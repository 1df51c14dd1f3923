// api.cu -- the remaining C-ABI entry points of include/risp.h: teardown, error text, parity getters.
#include "ctx.h"

using namespace risp_eri;

extern "C" void risp_destroy(risp_ctx *ctx)
{
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    cudaDeviceSynchronize();
    risp_free_workspace(ctx);
    if (ctx->w_Xin) cudaFree(ctx->w_Xin);
    if (ctx->q_C) cudaFree(ctx->q_C);
    if (ctx->w_Sout) cudaFree(ctx->w_Sout);
    double **bufs[] = {&ctx->d_Cocc, &ctx->d_CoccT, &ctx->d_Cvir, &ctx->d_eps, &ctx->d_boys, &ctx->d_MJ, &ctx->d_LinvJ, &ctx->d_MK, &ctx->d_MKinv, &ctx->d_TijP,
                       &ctx->d_TabP, &ctx->d_Tov, &ctx->d_LinvK};
    for (auto b : bufs) if (*b) cudaFree(*b);
    if (ctx->h_TijP) cudaFreeHost(ctx->h_TijP);
    if (ctx->h_TabP) cudaFreeHost(ctx->h_TabP);
    for (int c = 0; c < 6; ++c) { if (ctx->cls[c].d_pairs) cudaFree(ctx->cls[c].d_pairs); if (ctx->cls[c].d_permB) cudaFree(ctx->cls[c].d_permB); }
    if (ctx->d_prims) cudaFree(ctx->d_prims);
    if (ctx->d_oneel_shl) cudaFree(ctx->d_oneel_shl);
    if (ctx->d_prim_exp) cudaFree(ctx->d_prim_exp);
    if (ctx->d_prim_d) cudaFree(ctx->d_prim_d);
    if (ctx->d_cenJ) cudaFree(ctx->d_cenJ);
    if (ctx->d_cenK) cudaFree(ctx->d_cenK);
    if (ctx->ev_ok) {
        for (int i = 0; i < RISP_NEV; ++i) cudaEventDestroy(ctx->ev[i]);
        for (int b = 0; b < 2; ++b) { cudaEventDestroy(ctx->evStage[b]); cudaEventDestroy(ctx->evStageFree[b]); }
        cudaEventDestroy(ctx->evFork);
        for (int c = 0; c < 6; ++c) { cudaEventDestroy(ctx->evJoin[c]); cudaStreamDestroy(ctx->cls_st[c]); }
    }
    if (ctx->side) cudaStreamDestroy(ctx->side);
    delete ctx;
}

extern "C" const char *risp_last_error(const risp_ctx *ctx)
{
    if (!ctx) return "risp: no context (risp_setup was given a NULL argument or could not allocate)";
    return ctx->err.c_str();
}

extern "C" int risp_get_dims(const risp_ctx *ctx, risp_dims *out)
{
    if (!ctx || !out) return RISP_EINVAL;
    std::memset(out, 0, sizeof(*out));
    out->nao = ctx->nao; out->nocc = ctx->nocc; out->nvir = ctx->nvir; out->nauxJ = ctx->nauxJ; out->nauxK = ctx->nauxK;
    out->noccK = ctx->noccK; out->nvirK = ctx->nvirK; out->occK_first = ctx->occK0; out->virK_first = ctx->virK0;
    out->n_shell_pairs = ctx->n_shell_pairs; out->n_shell_pairs_kept = ctx->n_shell_pairs_kept; out->n_ao_pairs_kept = ctx->n_ao_pairs_kept;
    out->bytes_Tij = ctx->has_K ? (int64_t)ctx->nauxK * ctx->tri_o * 8 : 0;
    out->bytes_Tab = ctx->has_K ? (int64_t)ctx->nauxK * ctx->tri_v * 8 : 0;
    out->bytes_device_total = (int64_t)(ctx->setup_bytes + ctx->w_bytes);
    out->aux_chunk = ctx->plan.pc;
    out->nauxK_device = ctx->has_K ? ctx->nK_dev : 0;
    out->bytes_T_host = ctx->has_K ? (int64_t)(ctx->nauxK - ctx->nK_dev) * (ctx->tri_o + ctx->tri_v) * 8 : 0;
    out->j_sub_batch = ctx->plan.mj;
    out->j_panels = ctx->plan.panel_r0.empty() ? 0 : (int)ctx->plan.panel_r0.size() - 1;
    for (int c = 0; c < 6; ++c) out->pairs_per_class[c] = ctx->cls[c].npairs;
    out->n_aux_centres = ctx->ncenJ;
    return RISP_OK;
}

extern "C" int risp_get_timings(const risp_ctx *cctx, risp_timings *out)
{
    risp_ctx *ctx = const_cast<risp_ctx *>(cctx);
    if (!ctx || !out) return RISP_EINVAL;
    std::memset(out, 0, sizeof(*out));
    if (!ctx->last_m) return RISP_OK;
    RISP_CUDA_TRY(cudaEventSynchronize(ctx->ev[8]));
    auto el = [&](int a, int b) { float ms = 0; cudaEventElapsedTime(&ms, ctx->ev[a], ctx->ev[b]); return (double)ms * 1e-3; };
    out->total = el(0, 8);
    out->j_transform_in = el(0, 1); out->j_pass1 = el(1, 2); out->j_solve = el(2, 3); out->j_pass2 = el(3, 4); out->j_transform_out = el(4, 5);
    out->k_gather = el(5, 6); out->k_total = el(6, 7); out->assemble = el(7, 8);
    if (ctx->has_K) { out->k_gemm1 = el(11, 9); out->k_gemm2 = el(9, 10); }
    out->kernel_launches = ctx->tim.kernel_launches;
    out->first_chunk_naux = ctx->tim.first_chunk_naux;
    return RISP_OK;
}

extern "C" int risp_eri3c_shell(risp_ctx *ctx, int32_t shl_i, int32_t shl_j, int32_t aux_k, int32_t op, double *out_host)
{
    if (!ctx) return RISP_EINVAL;
    if (shl_i < 0 || shl_i >= ctx->nshl || shl_j < 0 || shl_j >= ctx->nshl || aux_k < 0 || aux_k >= (int)ctx->h_aux_l.size() || !out_host ||
        (op != 0 && op != 1)) {
        risp_set_error(ctx, "risp_eri3c_shell: index out of range");
        return RISP_EINVAL;
    }
    RISP_CUDA_TRY(cudaSetDevice(ctx->device));
    int A = shl_i, B = shl_j;
    bool swapped = ctx->h_shl_l[A] < ctx->h_shl_l[B];
    if (swapped) std::swap(A, B);
    ShellPair sp;
    std::vector<PrimPair> pp;
    risp_build_pair(ctx, A, B, sp, pp, -1.0);
    sp.aoA = 0; sp.aoB = 0;
    const int la = ctx->h_shl_l[A], lb = ctx->h_shl_l[B], nfa = 2 * la + 1, nfb = 2 * lb + 1;
    const int lk = ctx->h_aux_l[aux_k], nk = 2 * lk + 1;
    AuxCentre c;
    int at = ctx->h_aux_atom[aux_k];
    c.x = ctx->h_xyz[3 * at]; c.y = ctx->h_xyz[3 * at + 1]; c.z = ctx->h_xyz[3 * at + 2];
    c.g = ctx->h_aux_exp[aux_k];
    c.ns = std::pow(2.0 * c.g / 3.14159265358979323846, 0.75);
    c.np = c.ns * 2.0 * std::sqrt(c.g);
    c.ig = 1.0 / c.g;
    c.qs = lk == 0 ? 0 : -1; c.qp = lk == 1 ? 0 : -1;
    DevScratch scr;
    ShellPair *d_sp = nullptr; PrimPair *d_pp = nullptr; AuxCentre *d_c = nullptr; double *d_out = nullptr;
    RISP_CUDA_TRY(scr.alloc(d_sp, 1));
    RISP_CUDA_TRY(scr.alloc(d_pp, pp.size()));
    RISP_CUDA_TRY(scr.alloc(d_c, 1));
    RISP_CUDA_TRY(scr.alloc(d_out, (size_t)nk * nfa * nfb));
    RISP_CUDA_TRY(cudaMemcpy(d_sp, &sp, sizeof(sp), cudaMemcpyHostToDevice));
    RISP_CUDA_TRY(cudaMemcpy(d_pp, pp.data(), pp.size() * sizeof(PrimPair), cudaMemcpyHostToDevice));
    RISP_CUDA_TRY(cudaMemcpy(d_c, &c, sizeof(c), cudaMemcpyHostToDevice));
    OpParams o{1.0, 0.0, 0.0};
    if (op == 1) o = OpParams{ctx->alpha, ctx->beta, ctx->omega * ctx->omega};
    RISP_CUDA_TRY(risp_eri_fill(la, lb, lk == 1, op == 1, d_sp, 1, d_pp, d_c, 1, o, ctx->d_boys, d_out, (long long)nfa * nfb, nfb, 0, 0));
    std::vector<double> h((size_t)nk * nfa * nfb);
    RISP_CUDA_TRY(cudaMemcpy(h.data(), d_out, h.size() * sizeof(double), cudaMemcpyDeviceToHost));
    // h[k][a][b] -> out[i][j][k]
    const int nfi = swapped ? nfb : nfa, nfj = swapped ? nfa : nfb;
    for (int i = 0; i < nfi; ++i)
        for (int j = 0; j < nfj; ++j)
            for (int k = 0; k < nk; ++k) {
                int a = swapped ? j : i, b = swapped ? i : j;
                out_host[((size_t)i * nfj + j) * nk + k] = h[((size_t)k * nfa + a) * nfb + b];
            }
    return RISP_OK;
}

extern "C" int risp_get_stage(risp_ctx *ctx, int32_t which, const int64_t *sel, int64_t nsel, void *out_host)
{
    if (!ctx || !out_host) return RISP_EINVAL;
    RISP_CUDA_TRY(cudaSetDevice(ctx->device));
    RISP_CUDA_TRY(cudaDeviceSynchronize());
    const int m = ctx->last_m;
    double *out = (double *)out_host;
    DevScratch scr;
    auto need_mv = [&]() { if (!m) { risp_set_error(ctx, "risp_get_stage: no risp_matvec has run"); return true; } return false; };
    switch (which) {
    case RISP_STAGE_R:
    case RISP_STAGE_RTILDE: {
        if (need_mv()) return RISP_EINVAL;
        RISP_CUDA_TRY(cudaMemcpy2D(out, (size_t)m * 8, which == RISP_STAGE_R ? ctx->w_R : ctx->w_Rt, (size_t)RISP_MS * 8, (size_t)m * 8, ctx->nauxJ,
                                   cudaMemcpyDeviceToHost));
        return RISP_OK;
    }
    case RISP_STAGE_J:
        if (need_mv()) return RISP_EINVAL;
        if (!ctx->w_J) { risp_set_error(ctx, "risp_get_stage: J is kept only with RISP_FLAG_KEEP_STAGES"); return RISP_EINVAL; }
        RISP_CUDA_TRY(cudaMemcpy(out, ctx->w_J, (size_t)m * ctx->nocc * ctx->nvir * 8, cudaMemcpyDeviceToHost));
        return RISP_OK;
    case RISP_STAGE_K: {
        if (need_mv()) return RISP_EINVAL;
        size_t n = (size_t)m * ctx->nocc * ctx->nvir;
        if (!ctx->has_K) { std::memset(out, 0, n * 8); return RISP_OK; }
        double *tmp = nullptr;
        RISP_CUDA_TRY(scr.alloc(tmp, n));
        // K' of the last matvec (matvec.cu arena layout: behind X' in FP64 mode, first in the single-precision mode)
        const double *wKk = ctx->w_arena + (ctx->precision != RISP_PRECISION_FP64 ? 0 : (size_t)m * ctx->noccK * ctx->nv_p);
        RISP_CUDA_TRY(risp_scatter_window(wKk, tmp, m, ctx->nocc, ctx->nvir, ctx->occK0, ctx->noccK, ctx->virK0, ctx->nvirK, ctx->nv_p, 0));
        RISP_CUDA_TRY(cudaMemcpy(out, tmp, n * 8, cudaMemcpyDeviceToHost));
        return RISP_OK;
    }
    case RISP_STAGE_TIJ:
    case RISP_STAGE_TAB: {
        if (!ctx->has_K || !sel) { risp_set_error(ctx, "risp_get_stage: no K tensors / no selection"); return RISP_EINVAL; }
        const bool ij = which == RISP_STAGE_TIJ;
        const size_t n = ij ? ctx->noccK : ctx->nvirK, nK = ctx->nauxK;
        const long long tri = ij ? ctx->tri_o : ctx->tri_v;
        double *full = nullptr, *pk = nullptr;
        RISP_CUDA_TRY(scr.alloc(full, n * n));
        RISP_CUDA_TRY(scr.alloc(pk, (size_t)tri));
        for (int64_t s = 0; s < nsel; ++s) {
            if (sel[s] < 0 || sel[s] >= (int64_t)nK) { risp_set_error(ctx, "risp_get_stage: aux index out of range"); return RISP_EINVAL; }
            const double *src;
            if (sel[s] < ctx->nK_dev) src = (ij ? ctx->d_TijP : ctx->d_TabP) + (size_t)sel[s] * tri;
            else {
                RISP_CUDA_TRY(cudaMemcpy(pk, (ij ? ctx->h_TijP : ctx->h_TabP) + (size_t)(sel[s] - ctx->nK_dev) * tri, (size_t)tri * 8, cudaMemcpyHostToDevice));
                src = pk;
            }
            RISP_CUDA_TRY(risp_expand_sym(src, tri, (int)n, 1, full, (long long)n, 0, 0));
            RISP_CUDA_TRY(cudaMemcpy(out + s * n * n, full, n * n * 8, cudaMemcpyDeviceToHost));
        }
        return RISP_OK;
    }
    case RISP_STAGE_PAIRS:
        std::memcpy(out_host, ctx->h_kept_pairs.data(), ctx->h_kept_pairs.size() * sizeof(long long));
        return RISP_OK;
    case RISP_STAGE_METRIC_J:
        RISP_CUDA_TRY(cudaMemcpy(out, ctx->d_MJ, (size_t)ctx->nauxJ * ctx->nauxJ * 8, cudaMemcpyDeviceToHost));
        return RISP_OK;
    case RISP_STAGE_METRIC_K:
        if (!ctx->has_K) { risp_set_error(ctx, "risp_get_stage: no K metric"); return RISP_EINVAL; }
        RISP_CUDA_TRY(cudaMemcpy(out, ctx->d_MK, (size_t)ctx->nauxK_global * ctx->nauxK_global * 8, cudaMemcpyDeviceToHost));
        return RISP_OK;
    case RISP_STAGE_U: {
        // rebuilt from the e0-space U-bar that the last matvec left in place (pass 2 output)
        if (need_mv() || !sel || sel[0] < 0 || sel[0] >= m) return RISP_EINVAL;
        double *tmp = nullptr;
        const size_t n = (size_t)ctx->nao * ctx->ldao;
        RISP_CUDA_TRY(scr.alloc(tmp, n));
        RISP_CUDA_TRY(cudaMemset(tmp, 0, n * 8));
        for (int c = 0; c < 6; ++c)
            RISP_CUDA_TRY(risp_e0_to_U(ctx->cls[c], 0, ctx->cls[c].npairs, 1, (int)sel[0], 0, ctx->ldao, (long long)n, 0, ctx->w_dbar, tmp, 0));
        RISP_CUDA_TRY(cudaMemcpy2D(out, (size_t)ctx->nao * 8, tmp, (size_t)ctx->ldao * 8, (size_t)ctx->nao * 8, ctx->nao, cudaMemcpyDeviceToHost));
        return RISP_OK;
    }
    default:
        risp_set_error(ctx, "risp_get_stage: unknown stage");
        return RISP_EINVAL;
    }
}

// ---- debug exports (include/risp_debug.h; not part of the method)
// The DMMA GEMM on caller-provided DEVICE buffers: GEMM unit tests and the FP64 tensor-rate yardstick of bench.py.
// C = alpha op(A) op(B) + beta C, see GemmDesc in common.cuh.  variant 1: TMA kernel when the operands allow it, 0: cp.async kernel.
// c_rpg > 0: row r of C lives at (r / c_rpg) * c_gstride + (r % c_rpg) * ldc (the split-row epilogue of Eq. 22).
extern "C" int risp_debug_dgemm(int M, int N, int K, const double *A, long long lda, int a_kc, const double *B, long long ldb, int b_kc, double *C,
                                long long ldc, double alpha, double beta, int nbatch, long long sA, long long sB, long long sC, int variant,
                                int c_rpg, long long c_gstride, void *stream)
{
    GemmDesc d = gemm_desc(M, N, K, A, lda, a_kc != 0, B, ldb, b_kc != 0, C, ldc, alpha, beta);
    d.nb1 = nbatch; d.sA1 = sA; d.sB1 = sB; d.sC1 = sC;
    d.variant = variant; d.c_rpg = c_rpg; d.c_gstride = c_gstride;
    return risp_dgemm(d, (cudaStream_t)stream) == cudaSuccess ? RISP_OK : RISP_ECUDA;
}

extern "C" int risp_set_precision(risp_ctx *ctx, int32_t mode)
{
    if (!ctx) return RISP_EINVAL;
    if (mode != RISP_PRECISION_FP64 && mode != RISP_PRECISION_FP32_K && mode != RISP_PRECISION_FP32_JK) { risp_set_error(ctx, "risp_set_precision: unknown mode"); return RISP_EINVAL; }
    if (mode != RISP_PRECISION_FP64) {
        cudaDeviceProp prop;
        RISP_CUDA_TRY(cudaGetDeviceProperties(&prop, ctx->device));
        if (prop.major != 10) { risp_set_error(ctx, "risp_set_precision: the single-precision mode needs the tcgen05 tensor cores (sm_100)"); return RISP_EINVAL; }
    }
    if (mode == RISP_PRECISION_FP32_JK && ctx->precision != mode) {
        // the work space of this mode holds the bf16 planes of the J transforms too: plan it again at the next sigma-build
        RISP_CUDA_TRY(cudaSetDevice(ctx->device));
        RISP_CUDA_TRY(cudaDeviceSynchronize());
        risp_free_workspace(ctx);
    }
    ctx->precision = mode;
    return RISP_OK;
}

extern "C" int risp_debug_set_tc_plan(risp_ctx *ctx, int32_t eq22_shape, int32_t eq22_seg, int32_t eq23_shape, int32_t eq23_seg)
{
    if (!ctx || eq22_shape < -1 || eq22_shape > 2 || eq23_shape < -1 || eq23_shape > 2 || eq22_seg < 0 || eq23_seg < 0) return RISP_EINVAL;
    ctx->tc_shape22 = eq22_shape; ctx->tc_shape23 = eq23_shape; ctx->tc_seg22 = eq22_seg; ctx->tc_seg23 = eq23_seg;
    return RISP_OK;
}
