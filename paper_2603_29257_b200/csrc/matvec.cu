// matvec.cu -- risp_matvec: sigma = A X for a batch of m trial vectors (Eq. 10).
//
//   J (Eq. 11-17):  Y = X C_vir^T ; D = C_occ Y (Eq. 12) ; D -> e0 space ; pass 1 (Eq. 14) ;
//       R~ = L^-T L^-1 R (Eq. 15) ; pass 2 (Eq. 16) ; e0 space -> U ; Z = C_occ^T U ; J = Z C_vir (Eq. 17)
//   K (Eq. 18-23):  X' = X[window] ; per aux chunk  M^P = X' T_ab^P (Eq. 22) ; K' += T_ij^P M^P (Eq. 23)
//   sigma = (eps_a - eps_i) X + 2 J - K'  (K' only inside the window)
#include "ctx.h"

static void free_ws(risp_ctx *ctx)
{
    double **bufs[] = {&ctx->w_Y, &ctx->w_D, &ctx->w_dbar, &ctx->w_Rpart, &ctx->w_R, &ctx->w_Rt, &ctx->w_Rtmp, &ctx->w_J,
                       &ctx->w_Xk, &ctx->w_Kk, &ctx->w_M, &ctx->w_Xin, &ctx->w_Sout};
    for (auto b : bufs) { if (*b) cudaFree(*b); *b = nullptr; }
    ctx->m_cap = 0; ctx->w_bytes = 0;
}

int risp_ensure_workspace(risp_ctx *ctx, int m)
{
    if (m <= ctx->m_cap) return RISP_OK;
    free_ws(ctx);
    const size_t nao = ctx->nao, nocc = ctx->nocc, nvir = ctx->nvir, no = ctx->noccK, nv = ctx->nvirK;
    size_t fixed = ((size_t)m * nocc * nao + (size_t)m * nao * nao + (size_t)ctx->e_rows * RISP_MS +
                    (size_t)ctx->total_chunks * ctx->ncenJ_pad * 4 * RISP_MS + 3 * (size_t)ctx->nauxJ * RISP_MS + (size_t)m * nocc * nvir +
                    2 * (size_t)m * no * nv) * sizeof(double);
    // aux chunk of the K contraction: M[m][Pc][no][nv] within what is left of the budget (at most 4 GiB)
    int pc = 1;
    if (ctx->has_K) {
        size_t per_fn = (size_t)m * no * nv * sizeof(double);
        size_t avail = ctx->hbm_budget > ctx->setup_bytes + fixed ? ctx->hbm_budget - ctx->setup_bytes - fixed : 0;
        avail = std::min<size_t>(avail, (size_t)4 << 30);
        pc = (int)std::max<size_t>(1, std::min<size_t>((size_t)ctx->nauxK, avail / std::max<size_t>(per_fn, 1)));
    }
    ctx->aux_chunk = pc;
    auto A = [&](double *&p, size_t n) -> int {
        if (n == 0) { p = nullptr; return RISP_OK; }
        RISP_CUDA_TRY(cudaMalloc((void **)&p, n * sizeof(double)));
        ctx->w_bytes += n * sizeof(double);
        return RISP_OK;
    };
    int rc;
    if ((rc = A(ctx->w_Y, (size_t)m * nocc * nao))) return rc;
    if ((rc = A(ctx->w_D, (size_t)m * nao * nao))) return rc;
    if ((rc = A(ctx->w_dbar, (size_t)ctx->e_rows * RISP_MS))) return rc;
    if ((rc = A(ctx->w_Rpart, (size_t)ctx->total_chunks * ctx->ncenJ_pad * 4 * RISP_MS))) return rc;
    if ((rc = A(ctx->w_R, (size_t)ctx->nauxJ * RISP_MS))) return rc;
    if ((rc = A(ctx->w_Rt, (size_t)ctx->nauxJ * RISP_MS))) return rc;
    if ((rc = A(ctx->w_Rtmp, (size_t)ctx->nauxJ * RISP_MS))) return rc;
    if ((rc = A(ctx->w_J, (size_t)m * nocc * nvir))) return rc;
    if (ctx->has_K) {
        if ((rc = A(ctx->w_Xk, (size_t)m * no * nv))) return rc;
        if ((rc = A(ctx->w_Kk, (size_t)m * no * nv))) return rc;
        if ((rc = A(ctx->w_M, (size_t)m * pc * no * nv))) return rc;
    }
    RISP_CUDA_TRY(cudaMemset(ctx->w_Rpart, 0, (size_t)ctx->total_chunks * ctx->ncenJ_pad * 4 * RISP_MS * sizeof(double)));
    ctx->m_cap = m;
    return RISP_OK;
}

int risp_matvec_impl(risp_ctx *ctx, int m, const double *X, double *sigma, cudaStream_t st)
{
    const int nao = ctx->nao, nocc = ctx->nocc, nvir = ctx->nvir, nmo = ctx->nmo, nJ = ctx->nauxJ;
    const int no = ctx->noccK, nv = ctx->nvirK, nK = ctx->nauxK;
    int launches = 0;
    cudaEvent_t *ev = ctx->ev;
    RISP_CUDA_TRY(cudaEventRecord(ev[0], st));
    // ---------------- J: AO transition density (Eq. 12)
    {
        GemmDesc d = gemm_desc(m * nocc, nao, nvir, X, nvir, true, ctx->d_C + nocc, nmo, true, ctx->w_Y, nao);
        RISP_CUDA_TRY(risp_dgemm(d, st)); ++launches;
        GemmDesc e = gemm_desc(nao, nao, nocc, ctx->d_C, nmo, true, ctx->w_Y, nao, false, ctx->w_D, nao);
        e.nb1 = m; e.sB1 = (long long)nocc * nao; e.sC1 = (long long)nao * nao;
        RISP_CUDA_TRY(risp_dgemm(e, st)); ++launches;
        for (int c = 0; c < 6; ++c) if (ctx->cls[c].npairs) { RISP_CUDA_TRY(risp_dens_to_e0(ctx->cls[c], m, nao, ctx->w_D, ctx->w_dbar, st)); ++launches; }
    }
    RISP_CUDA_TRY(cudaEventRecord(ev[1], st));
    // ---------------- pass 1: R_mQ (Eq. 14)
    for (int c = 0; c < 6; ++c)
        if (ctx->cls[c].npairs) {
            RISP_CUDA_TRY(risp_j_pass1(ctx->cls[c], ctx->d_prims, ctx->d_cenJ, ctx->ncenJ, ctx->ncenJ_pad, ctx->d_boys, ctx->w_dbar, ctx->w_Rpart, st));
            ++launches;
        }
    RISP_CUDA_TRY(risp_j_reduce_R(ctx->w_Rpart, ctx->total_chunks, ctx->d_cenJ, ctx->ncenJ, ctx->ncenJ_pad, ctx->w_R, st)); ++launches;
    RISP_CUDA_TRY(cudaEventRecord(ev[2], st));
    // ---------------- R~ = (P|Q)^-1 R = L^-T (L^-1 R)  (Eq. 15)
    {
        GemmDesc d = gemm_desc(nJ, RISP_MS, nJ, ctx->d_LinvJ, nJ, true, ctx->w_R, RISP_MS, false, ctx->w_Rtmp, RISP_MS);
        RISP_CUDA_TRY(risp_dgemm(d, st)); ++launches;
        GemmDesc e = gemm_desc(nJ, RISP_MS, nJ, ctx->d_LinvJ, nJ, false, ctx->w_Rtmp, RISP_MS, false, ctx->w_Rt, RISP_MS);
        RISP_CUDA_TRY(risp_dgemm(e, st)); ++launches;
    }
    RISP_CUDA_TRY(cudaEventRecord(ev[3], st));
    // ---------------- pass 2: U (Eq. 16), into the e0 buffer
    for (int c = 0; c < 6; ++c)
        if (ctx->cls[c].npairs) {
            RISP_CUDA_TRY(risp_j_pass2(ctx->cls[c], ctx->d_prims, ctx->d_cenJ, ctx->ncenJ, ctx->d_boys, ctx->w_Rt, ctx->w_dbar, st));
            ++launches;
        }
    RISP_CUDA_TRY(cudaEventRecord(ev[4], st));
    // ---------------- back-transform (Eq. 17)
    {
        RISP_CUDA_TRY(cudaMemsetAsync(ctx->w_D, 0, (size_t)m * nao * nao * sizeof(double), st));
        for (int c = 0; c < 6; ++c) if (ctx->cls[c].npairs) { RISP_CUDA_TRY(risp_e0_to_U(ctx->cls[c], m, nao, ctx->w_dbar, ctx->w_D, st)); ++launches; }
        GemmDesc d = gemm_desc(nocc, nao, nao, ctx->d_C, nmo, false, ctx->w_D, nao, false, ctx->w_Y, nao);
        d.nb1 = m; d.sB1 = (long long)nao * nao; d.sC1 = (long long)nocc * nao;
        RISP_CUDA_TRY(risp_dgemm(d, st)); ++launches;
        GemmDesc e = gemm_desc(m * nocc, nvir, nao, ctx->w_Y, nao, true, ctx->d_C + nocc, nmo, false, ctx->w_J, nvir);
        RISP_CUDA_TRY(risp_dgemm(e, st)); ++launches;
    }
    RISP_CUDA_TRY(cudaEventRecord(ev[5], st));
    // ---------------- K (Eq. 22-23)
    if (ctx->has_K) {
        RISP_CUDA_TRY(risp_gather_window(X, ctx->w_Xk, m, nocc, nvir, ctx->occK0, no, ctx->virK0, nv, st)); ++launches;
        RISP_CUDA_TRY(cudaEventRecord(ev[6], st));
        const int pc = ctx->aux_chunk;
        for (int p0 = 0; p0 < nK; p0 += pc) {
            int np = std::min(pc, nK - p0);
            // M[mi][P][j][a] = sum_b X'[mi][j][b] T_ab^P[a][b]; rows (mi,j) of one P are split by mi
            GemmDesc d = gemm_desc(m * no, nv, nv, ctx->w_Xk, nv, true, ctx->d_Tab + (long long)p0 * nv * nv, nv, true, ctx->w_M, nv);
            d.nb1 = np; d.sB1 = (long long)nv * nv; d.sC1 = (long long)no * nv;
            d.c_rpg = no; d.c_gstride = (long long)np * no * nv;
            RISP_CUDA_TRY(risp_dgemm(d, st)); ++launches;
            if (p0 == 0) RISP_CUDA_TRY(cudaEventRecord(ev[9], st));
            // K'[mi][i][a] (+)= sum_{(P,j)} T_ij[i][(P,j)] M[mi][(P,j)][a]
            GemmDesc e = gemm_desc(no, nv, np * no, ctx->d_Tij + (long long)p0 * no, (long long)nK * no, true, ctx->w_M, nv, false, ctx->w_Kk, nv,
                                   1.0, p0 == 0 ? 0.0 : 1.0);
            e.nb1 = m; e.sB1 = (long long)np * no * nv; e.sC1 = (long long)no * nv;
            RISP_CUDA_TRY(risp_dgemm(e, st)); ++launches;
            if (p0 == 0) { RISP_CUDA_TRY(cudaEventRecord(ev[10], st)); ctx->tim.first_chunk_naux = np; }
        }
    } else {
        RISP_CUDA_TRY(cudaEventRecord(ev[6], st));
    }
    RISP_CUDA_TRY(cudaEventRecord(ev[7], st));
    // ---------------- sigma (Eq. 10)
    RISP_CUDA_TRY(risp_assemble_sigma(X, ctx->w_J, ctx->w_Kk, ctx->d_eps, sigma, m, nocc, nvir, ctx->occK0, no, ctx->virK0, nv, ctx->has_K ? 1 : 0, st));
    ++launches;
    RISP_CUDA_TRY(cudaEventRecord(ev[8], st));
    ctx->tim.kernel_launches = launches;
    ctx->last_m = m;
    return RISP_OK;
}

extern "C" int risp_matvec(risp_ctx *ctx, int32_t m, const double *X_dev, double *sigma_dev, void *cuda_stream)
{
    if (!ctx) return RISP_EINVAL;
    if (m <= 0 || m > RISP_MS || !X_dev || !sigma_dev) { risp_set_error(ctx, "risp_matvec: need 1 <= m <= 32 and non-NULL device pointers"); return RISP_EINVAL; }
    size_t bytes = (size_t)m * ctx->nocc * ctx->nvir * sizeof(double);
    const char *x = (const char *)X_dev, *s = (const char *)sigma_dev;
    if (x < s + bytes && s < x + bytes) { risp_set_error(ctx, "risp_matvec: X and sigma overlap"); return RISP_EINVAL; }
    RISP_CUDA_TRY(cudaSetDevice(ctx->device));
    int rc = risp_ensure_workspace(ctx, m);
    if (rc) return rc;
    return risp_matvec_impl(ctx, m, X_dev, sigma_dev, (cudaStream_t)cuda_stream);
}

extern "C" int risp_matvec_host(risp_ctx *ctx, int32_t m, const double *X_host, double *sigma_host)
{
    if (!ctx) return RISP_EINVAL;
    if (m <= 0 || m > RISP_MS || !X_host || !sigma_host) { risp_set_error(ctx, "risp_matvec_host: need 1 <= m <= 32 and non-NULL host pointers"); return RISP_EINVAL; }
    RISP_CUDA_TRY(cudaSetDevice(ctx->device));
    int rc = risp_ensure_workspace(ctx, m);
    if (rc) return rc;
    size_t n = (size_t)ctx->m_cap * ctx->nocc * ctx->nvir, bytes = (size_t)m * ctx->nocc * ctx->nvir * sizeof(double);
    if (!ctx->w_Xin) {
        RISP_CUDA_TRY(cudaMalloc((void **)&ctx->w_Xin, n * sizeof(double)));
        RISP_CUDA_TRY(cudaMalloc((void **)&ctx->w_Sout, n * sizeof(double)));
        ctx->w_bytes += 2 * n * sizeof(double);
    }
    RISP_CUDA_TRY(cudaMemcpyAsync(ctx->w_Xin, X_host, bytes, cudaMemcpyHostToDevice, 0));
    rc = risp_matvec_impl(ctx, m, ctx->w_Xin, ctx->w_Sout, 0);
    if (rc) return rc;
    RISP_CUDA_TRY(cudaMemcpyAsync(sigma_host, ctx->w_Sout, bytes, cudaMemcpyDeviceToHost, 0));
    RISP_CUDA_TRY(cudaStreamSynchronize(0));
    return RISP_OK;
}
