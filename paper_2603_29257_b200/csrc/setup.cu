// setup.cu -- risp_setup: everything of the sigma-build that does not depend on the trial vectors.
//
//   a0  screened shell-pair list, primitive-pair data                     ("screened non-zero AO pairs")
//   a1  metrics (P|Q)_J (Coulomb, s+p) and (P|J^|Q)_K (Eq. 26), Cholesky
//   a2  exchange-space window
//   a3  T_ij^P = sum_Q (ij|Q)(Q|P)^-1 (Eq. 20), T_ab^P = (ab|P) (Eq. 21, reading G3)
#include "ctx.h"
#include <algorithm>
#include <cmath>

using namespace risp_eri;

void risp_set_error(risp_ctx *ctx, const std::string &msg)
{
    if (ctx) ctx->err = msg;
}

namespace {

const double PI = 3.14159265358979323846;
const double HARTREE_EV = 27.211386245988;

double gamma_half(int l)   // Gamma(l + 3/2)
{
    double g = std::sqrt(PI) / 2;
    for (int k = 0; k < l; ++k) g *= (k + 1.5);
    return g;
}
double radial_norm(double a, int l) { return std::sqrt(2.0 * std::pow(2.0 * a, l + 1.5) / gamma_half(l)); }

// Boys table F_k(i*dx): ascending series at the top order (positive terms), then downward recursion, in long double
std::vector<double> make_boys_table()
{
    std::vector<double> tab((size_t)BOYS_NX * BOYS_NK);
    const int K = BOYS_NK - 1;
    for (int i = 0; i < BOYS_NX; ++i) {
        long double x = (long double)i * (long double)BOYS_DX;
        long double term = 1.0L / (2 * K + 1), sum = term;
        for (int j = 1; j < 600; ++j) {
            term *= 2.0L * x / (2 * K + 2 * j + 1);
            sum += term;
            if (term < 1e-21L * sum) break;
        }
        long double ex = expl(-x), f = ex * sum;
        tab[(size_t)i * BOYS_NK + K] = (double)f;
        for (int k = K; k > 0; --k) {
            f = (2.0L * x * f + ex) / (2 * k - 1);
            tab[(size_t)i * BOYS_NK + k - 1] = (double)f;
        }
    }
    return tab;
}

template <class T>
int upload(risp_ctx *ctx, T *&dst, const T *src, size_t n)
{
    dst = nullptr;
    if (n == 0) return RISP_OK;
    RISP_CUDA_TRY(cudaMalloc((void **)&dst, n * sizeof(T)));
    RISP_CUDA_TRY(cudaMemcpy(dst, src, n * sizeof(T), cudaMemcpyHostToDevice));
    ctx->setup_bytes += n * sizeof(T);
    return RISP_OK;
}
template <class T>
int dalloc(risp_ctx *ctx, T *&dst, size_t n)
{
    dst = nullptr;
    if (n == 0) return RISP_OK;
    RISP_CUDA_TRY(cudaMalloc((void **)&dst, n * sizeof(T)));
    ctx->setup_bytes += n * sizeof(T);
    return RISP_OK;
}

int class_index(int la, int lb) { return la * (la + 1) / 2 + lb; }   // (0,0)=0 (1,0)=1 (1,1)=2 (2,0)=3 (2,1)=4 (2,2)=5

// group aux shells into centres (one exponent, an s and/or a p shell on one atom)
void build_centres(const risp_ctx *ctx, const std::vector<int> &fn_of_shell, std::vector<AuxCentre> &cen)
{
    cen.clear();
    int naux = (int)ctx->h_aux_l.size();
    std::vector<char> used(naux, 0);
    for (int s = 0; s < naux; ++s) {
        if (used[s] || fn_of_shell[s] < 0) continue;
        AuxCentre c;
        int at = ctx->h_aux_atom[s];
        c.x = ctx->h_xyz[3 * at]; c.y = ctx->h_xyz[3 * at + 1]; c.z = ctx->h_xyz[3 * at + 2];
        c.g = ctx->h_aux_exp[s];
        c.ns = std::pow(2.0 * c.g / PI, 0.75);
        c.np = c.ns * 2.0 * std::sqrt(c.g);
        c.qs = c.qp = -1;
        for (int t = s; t < naux; ++t) {
            if (used[t] || fn_of_shell[t] < 0 || ctx->h_aux_atom[t] != at || ctx->h_aux_exp[t] != c.g) continue;
            if (ctx->h_aux_l[t] == 0 && c.qs < 0) { c.qs = fn_of_shell[t]; used[t] = 1; }
            else if (ctx->h_aux_l[t] == 1 && c.qp < 0) { c.qp = fn_of_shell[t]; used[t] = 1; }
        }
        cen.push_back(c);
    }
}

// metric (P|op|Q) over one aux set, using the 3c engine with each aux function as a one-primitive "AO shell"
// paired with the constant function (exponent 0): (P 1|Q) = (P|Q).
int build_metric(risp_ctx *ctx, const std::vector<int> &fn_of_shell, int nfn, const AuxCentre *d_cen, int ncen, OpParams op, bool erf_op,
                 double *d_M)
{
    bool hasp = false;
    for (size_t s = 0; s < fn_of_shell.size(); ++s) if (fn_of_shell[s] >= 0 && ctx->h_aux_l[s] == 1) hasp = true;
    for (int l = 0; l <= 1; ++l) {
        std::vector<ShellPair> sp;
        std::vector<PrimPair> pp;
        for (size_t s = 0; s < fn_of_shell.size(); ++s) {
            if (fn_of_shell[s] < 0 || ctx->h_aux_l[s] != l) continue;
            int at = ctx->h_aux_atom[s];
            double g = ctx->h_aux_exp[s];
            ShellPair r;
            r.Ax = ctx->h_xyz[3 * at]; r.Ay = ctx->h_xyz[3 * at + 1]; r.Az = ctx->h_xyz[3 * at + 2];
            r.ABx = r.ABy = r.ABz = 0.0;
            r.aoA = fn_of_shell[s]; r.aoB = 0; r.ppoff = (int)pp.size(); r.npp = 1; r.shA = 0; r.shB = 1; r.pad0 = r.pad1 = 0;
            PrimPair p;
            p.p = g; p.Px = r.Ax; p.Py = r.Ay; p.Pz = r.Az;
            p.cc = radial_norm(g, l) * std::sqrt(4.0 * PI) * 2.0 * std::pow(PI, 2.5) / g;
            sp.push_back(r); pp.push_back(p);
        }
        if (sp.empty()) continue;
        ShellPair *d_sp = nullptr; PrimPair *d_pp = nullptr;
        RISP_CUDA_TRY(cudaMalloc((void **)&d_sp, sp.size() * sizeof(ShellPair)));
        RISP_CUDA_TRY(cudaMalloc((void **)&d_pp, pp.size() * sizeof(PrimPair)));
        RISP_CUDA_TRY(cudaMemcpy(d_sp, sp.data(), sp.size() * sizeof(ShellPair), cudaMemcpyHostToDevice));
        RISP_CUDA_TRY(cudaMemcpy(d_pp, pp.data(), pp.size() * sizeof(PrimPair), cudaMemcpyHostToDevice));
        // out[q*nfn + (aoA + i)*1 + 0]
        RISP_CUDA_TRY(risp_eri_fill(l, 0, hasp, erf_op, d_sp, (int)sp.size(), d_pp, d_cen, ncen, op, ctx->d_boys, d_M, nfn, 1, 0, 0));
        RISP_CUDA_TRY(cudaDeviceSynchronize());
        cudaFree(d_sp); cudaFree(d_pp);
    }
    return RISP_OK;
}

}  // namespace

// Build the shell-pair record and its primitive pairs for (shA, shB), l(shA) >= l(shB).  Primitive pairs whose
// magnitude estimate is below prim_tol are dropped.  Returns the pair's magnitude estimate through sp.pad0/pad1 unused;
// the estimate is returned as the function value scaled: < 0 never.
static double pair_estimate_and_build(const risp_ctx *ctx, int shA, int shB, ShellPair &sp, std::vector<PrimPair> &pp, double prim_tol,
                                      double vmax)
{
    int atA = ctx->h_shl_atom[shA], atB = ctx->h_shl_atom[shB];
    int la = ctx->h_shl_l[shA], lb = ctx->h_shl_l[shB];
    const double *A = &ctx->h_xyz[3 * atA], *B = &ctx->h_xyz[3 * atB];
    sp.Ax = A[0]; sp.Ay = A[1]; sp.Az = A[2];
    sp.ABx = A[0] - B[0]; sp.ABy = A[1] - B[1]; sp.ABz = A[2] - B[2];
    sp.aoA = ctx->h_shl_ao[shA]; sp.aoB = ctx->h_shl_ao[shB];
    sp.shA = shA; sp.shB = shB; sp.pad0 = sp.pad1 = 0;
    sp.ppoff = (int)pp.size();
    double R2 = sp.ABx * sp.ABx + sp.ABy * sp.ABy + sp.ABz * sp.ABz;
    double total = 0.0;
    for (int ka = 0; ka < ctx->h_shl_nprim[shA]; ++ka)
        for (int kb = 0; kb < ctx->h_shl_nprim[shB]; ++kb) {
            double a = ctx->h_prim_exp[ctx->h_shl_poff[shA] + ka], b = ctx->h_prim_exp[ctx->h_shl_poff[shB] + kb];
            double da = ctx->h_prim_d[ctx->h_shl_poff[shA] + ka], db = ctx->h_prim_d[ctx->h_shl_poff[shB] + kb];
            double p = a + b, mu = a * b / p;
            double kab = std::exp(-mu * R2);
            // magnitude estimate of max_P |(ab|P)|: integral of |chi_a chi_b| times the largest aux potential
            double s = 2.0 / std::sqrt(p), rPA = b / p * std::sqrt(R2), rPB = a / p * std::sqrt(R2);
            double est = std::fabs(da * db) * kab * std::pow(PI / p, 1.5) * std::pow(s + rPA, la) * std::pow(s + rPB, lb) * vmax;
            total += est;
            if (est < prim_tol) continue;
            PrimPair q;
            q.p = p;
            q.Px = (a * A[0] + b * B[0]) / p; q.Py = (a * A[1] + b * B[1]) / p; q.Pz = (a * A[2] + b * B[2]) / p;
            q.cc = da * db * kab * 2.0 * std::pow(PI, 2.5) / p;
            pp.push_back(q);
        }
    sp.npp = (int)pp.size() - sp.ppoff;
    return total;
}

int risp_build_pair(risp_ctx *ctx, int shA, int shB, ShellPair &sp, std::vector<PrimPair> &pp, double prim_tol)
{
    pair_estimate_and_build(ctx, shA, shB, sp, pp, prim_tol, 1.0);
    return RISP_OK;
}

extern "C" int risp_setup(const risp_system *sys, const risp_options *opt_in, risp_ctx **out)
{
    if (!out) return RISP_EINVAL;
    *out = nullptr;
    if (!sys) return RISP_EINVAL;
    risp_ctx *ctx = new risp_ctx();
    *out = ctx;   // returned even on failure so that risp_last_error() can be read; caller destroys it
    for (int c = 0; c < 6; ++c) { ctx->cls[c].npairs = 0; ctx->cls[c].d_pairs = nullptr; }
    risp_options opt;
    std::memset(&opt, 0, sizeof(opt));
    if (opt_in) opt = *opt_in;
    // ---------------------------------------------------------------- validation
    auto bad = [&](const char *m) { risp_set_error(ctx, std::string("risp_setup: ") + m); return RISP_EINVAL; };
    if (sys->natm <= 0 || sys->nshl <= 0 || sys->naux < 0 || sys->nao <= 0 || sys->nocc <= 0 || sys->nvir <= 0) return bad("non-positive size");
    if (!sys->xyz_bohr || !sys->shl_atom || !sys->shl_l || !sys->shl_nprim || !sys->shl_poff || !sys->prim_exp || !sys->prim_coef || !sys->C ||
        !sys->eps || (sys->naux > 0 && (!sys->aux_atom || !sys->aux_l || !sys->aux_exp || !sys->aux_in_K)))
        return bad("NULL array");
    if (sys->nocc + sys->nvir > sys->nao) return bad("nocc + nvir > nao");
    int nao_chk = 0, nprim_tot = 0;
    for (int s = 0; s < sys->nshl; ++s) {
        if (sys->shl_l[s] < 0 || sys->shl_l[s] > 2) return bad("AO shell l outside 0..2");
        if (sys->shl_nprim[s] < 1) return bad("AO shell without primitives");
        if (sys->shl_atom[s] < 0 || sys->shl_atom[s] >= sys->natm) return bad("shl_atom out of range");
        nao_chk += 2 * sys->shl_l[s] + 1;
        nprim_tot = std::max(nprim_tot, sys->shl_poff[s] + sys->shl_nprim[s]);
    }
    if (nao_chk != sys->nao) return bad("nao != sum(2l+1)");
    for (int s = 0; s < sys->naux; ++s) {
        if (sys->aux_l[s] < 0 || sys->aux_l[s] > 1) return bad("aux shell l outside 0..1");
        if (sys->aux_atom[s] < 0 || sys->aux_atom[s] >= sys->natm) return bad("aux_atom out of range");
        if (!(sys->aux_exp[s] > 0)) return bad("aux exponent not positive");
    }
    for (int k = 0; k < nprim_tot; ++k) if (!(sys->prim_exp[k] > 0)) return bad("primitive exponent not positive");
    if (sys->omega < 0) return bad("omega < 0");

    ctx->device = opt.device;
    RISP_CUDA_TRY(cudaSetDevice(opt.device));
    ctx->natm = sys->natm; ctx->nshl = sys->nshl; ctx->nao = sys->nao; ctx->nocc = sys->nocc; ctx->nvir = sys->nvir;
    ctx->nmo = sys->nocc + sys->nvir;
    ctx->alpha = sys->alpha; ctx->beta = sys->beta; ctx->omega = sys->omega;
    ctx->h_xyz.assign(sys->xyz_bohr, sys->xyz_bohr + 3 * sys->natm);
    ctx->h_shl_atom.assign(sys->shl_atom, sys->shl_atom + sys->nshl);
    ctx->h_shl_l.assign(sys->shl_l, sys->shl_l + sys->nshl);
    ctx->h_shl_nprim.assign(sys->shl_nprim, sys->shl_nprim + sys->nshl);
    ctx->h_shl_poff.assign(sys->shl_poff, sys->shl_poff + sys->nshl);
    ctx->h_prim_exp.assign(sys->prim_exp, sys->prim_exp + nprim_tot);
    ctx->h_prim_d.assign(nprim_tot, 0.0);
    ctx->h_shl_ao.resize(sys->nshl);
    ctx->h_eps.assign(sys->eps, sys->eps + ctx->nmo);
    {
        int off = 0;
        for (int s = 0; s < sys->nshl; ++s) {
            ctx->h_shl_ao[s] = off; off += 2 * sys->shl_l[s] + 1;
            int l = sys->shl_l[s], np = sys->shl_nprim[s], po = sys->shl_poff[s];
            double nrm = 0.0;
            for (int k = 0; k < np; ++k)
                for (int q = 0; q < np; ++q)
                    nrm += sys->prim_coef[po + k] * sys->prim_coef[po + q] * radial_norm(sys->prim_exp[po + k], l) *
                           radial_norm(sys->prim_exp[po + q], l) * gamma_half(l) / (2.0 * std::pow(sys->prim_exp[po + k] + sys->prim_exp[po + q], l + 1.5));
            if (!(nrm > 0)) return bad("contracted shell has zero norm");
            for (int k = 0; k < np; ++k) ctx->h_prim_d[po + k] = sys->prim_coef[po + k] * radial_norm(sys->prim_exp[po + k], l) / std::sqrt(nrm);
        }
    }
    ctx->h_aux_atom.assign(sys->aux_atom, sys->aux_atom + sys->naux);
    ctx->h_aux_l.assign(sys->aux_l, sys->aux_l + sys->naux);
    ctx->h_aux_exp.assign(sys->aux_exp, sys->aux_exp + sys->naux);
    ctx->h_aux_fn.assign(sys->naux, -1); ctx->h_aux_fnK.assign(sys->naux, -1);
    for (int s = 0; s < sys->naux; ++s) {
        ctx->h_aux_fn[s] = ctx->nauxJ; ctx->nauxJ += 2 * sys->aux_l[s] + 1;
        if (sys->aux_in_K[s]) { ctx->h_aux_fnK[s] = ctx->nauxK; ctx->nauxK += 2 * sys->aux_l[s] + 1; }
    }
    if (ctx->nauxJ == 0) return bad("empty auxiliary basis");

    // ---------------------------------------------------------------- a2: window (reading G6: absolute energies)
    {
        double cut = sys->cutoff_ev;
        int o0 = 0, o1 = ctx->nocc, v0 = 0, v1 = ctx->nvir;
        if (cut > 0 && std::isfinite(cut)) {
            while (o0 < ctx->nocc && !(ctx->h_eps[o0] * HARTREE_EV > -cut)) ++o0;
            o1 = o0;
            while (o1 < ctx->nocc && ctx->h_eps[o1] * HARTREE_EV > -cut) ++o1;
            while (v0 < ctx->nvir && !(ctx->h_eps[ctx->nocc + v0] * HARTREE_EV < cut)) ++v0;
            v1 = v0;
            while (v1 < ctx->nvir && ctx->h_eps[ctx->nocc + v1] * HARTREE_EV < cut) ++v1;
            for (int i = o1; i < ctx->nocc; ++i) if (ctx->h_eps[i] * HARTREE_EV > -cut) return bad("eps not ascending: window is not contiguous");
            for (int a = v1; a < ctx->nvir; ++a) if (ctx->h_eps[ctx->nocc + a] * HARTREE_EV < cut) return bad("eps not ascending: window is not contiguous");
        }
        ctx->occK0 = o0; ctx->noccK = o1 - o0; ctx->virK0 = v0; ctx->nvirK = v1 - v0;
        ctx->has_K = (sys->alpha != 0.0 || sys->beta != 0.0) && ctx->nauxK > 0 && ctx->noccK > 0 && ctx->nvirK > 0;
    }

    // ---------------------------------------------------------------- device constants
    {
        std::vector<double> tab = make_boys_table();
        int rc;
        if ((rc = upload(ctx, ctx->d_boys, tab.data(), tab.size()))) return rc;
        if ((rc = upload(ctx, ctx->d_C, sys->C, (size_t)ctx->nao * ctx->nmo))) return rc;
        if ((rc = upload(ctx, ctx->d_eps, sys->eps, (size_t)ctx->nmo))) return rc;
    }
    std::vector<AuxCentre> cenJ, cenK;
    build_centres(ctx, ctx->h_aux_fn, cenJ);
    build_centres(ctx, ctx->h_aux_fnK, cenK);
    ctx->ncenJ = (int)cenJ.size(); ctx->ncenK = (int)cenK.size();
    ctx->ncenJ_pad = (ctx->ncenJ + 7) / 8 * 8;
    { int rc; if ((rc = upload(ctx, ctx->d_cenJ, cenJ.data(), cenJ.size()))) return rc; if ((rc = upload(ctx, ctx->d_cenK, cenK.data(), cenK.size()))) return rc; }

    // ---------------------------------------------------------------- a0: screened shell-pair list
    {
        double tau = opt.screen_tol == 0.0 ? 1e-13 : opt.screen_tol;
        double gmin = 1e300;
        for (int s = 0; s < sys->naux; ++s) gmin = std::min(gmin, sys->aux_exp[s]);
        double vmax = 2.0 * 4.48 * std::pow(gmin, -0.25);    // ~ 2 x the peak potential of a unit-normalised s aux Gaussian
        std::vector<ShellPair> pairs[6];
        std::vector<PrimPair> prims;
        ctx->n_shell_pairs = (long long)sys->nshl * (sys->nshl + 1) / 2;
        for (int sa = 0; sa < sys->nshl; ++sa)
            for (int sb = 0; sb <= sa; ++sb) {
                int A = sa, B = sb;
                if (sys->shl_l[A] < sys->shl_l[B]) std::swap(A, B);
                ShellPair sp;
                size_t mark = prims.size();
                double est = pair_estimate_and_build(ctx, A, B, sp, prims, tau < 0 ? -1.0 : tau * 1e-3, vmax);
                if ((tau >= 0 && est < tau) || sp.npp == 0) { prims.resize(mark); continue; }
                pairs[class_index(sys->shl_l[A], sys->shl_l[B])].push_back(sp);
                ctx->h_kept_pairs.push_back(A); ctx->h_kept_pairs.push_back(B);
                ctx->n_ao_pairs_kept += (A == B) ? (long long)(2 * sys->shl_l[A] + 1) * (2 * sys->shl_l[A] + 2) / 2
                                                 : (long long)(2 * sys->shl_l[A] + 1) * (2 * sys->shl_l[B] + 1);
            }
        long long e_off = 0, total_pairs = 0;
        for (int c = 0; c < 6; ++c) total_pairs += (long long)pairs[c].size();
        ctx->n_shell_pairs_kept = total_pairs;
        int chunk = (int)std::max<long long>(64, (total_pairs + 511) / 512);
        chunk = (chunk + 15) / 16 * 16;
        int chunk_base = 0;
        static const int LA[6] = {0, 1, 1, 2, 2, 2}, LB[6] = {0, 0, 1, 0, 1, 2};
        for (int c = 0; c < 6; ++c) {
            PairClass &pc = ctx->cls[c];
            pc.la = LA[c]; pc.lb = LB[c]; pc.npairs = (int)pairs[c].size();
            pc.e_off = e_off; e_off += (long long)pc.npairs * ne_of(pc.la, pc.lb);
            pc.chunk = chunk; pc.nchunks = (pc.npairs + chunk - 1) / chunk; pc.chunk_base = chunk_base; chunk_base += pc.nchunks;
            int rc;
            if ((rc = upload(ctx, pc.d_pairs, pairs[c].data(), pairs[c].size()))) return rc;
        }
        ctx->e_rows = e_off; ctx->total_chunks = chunk_base;
        int rc;
        if ((rc = upload(ctx, ctx->d_prims, prims.data(), prims.size()))) return rc;
    }

    // ---------------------------------------------------------------- a1: metrics, Cholesky, inverses
    {
        int rc, info = 0;
        size_t nJ = (size_t)ctx->nauxJ;
        if ((rc = dalloc(ctx, ctx->d_MJ, nJ * nJ))) return rc;
        if ((rc = dalloc(ctx, ctx->d_LinvJ, nJ * nJ))) return rc;
        if ((rc = build_metric(ctx, ctx->h_aux_fn, ctx->nauxJ, ctx->d_cenJ, ctx->ncenJ, OpParams{1.0, 0.0, 0.0}, false, ctx->d_MJ))) return rc;
        double *tmp = nullptr;
        RISP_CUDA_TRY(cudaMalloc((void **)&tmp, nJ * nJ * sizeof(double)));
        RISP_CUDA_TRY(cudaMemcpy(tmp, ctx->d_MJ, nJ * nJ * sizeof(double), cudaMemcpyDeviceToDevice));
        RISP_CUDA_TRY(risp_cholesky_inverse(tmp, ctx->d_LinvJ, ctx->nauxJ, &info, 0));
        cudaFree(tmp);
        if (info) { risp_set_error(ctx, "risp_setup: Coulomb metric (P|Q)_J not positive definite at pivot " + std::to_string(info)); return RISP_ENOTPD; }
        if (ctx->has_K) {
            size_t nK = (size_t)ctx->nauxK;
            if ((rc = dalloc(ctx, ctx->d_MK, nK * nK))) return rc;
            if ((rc = dalloc(ctx, ctx->d_MKinv, nK * nK))) return rc;
            OpParams opK{sys->alpha, sys->beta, sys->omega * sys->omega};
            if ((rc = build_metric(ctx, ctx->h_aux_fnK, ctx->nauxK, ctx->d_cenK, ctx->ncenK, opK, true, ctx->d_MK))) return rc;
            double *tmpL = nullptr, *tmpI = nullptr;
            RISP_CUDA_TRY(cudaMalloc((void **)&tmpL, nK * nK * sizeof(double)));
            RISP_CUDA_TRY(cudaMalloc((void **)&tmpI, nK * nK * sizeof(double)));
            RISP_CUDA_TRY(cudaMemcpy(tmpL, ctx->d_MK, nK * nK * sizeof(double), cudaMemcpyDeviceToDevice));
            RISP_CUDA_TRY(risp_cholesky_inverse(tmpL, tmpI, ctx->nauxK, &info, 0));
            if (!info) {
                // (P|Q)^-1 = L^-T L^-1
                GemmDesc d = gemm_desc(ctx->nauxK, ctx->nauxK, ctx->nauxK, tmpI, ctx->nauxK, false, tmpI, ctx->nauxK, false, ctx->d_MKinv, ctx->nauxK);
                RISP_CUDA_TRY(risp_dgemm(d, 0));
                RISP_CUDA_TRY(cudaDeviceSynchronize());
            }
            cudaFree(tmpL); cudaFree(tmpI);
            if (info) { risp_set_error(ctx, "risp_setup: exchange metric (P|J^|Q)_K not positive definite at pivot " + std::to_string(info)); return RISP_ENOTPD; }
        }
    }

    // ---------------------------------------------------------------- budgets
    {
        size_t free_b = 0, total_b = 0;
        RISP_CUDA_TRY(cudaMemGetInfo(&free_b, &total_b));
        ctx->hbm_budget = opt.hbm_budget_bytes ? opt.hbm_budget_bytes : (size_t)(0.85 * (double)free_b);
        ctx->host_budget = opt.host_budget_bytes ? opt.host_budget_bytes : ((size_t)8 << 30);
    }

    // ---------------------------------------------------------------- a3: K tensors
    if (ctx->has_K) {
        int rc;
        const int nao = ctx->nao, no = ctx->noccK, nv = ctx->nvirK, nK = ctx->nauxK, nmo = ctx->nmo;
        size_t bytes_T = ((size_t)nK * no * no + (size_t)nK * nv * nv) * sizeof(double);
        if (bytes_T > ctx->hbm_budget) { risp_set_error(ctx, "risp_setup: K tensors exceed the HBM budget (host spill not built yet)"); return RISP_ENOMEM; }
        if ((rc = dalloc(ctx, ctx->d_Tij, (size_t)nK * no * no))) return rc;
        if ((rc = dalloc(ctx, ctx->d_Tab, (size_t)nK * nv * nv))) return rc;
        double *Bij = nullptr;
        RISP_CUDA_TRY(cudaMalloc((void **)&Bij, (size_t)nK * no * no * sizeof(double)));
        // chunk of K centres: G[Pc][nao][nao] + H[Pc][nao][max(no,nv)] within ~2 GiB
        size_t per_fn = ((size_t)nao * nao + (size_t)nao * std::max(no, nv)) * sizeof(double);
        int max_fn = (int)std::max<size_t>(4, std::min<size_t>((size_t)nK, ((size_t)2 << 30) / per_fn));
        double *G = nullptr, *H = nullptr;
        RISP_CUDA_TRY(cudaMalloc((void **)&G, (size_t)max_fn * nao * nao * sizeof(double)));
        RISP_CUDA_TRY(cudaMalloc((void **)&H, (size_t)max_fn * nao * std::max(no, nv) * sizeof(double)));
        OpParams opK{sys->alpha, sys->beta, sys->omega * sys->omega};
        bool haspK = false;
        for (auto &c : cenK) if (c.qp >= 0) haspK = true;
        int c0 = 0;
        while (c0 < ctx->ncenK) {
            // centres are created in function order, so a run of centres covers a contiguous function range only if
            // each centre's functions are contiguous; take function range [f0, f1)
            int c1 = c0, f0 = 1 << 30, f1 = -1;
            while (c1 < ctx->ncenK) {
                int lo = 1 << 30, hi = -1;
                if (cenK[c1].qs >= 0) { lo = std::min(lo, cenK[c1].qs); hi = std::max(hi, cenK[c1].qs + 1); }
                if (cenK[c1].qp >= 0) { lo = std::min(lo, cenK[c1].qp); hi = std::max(hi, cenK[c1].qp + 3); }
                int nf0 = std::min(f0, lo), nf1 = std::max(f1, hi);
                if (c1 > c0 && nf1 - nf0 > max_fn) break;
                f0 = nf0; f1 = nf1; ++c1;
            }
            int nf = f1 - f0;
            if (nf > max_fn) { risp_set_error(ctx, "risp_setup: K aux functions of one centre are not contiguous"); return RISP_EINVAL; }
            RISP_CUDA_TRY(cudaMemsetAsync(G, 0, (size_t)nf * nao * nao * sizeof(double), 0));
            for (int c = 0; c < 6; ++c) {
                const PairClass &pc = ctx->cls[c];
                RISP_CUDA_TRY(risp_eri_fill(pc.la, pc.lb, haspK, true, pc.d_pairs, pc.npairs, ctx->d_prims, ctx->d_cenK + c0, c1 - c0, opK, ctx->d_boys,
                                            G - (long long)f0 * nao * nao, (long long)nao * nao, nao, 1, 0));
            }
            // occupied window: H[P] = G[P] C_o' ; B_ij[P] = C_o'^T H[P]
            GemmDesc d1 = gemm_desc(nao, no, nao, G, nao, true, ctx->d_C + ctx->occK0, nmo, false, H, no);
            d1.nb1 = nf; d1.sA1 = (long long)nao * nao; d1.sC1 = (long long)nao * no;
            RISP_CUDA_TRY(risp_dgemm(d1, 0));
            GemmDesc d2 = gemm_desc(no, no, nao, ctx->d_C + ctx->occK0, nmo, false, H, no, false, Bij + (long long)f0 * no * no, no);
            d2.nb1 = nf; d2.sB1 = (long long)nao * no; d2.sC1 = (long long)no * no;
            RISP_CUDA_TRY(risp_dgemm(d2, 0));
            // virtual window: T_ab^P = C_v'^T G[P] C_v'   (Eq. 21)
            const double *Cv = ctx->d_C + ctx->nocc + ctx->virK0;
            GemmDesc d3 = gemm_desc(nao, nv, nao, G, nao, true, Cv, nmo, false, H, nv);
            d3.nb1 = nf; d3.sA1 = (long long)nao * nao; d3.sC1 = (long long)nao * nv;
            RISP_CUDA_TRY(risp_dgemm(d3, 0));
            GemmDesc d4 = gemm_desc(nv, nv, nao, Cv, nmo, false, H, nv, false, ctx->d_Tab + (long long)f0 * nv * nv, nv);
            d4.nb1 = nf; d4.sB1 = (long long)nao * nv; d4.sC1 = (long long)nv * nv;
            RISP_CUDA_TRY(risp_dgemm(d4, 0));
            c0 = c1;
        }
        // T_ij^P = sum_Q (P|Q)^-1 B_ij^Q   (Eq. 20), stored Tij[i][P][j]
        GemmDesc d5 = gemm_desc(nK, no, nK, ctx->d_MKinv, nK, true, Bij, (long long)no * no, false, ctx->d_Tij, no);
        d5.nb1 = no; d5.sB1 = no; d5.sC1 = (long long)nK * no;
        RISP_CUDA_TRY(risp_dgemm(d5, 0));
        RISP_CUDA_TRY(cudaDeviceSynchronize());
        cudaFree(G); cudaFree(H); cudaFree(Bij);
    }
    RISP_CUDA_TRY(cudaDeviceSynchronize());
    RISP_CUDA_TRY(cudaStreamCreateWithFlags(&ctx->side, cudaStreamNonBlocking));
    for (int i = 0; i < 12; ++i) RISP_CUDA_TRY(cudaEventCreate(&ctx->ev[i]));
    ctx->ev_ok = true;
    std::memset(&ctx->tim, 0, sizeof(ctx->tim));
    return RISP_OK;
}
