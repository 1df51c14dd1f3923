// setup.cu -- risp_setup: everything of the sigma-build that does not depend on the trial vectors.
//
//   a0  screened shell-pair list, primitive-pair data                     ("screened non-zero AO pairs")
//   a1  metrics (P|Q)_J (Coulomb, s+p) and (P|J^|Q)_K (Eq. 26), Cholesky
//   a2  exchange-space window
//   a3  T_ij^P = sum_Q (ij|Q)(Q|P)^-1 (Eq. 20), T_ab^P = (ab|P) (Eq. 21, reading G3)
#include "ctx.h"
#include <algorithm>
#include <cmath>
#include <unistd.h>

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
        c.ig = 1.0 / c.g;
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
            p.hp = 0.5 / g;
            sp.push_back(r); pp.push_back(p);
        }
        if (sp.empty()) continue;
        DevScratch scr;
        ShellPair *d_sp = nullptr; PrimPair *d_pp = nullptr;
        RISP_CUDA_TRY(scr.alloc(d_sp, sp.size()));
        RISP_CUDA_TRY(scr.alloc(d_pp, pp.size()));
        RISP_CUDA_TRY(cudaMemcpy(d_sp, sp.data(), sp.size() * sizeof(ShellPair), cudaMemcpyHostToDevice));
        RISP_CUDA_TRY(cudaMemcpy(d_pp, pp.data(), pp.size() * sizeof(PrimPair), cudaMemcpyHostToDevice));
        // out[q*nfn + (aoA + i)*1 + 0]
        RISP_CUDA_TRY(risp_eri_fill(l, 0, hasp, erf_op, d_sp, (int)sp.size(), d_pp, d_cen, ncen, op, ctx->d_boys, d_M, nfn, 1, 0, 0));
        RISP_CUDA_TRY(cudaDeviceSynchronize());
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
            q.hp = 0.5 / p;
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
    for (int c = 0; c < 6; ++c) { ctx->cls[c].npairs = 0; ctx->cls[c].d_pairs = nullptr; ctx->cls[c].d_permB = nullptr; }
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
    ctx->nauxK_global = ctx->nauxK;

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
    ctx->flags = opt.flags;
    ctx->shard_count = opt.shard_count > 1 ? opt.shard_count : 1;
    ctx->shard_rank = ctx->shard_count > 1 ? opt.shard_rank : 0;
    if (ctx->shard_rank < 0 || ctx->shard_rank >= ctx->shard_count) return bad("shard_rank outside [0, shard_count)");
    if (ctx->shard_count > 1 && (opt.flags & (RISP_FLAG_TDDFT | RISP_FLAG_SPILL_HALF))) return bad("a sharded context supports neither RISP_FLAG_TDDFT nor host-spilled K slices");
    ctx->max_batch = opt.max_batch > 0 ? std::min(opt.max_batch, RISP_MS) : RISP_MS;
    auto even = [](int n) { return (n + 1) & ~1; };
    ctx->ldao = even(ctx->nao); ctx->ldocc = even(ctx->nocc); ctx->ldvir = even(ctx->nvir);
    ctx->no_p = even(ctx->noccK); ctx->nv_p = even(ctx->nvirK);
    {
        std::vector<double> tab = make_boys_table();
        int rc;
        if ((rc = upload(ctx, ctx->d_boys, tab.data(), tab.size()))) return rc;
        // C split into its occupied and virtual column blocks, each with an even leading dimension (16-byte TMA strides)
        std::vector<double> co((size_t)ctx->nao * ctx->ldocc, 0.0), cv((size_t)ctx->nao * ctx->ldvir, 0.0);
        for (int mu = 0; mu < ctx->nao; ++mu) {
            std::memcpy(&co[(size_t)mu * ctx->ldocc], sys->C + (size_t)mu * ctx->nmo, (size_t)ctx->nocc * sizeof(double));
            std::memcpy(&cv[(size_t)mu * ctx->ldvir], sys->C + (size_t)mu * ctx->nmo + ctx->nocc, (size_t)ctx->nvir * sizeof(double));
        }
        if ((rc = upload(ctx, ctx->d_Cocc, co.data(), co.size()))) return rc;
        {
            std::vector<double> cot((size_t)ctx->nocc * ctx->ldao, 0.0);
            for (int mu = 0; mu < ctx->nao; ++mu)
                for (int i = 0; i < ctx->nocc; ++i) cot[(size_t)i * ctx->ldao + mu] = sys->C[(size_t)mu * ctx->nmo + i];
            if ((rc = upload(ctx, ctx->d_CoccT, cot.data(), cot.size()))) return rc;
        }
        if ((rc = upload(ctx, ctx->d_Cvir, cv.data(), cv.size()))) return rc;
        if ((rc = upload(ctx, ctx->d_eps, sys->eps, (size_t)ctx->nmo))) return rc;
    }
    for (int s = 0; s < sys->nshl; ++s) if ((ctx->h_shl_ao[s] & 1) == 0) ctx->h_even_shell_ao.push_back(ctx->h_shl_ao[s]);
    std::vector<AuxCentre> cenJ, cenK;
    build_centres(ctx, ctx->h_aux_fn, cenJ);
    build_centres(ctx, ctx->h_aux_fnK, cenK);
    ctx->ncenJ = (int)cenJ.size(); ctx->ncenK = (int)cenK.size();
    ctx->ncenJ_pad = (ctx->ncenJ + 7) / 8 * 8;
    { int rc; if ((rc = upload(ctx, ctx->d_cenJ, cenJ.data(), cenJ.size()))) return rc; if ((rc = upload(ctx, ctx->d_cenK, cenK.data(), cenK.size()))) return rc; }

    // ---------------------------------------------------------------- a0: screened shell-pair list
    std::vector<ShellPair> pairs[6];
    std::vector<PrimPair> prims;
    // (re)install the pair classes from `pairs`: sorted lists, panel indices, e0 offsets, pass-1 chunking, device copies
    auto install_pairs = [&]() -> int {
        long long e_off = 0, total_pairs = 0;
        ctx->h_kept_pairs.clear(); ctx->n_ao_pairs_kept = 0;
        for (int c = 0; c < 6; ++c) total_pairs += (long long)pairs[c].size();
        ctx->n_shell_pairs_kept = total_pairs;
        // pass-1 chunking per class: about 16 CTAs per SM over (pair chunks) x (groups of 8 aux centres), at least 16 pairs per chunk
        const int cta_per_chunk = (ctx->ncenJ + 7) / 8;
        const int want_chunks = std::max(1, (16 * 148 + cta_per_chunk - 1) / cta_per_chunk);
        int chunk_base = 0;
        static const int LA[6] = {0, 1, 1, 2, 2, 2}, LB[6] = {0, 0, 1, 0, 1, 2};
        for (int c = 0; c < 6; ++c) {
            PairClass &pc = ctx->cls[c];
            if (pc.d_pairs) { cudaFree(pc.d_pairs); pc.d_pairs = nullptr; ctx->setup_bytes -= (size_t)pc.npairs * sizeof(ShellPair); }
            if (pc.d_permB) { cudaFree(pc.d_permB); pc.d_permB = nullptr; ctx->setup_bytes -= (size_t)pc.npairs * sizeof(int); }
            // sorted by the first AO of shell A: a panel of AO rows of D / U is then a contiguous pair range
            std::stable_sort(pairs[c].begin(), pairs[c].end(), [](const ShellPair &x, const ShellPair &y) { return x.aoA < y.aoA; });
            pc.la = LA[c]; pc.lb = LB[c]; pc.npairs = (int)pairs[c].size();
            pc.h_aoA.resize(pc.npairs);
            for (int k = 0; k < pc.npairs; ++k) {
                const ShellPair &q = pairs[c][k];
                pc.h_aoA[k] = q.aoA;
                ctx->h_kept_pairs.push_back(q.shA); ctx->h_kept_pairs.push_back(q.shB);
                ctx->n_ao_pairs_kept += (q.shA == q.shB) ? (long long)(2 * pc.la + 1) * (2 * pc.la + 2) / 2 : (long long)(2 * pc.la + 1) * (2 * pc.lb + 1);
            }
            {   // second index of the same pairs, sorted by the first AO of shell B (row panels that hold the rows of B)
                std::vector<int> perm(pc.npairs);
                for (int k = 0; k < pc.npairs; ++k) perm[k] = k;
                std::stable_sort(perm.begin(), perm.end(), [&](int x, int y) { return pairs[c][x].aoB < pairs[c][y].aoB; });
                pc.h_aoB.resize(pc.npairs);
                for (int k = 0; k < pc.npairs; ++k) pc.h_aoB[k] = pairs[c][perm[k]].aoB;
                int rcp;
                if ((rcp = upload(ctx, pc.d_permB, perm.data(), perm.size()))) return rcp;
            }
            pc.e_off = e_off; e_off += (long long)pc.npairs * ne_of(pc.la, pc.lb);
            {
                const int nch = std::max(1, std::min((pc.npairs + 15) / 16, want_chunks));
                int chunk = (pc.npairs + nch - 1) / nch;
                chunk = std::max(16, (chunk + 15) / 16 * 16);
                pc.chunk = chunk; pc.nchunks = (pc.npairs + chunk - 1) / chunk; pc.chunk_base = chunk_base; chunk_base += pc.nchunks;
            }
            int rc;
            if ((rc = upload(ctx, pc.d_pairs, pairs[c].data(), pairs[c].size()))) return rc;
        }
        ctx->e_rows = e_off; ctx->total_chunks = chunk_base;
        return RISP_OK;
    };
    {
        double tau = opt.screen_tol == 0.0 ? 1e-13 : opt.screen_tol;
        double gmin = 1e300;
        for (int s = 0; s < sys->naux; ++s) gmin = std::min(gmin, sys->aux_exp[s]);
        double vmax = 2.0 * 4.48 * std::pow(gmin, -0.25);    // ~ 2 x the peak potential of a unit-normalised s aux Gaussian
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
            }
        int rc;
        if ((rc = install_pairs())) return rc;      // the whole list: the K-tensor build below needs (mu nu|P) on every kept pair
        if ((rc = upload(ctx, ctx->d_prims, prims.data(), prims.size()))) return rc;
    }

    // ---------------------------------------------------------------- a1: metrics, Cholesky, inverses
    {
        int rc, info = 0;
        size_t nJ = (size_t)ctx->nauxJ;
        if ((rc = dalloc(ctx, ctx->d_MJ, nJ * nJ))) return rc;
        if ((rc = dalloc(ctx, ctx->d_LinvJ, nJ * nJ))) return rc;
        if ((rc = build_metric(ctx, ctx->h_aux_fn, ctx->nauxJ, ctx->d_cenJ, ctx->ncenJ, OpParams{1.0, 0.0, 0.0}, false, ctx->d_MJ))) return rc;
        DevScratch scr;
        double *tmp = nullptr;
        RISP_CUDA_TRY(scr.alloc(tmp, nJ * nJ));
        RISP_CUDA_TRY(cudaMemcpy(tmp, ctx->d_MJ, nJ * nJ * sizeof(double), cudaMemcpyDeviceToDevice));
        RISP_CUDA_TRY(risp_cholesky_inverse(tmp, ctx->d_LinvJ, ctx->nauxJ, &info, 0));
        scr.release(tmp);
        if (info) { risp_set_error(ctx, "risp_setup: Coulomb metric (P|Q)_J not positive definite at pivot " + std::to_string(info)); return RISP_ENOTPD; }
        if (ctx->has_K) {
            size_t nK = (size_t)ctx->nauxK;
            if ((rc = dalloc(ctx, ctx->d_MK, nK * nK))) return rc;
            if ((rc = dalloc(ctx, ctx->d_MKinv, nK * nK))) return rc;
            OpParams opK{sys->alpha, sys->beta, sys->omega * sys->omega};
            if ((rc = build_metric(ctx, ctx->h_aux_fnK, ctx->nauxK, ctx->d_cenK, ctx->ncenK, opK, true, ctx->d_MK))) return rc;
            double *tmpL = nullptr, *tmpI = nullptr;
            RISP_CUDA_TRY(scr.alloc(tmpL, nK * nK));
            RISP_CUDA_TRY(scr.alloc(tmpI, nK * nK));
            RISP_CUDA_TRY(cudaMemcpy(tmpL, ctx->d_MK, nK * nK * sizeof(double), cudaMemcpyDeviceToDevice));
            RISP_CUDA_TRY(risp_cholesky_inverse(tmpL, tmpI, ctx->nauxK, &info, 0));
            if (!info && (ctx->flags & RISP_FLAG_TDDFT)) {      // full TDDFT whitens (ov|J^|Q) with L_K^-1 (symmetric placement of the metric)
                if ((rc = dalloc(ctx, ctx->d_LinvK, nK * nK))) return rc;
                RISP_CUDA_TRY(cudaMemcpy(ctx->d_LinvK, tmpI, nK * nK * sizeof(double), cudaMemcpyDeviceToDevice));
            }
            if (!info) {
                // (P|Q)^-1 = L^-T L^-1
                GemmDesc d = gemm_desc(ctx->nauxK, ctx->nauxK, ctx->nauxK, tmpI, ctx->nauxK, false, tmpI, ctx->nauxK, false, ctx->d_MKinv, ctx->nauxK);
                RISP_CUDA_TRY(risp_dgemm(d, 0));
                RISP_CUDA_TRY(cudaDeviceSynchronize());
            }
            if (info) { risp_set_error(ctx, "risp_setup: exchange metric (P|J^|Q)_K not positive definite at pivot " + std::to_string(info)); return RISP_ENOTPD; }
        }
    }

    // ---------------------------------------------------------------- budgets
    size_t free_b = 0, total_b = 0;
    RISP_CUDA_TRY(cudaMemGetInfo(&free_b, &total_b));
    ctx->hbm_budget = opt.hbm_budget_bytes ? opt.hbm_budget_bytes : (size_t)(0.85 * (double)free_b) + ctx->setup_bytes;
    if (opt.host_budget_bytes) ctx->host_budget = opt.host_budget_bytes;
    else {   // half of the physical host memory
        const long pages = sysconf(_SC_PHYS_PAGES), psz = sysconf(_SC_PAGE_SIZE);
        ctx->host_budget = pages > 0 && psz > 0 ? (size_t)pages * (size_t)psz / 2 : ((size_t)8 << 30);
    }

    // ---------------------------------------------------------------- a3: K tensors, packed lower triangles (Eq. 20-21)
    if (ctx->has_K) {
        int rc;
        const int nao = ctx->nao, no = ctx->noccK, nv = ctx->nvirK, nK = ctx->nauxK, no_p = ctx->no_p, nv_p = ctx->nv_p;
        const long long ldao = ctx->ldao;
        ctx->tri_o = (long long)no * (no + 1) / 2; ctx->tri_v = (long long)nv * (nv + 1) / 2;
        const long long tri_o = ctx->tri_o, tri_v = ctx->tri_v;
        // ---- placement: what the budget leaves after the work space of a max_batch matvec (and, with the default budget, the
        //      caller's X and sigma) holds the first nK_dev slices; the others go to pinned host memory
        {
            const size_t slice = (size_t)(tri_o + tri_v) * 8;
            const size_t dimb = (size_t)ctx->nocc * ctx->nvir * 8;
            size_t reserve = ((size_t)ctx->e_rows * RISP_MS + (size_t)ctx->total_chunks * ctx->ncenJ_pad * 4 * RISP_MS + 3 * (size_t)ctx->nauxJ * RISP_MS) * 8;
            if (!opt.hbm_budget_bytes) reserve += 2 * (size_t)ctx->max_batch * dimb;
            if (ctx->flags & RISP_FLAG_KEEP_STAGES) reserve += (size_t)ctx->max_batch * dimb;
            if (ctx->flags & RISP_FLAG_TDDFT) reserve += (size_t)nK * no * nv_p * 8 + (!opt.hbm_budget_bytes ? (size_t)ctx->max_batch * dimb : 0);
            size_t left = ctx->hbm_budget > ctx->setup_bytes + reserve ? ctx->hbm_budget - ctx->setup_bytes - reserve : 0;
            // work space if everything had to be streamed (upper bound of the staging need), then the slices
            MatvecPlan tmp;
            ctx->nK_dev = 0;
            size_t ws = risp_plan_workspace(ctx, ctx->max_batch, left, tmp, true);
            if (ws == 0) { risp_set_error(ctx, "risp_setup: the HBM budget is too small for the matvec work space"); return RISP_ENOMEM; }
            left -= std::min(left, ws);
            ctx->nK_dev = (int)std::min<size_t>((size_t)nK, left / slice);
            if (ctx->flags & RISP_FLAG_SPILL_HALF) ctx->nK_dev = std::min(ctx->nK_dev, nK / 2);
            if (ctx->shard_count > 1) {
                // sharded: this rank keeps the slices of its own aux centres only, all of them in HBM; every (ij|Q) is needed while
                // the metric is applied (Eq. 20 mixes all Q), so T_ij is built whole and cut down afterwards
                int nloc = 0;
                for (int c = 0; c < ctx->ncenK; ++c)
                    if (c % ctx->shard_count == ctx->shard_rank) nloc += (cenK[c].qs >= 0 ? 1 : 0) + (cenK[c].qp >= 0 ? 3 : 0);
                if ((size_t)nK * tri_o * 8 + (size_t)nloc * tri_v * 8 > left) {
                    risp_set_error(ctx, "risp_setup: a sharded context keeps its K slices in HBM; the budget is too small (use more shards)");
                    return RISP_ENOMEM;
                }
                ctx->nK_dev = nK;
            }
        }
        const bool sharded = ctx->shard_count > 1;
        std::vector<int> loc_of(nK, -1);                 // sharded: index of a K function among this rank's slices, or -1
        int nK_loc = 0;
        for (int c = 0; c < ctx->ncenK; ++c) {
            if (sharded && c % ctx->shard_count != ctx->shard_rank) continue;
            if (cenK[c].qs >= 0) loc_of[cenK[c].qs] = nK_loc++;
            if (cenK[c].qp >= 0) for (int t = 0; t < 3; ++t) loc_of[cenK[c].qp + t] = nK_loc++;
        }
        const int nK_host = nK - ctx->nK_dev;
        // ---- scratch for a chunk of aux functions: G[f][nao][ldao], H[f][nao][max(no_p,nv_p)], full B / T[f][n][n_p], packed
        const size_t nmax_p = (size_t)std::max(no_p, nv_p), sq = std::max((size_t)no * no_p, (size_t)nv * nv_p);
        const size_t per_fn = ((size_t)nao * ldao + (size_t)nao * nmax_p + sq + (size_t)std::max(tri_o, tri_v)) * sizeof(double);
        bool haspK = false;
        for (auto &c : cenK) if (c.qp >= 0) haspK = true;
        int max_fn = (int)std::max<size_t>(haspK ? 4 : 1, std::min<size_t>((size_t)nK, ((size_t)3 << 30) / per_fn));
        if (ctx->flags & RISP_FLAG_SMALL_KBUILD) max_fn = std::min(max_fn, 5);
        DevScratch scr;                                  // every temporary of the build: released on any return
        double *G = nullptr, *H = nullptr, *F = nullptr, *Pk = nullptr, *CoK = nullptr, *CvK = nullptr, *BP = nullptr, *BPr = nullptr, *tmpc = nullptr;
        AuxCentre *d_cenRun = nullptr;
        RISP_CUDA_TRY(scr.alloc(G, (size_t)max_fn * nao * ldao));
        RISP_CUDA_TRY(scr.alloc(H, (size_t)max_fn * nao * nmax_p));
        RISP_CUDA_TRY(scr.alloc(F, (size_t)max_fn * sq));
        RISP_CUDA_TRY(scr.alloc(Pk, (size_t)max_fn * std::max(tri_o, tri_v)));
        RISP_CUDA_TRY(scr.alloc(d_cenRun, (size_t)ctx->ncenK));
        double *Fov = nullptr;
        if (ctx->flags & RISP_FLAG_TDDFT) {      // T_ia^P': kept whole in HBM; needed by the (ib|ja) term of Eq. 2 only
            if ((rc = dalloc(ctx, ctx->d_Tov, (size_t)nK * no * nv_p))) { risp_set_error(ctx, "risp_setup: the (ia|P) tensor of full TDDFT does not fit in HBM"); return rc; }
            RISP_CUDA_TRY(cudaMemset(ctx->d_Tov, 0, (size_t)nK * no * nv_p * sizeof(double)));
            RISP_CUDA_TRY(scr.alloc(Fov, (size_t)max_fn * no * nv_p));
        }
        // window blocks of C with even leading dimensions and aligned bases
        RISP_CUDA_TRY(scr.alloc(CoK, (size_t)nao * no_p));
        RISP_CUDA_TRY(scr.alloc(CvK, (size_t)nao * nv_p));
        RISP_CUDA_TRY(cudaMemset(CoK, 0, (size_t)nao * no_p * sizeof(double)));
        RISP_CUDA_TRY(cudaMemset(CvK, 0, (size_t)nao * nv_p * sizeof(double)));
        RISP_CUDA_TRY(cudaMemcpy2D(CoK, (size_t)no_p * 8, ctx->d_Cocc + ctx->occK0, (size_t)ctx->ldocc * 8, (size_t)no * 8, nao, cudaMemcpyDeviceToDevice));
        RISP_CUDA_TRY(cudaMemcpy2D(CvK, (size_t)nv_p * 8, ctx->d_Cvir + ctx->virK0, (size_t)ctx->ldvir * 8, (size_t)nv * 8, nao, cudaMemcpyDeviceToDevice));
        // all (ij|Q) slices, packed, in HBM until the metric has been applied (Eq. 20 mixes every Q): the first nK_dev of them
        // in their final place, the others in a block that is copied to the host and freed afterwards
        if (ctx->nK_dev > 0) { if ((rc = dalloc(ctx, ctx->d_TijP, (size_t)ctx->nK_dev * tri_o))) return rc; }
        if (nK_host > 0) RISP_CUDA_TRY(scr.alloc(BPr, (size_t)nK_host * tri_o));
        BP = ctx->d_TijP;
        auto bp_slice = [&](int f) { return f < ctx->nK_dev ? BP + (size_t)f * tri_o : BPr + (size_t)(f - ctx->nK_dev) * tri_o; };
        if (nK_host > 0) {
            RISP_CUDA_TRY(cudaHostAlloc((void **)&ctx->h_TijP, (size_t)nK_host * tri_o * sizeof(double), cudaHostAllocDefault));
            RISP_CUDA_TRY(cudaHostAlloc((void **)&ctx->h_TabP, (size_t)nK_host * tri_v * sizeof(double), cudaHostAllocDefault));
        }
        OpParams opK{sys->alpha, sys->beta, sys->omega * sys->omega};
        for (int pass = 0; pass < 2; ++pass) {          // pass 0: occupied window -> BP ; pass 1: virtual window -> T_ab
            if (pass == 1 && ctx->nK_dev > 0) { if ((rc = dalloc(ctx, ctx->d_TabP, (size_t)(sharded ? nK_loc : ctx->nK_dev) * tri_v))) return rc; }
            const int n = pass == 0 ? no : nv, n_p = pass == 0 ? no_p : nv_p;
            const long long tri = pass == 0 ? tri_o : tri_v;
            const double *Cw = pass == 0 ? CoK : CvK;
            int c0 = 0;
            while (c0 < ctx->ncenK) {
                // a run of centres with at most max_fn functions; inside the run the functions get compact indices 0 .. nf-1, so the
                // order of the caller's aux shells (grouped by atom, or all s shells first) does not matter: fn_of[j] is the
                // function's index in the K auxiliary set
                std::vector<AuxCentre> run;
                std::vector<int> fn_of;
                int c1 = c0;
                while (c1 < ctx->ncenK) {
                    if (pass == 1 && sharded && c1 % ctx->shard_count != ctx->shard_rank) { ++c1; continue; }      // (ab|P): own centres only
                    const int add = (cenK[c1].qs >= 0 ? 1 : 0) + (cenK[c1].qp >= 0 ? 3 : 0);
                    if (c1 > c0 && (int)fn_of.size() + add > max_fn) break;
                    AuxCentre cc = cenK[c1];
                    if (cc.qs >= 0) { fn_of.push_back(cc.qs); cc.qs = (int)fn_of.size() - 1; }
                    if (cc.qp >= 0) { for (int t = 0; t < 3; ++t) fn_of.push_back(cenK[c1].qp + t); cc.qp = (int)fn_of.size() - 3; }
                    run.push_back(cc);
                    ++c1;
                }
                const int nf = (int)fn_of.size();
                if (nf == 0) { c0 = c1; continue; }
                RISP_CUDA_TRY(cudaMemcpy(d_cenRun, run.data(), run.size() * sizeof(AuxCentre), cudaMemcpyHostToDevice));
                RISP_CUDA_TRY(cudaMemsetAsync(G, 0, (size_t)nf * nao * ldao * sizeof(double), 0));
                for (int c = 0; c < 6; ++c) {
                    const PairClass &pc = ctx->cls[c];
                    RISP_CUDA_TRY(risp_eri_fill(pc.la, pc.lb, haspK, true, pc.d_pairs, pc.npairs, ctx->d_prims, d_cenRun, (int)run.size(), opK, ctx->d_boys, G,
                                                (long long)nao * ldao, ldao, 1, 0));
                }
                // H[P] = (mu nu|P) C_w ; F[P] = C_w^T H[P]      (Eq. 20-21 before the metric)
                GemmDesc d1 = gemm_desc(nao, n, nao, G, ldao, true, Cw, n_p, false, H, n_p);
                d1.nb1 = nf; d1.sA1 = (long long)nao * ldao; d1.sC1 = (long long)nao * n_p;
                RISP_CUDA_TRY(risp_dgemm(d1, 0));
                GemmDesc d2 = gemm_desc(n, n, nao, Cw, n_p, false, H, n_p, false, F, n_p);
                d2.nb1 = nf; d2.sB1 = (long long)nao * n_p; d2.sC1 = (long long)n * n_p;
                RISP_CUDA_TRY(risp_dgemm(d2, 0));
                if (pass == 0) {
                    for (int j = 0; j < nf; ++j)
                        RISP_CUDA_TRY(risp_pack_sym(F + (size_t)j * n * n_p, (long long)n * n_p, n_p, n, 1, bp_slice(fn_of[j]), tri, 0));
                } else {
                    if (ctx->d_Tov) {      // (ia|J^|P) = C_o'^T [(mu nu|P) C_v'] from the half-transformed H of this pass
                        GemmDesc d3 = gemm_desc(no, nv, nao, CoK, no_p, false, H, nv_p, false, Fov, nv_p);
                        d3.nb1 = nf; d3.sB1 = (long long)nao * nv_p; d3.sC1 = (long long)no * nv_p;
                        RISP_CUDA_TRY(risp_dgemm(d3, 0));
                        for (int j = 0; j < nf; ++j)
                            RISP_CUDA_TRY(cudaMemcpy2DAsync(ctx->d_Tov + (size_t)fn_of[j] * no * nv_p, (size_t)nv_p * 8, Fov + (size_t)j * no * nv_p, (size_t)nv_p * 8,
                                                            (size_t)nv * 8, no, cudaMemcpyDeviceToDevice, 0));
                    }
                    RISP_CUDA_TRY(risp_pack_sym(F, (long long)n * n_p, n_p, n, nf, Pk, tri, 0));
                    for (int j = 0; j < nf; ++j) {
                        const int f = sharded ? loc_of[fn_of[j]] : fn_of[j];
                        const double *src = Pk + (size_t)j * tri;
                        if (f < ctx->nK_dev) RISP_CUDA_TRY(cudaMemcpyAsync(ctx->d_TabP + (size_t)f * tri, src, (size_t)tri * 8, cudaMemcpyDeviceToDevice, 0));
                        else RISP_CUDA_TRY(cudaMemcpyAsync(ctx->h_TabP + (size_t)(f - ctx->nK_dev) * tri, src, (size_t)tri * 8, cudaMemcpyDeviceToHost, 0));
                    }
                }
                RISP_CUDA_TRY(cudaStreamSynchronize(0));      // d_cenRun and the scratch are reused by the next run
                c0 = c1;
            }
            if (pass == 0) {
                // T_ij^P = sum_Q (P|Q)^-1 (ij|Q)   (Eq. 20): [BP; BPr] <- MKinv [BP; BPr], in column panels, in place
                const int nKd = ctx->nK_dev;
                long long w = std::min<long long>(tri_o, std::max<long long>(2, (((long long)1 << 30) / ((long long)nK * 8)) & ~1LL));
                RISP_CUDA_TRY(scr.alloc(tmpc, (size_t)nK * w));
                for (long long col = 0; col < tri_o; col += w) {
                    const int wc = (int)std::min<long long>(w, tri_o - col);
                    if (nKd > 0) {
                        GemmDesc d5 = gemm_desc(nK, wc, nKd, ctx->d_MKinv, nK, true, BP + col, tri_o, false, tmpc, w);
                        RISP_CUDA_TRY(risp_dgemm(d5, 0));
                    }
                    if (nK_host > 0) {
                        GemmDesc d6 = gemm_desc(nK, wc, nK_host, ctx->d_MKinv + nKd, nK, true, BPr + col, tri_o, false, tmpc, w, 1.0, nKd > 0 ? 1.0 : 0.0);
                        RISP_CUDA_TRY(risp_dgemm(d6, 0));
                    }
                    if (nKd > 0)
                        RISP_CUDA_TRY(cudaMemcpy2DAsync(BP + col, (size_t)tri_o * 8, tmpc, (size_t)w * 8, (size_t)wc * 8, nKd, cudaMemcpyDeviceToDevice, 0));
                    if (nK_host > 0)
                        RISP_CUDA_TRY(cudaMemcpy2DAsync(BPr + col, (size_t)tri_o * 8, tmpc + (size_t)nKd * w, (size_t)w * 8, (size_t)wc * 8, nK_host,
                                                        cudaMemcpyDeviceToDevice, 0));
                }
                RISP_CUDA_TRY(cudaDeviceSynchronize());
                scr.release(tmpc);
                if (nK_host > 0) {
                    RISP_CUDA_TRY(cudaMemcpy(ctx->h_TijP, BPr, (size_t)nK_host * tri_o * 8, cudaMemcpyDeviceToHost));
                    scr.release(BPr);
                }
            }
        }
        RISP_CUDA_TRY(cudaDeviceSynchronize());
        if (sharded) {
            double *loc = nullptr;
            if (nK_loc > 0) RISP_CUDA_TRY(cudaMalloc((void **)&loc, (size_t)nK_loc * tri_o * 8));
            for (int f = 0; f < nK; ++f)
                if (loc_of[f] >= 0) RISP_CUDA_TRY(cudaMemcpyAsync(loc + (size_t)loc_of[f] * tri_o, ctx->d_TijP + (size_t)f * tri_o, (size_t)tri_o * 8, cudaMemcpyDeviceToDevice, 0));
            RISP_CUDA_TRY(cudaDeviceSynchronize());
            cudaFree(ctx->d_TijP);
            ctx->setup_bytes -= (size_t)(nK - nK_loc) * tri_o * 8;
            ctx->d_TijP = loc;
            ctx->nauxK_global = nK; ctx->nauxK = nK_loc; ctx->nK_dev = nK_loc;
            if (nK_loc == 0) ctx->has_K = false;
        }
        if (ctx->d_Tov) {
            // T^P <- sum_Q L_K^-1[P][Q] (ov|J^|Q): [nK x nK] x [nK x (o' v')] in column panels, in place
            const long long cols = (long long)no * nv_p;
            const long long w = std::min<long long>(cols, std::max<long long>(2, (((long long)1 << 30) / ((long long)nK * 8)) & ~1LL));
            double *tmpw = nullptr;
            RISP_CUDA_TRY(scr.alloc(tmpw, (size_t)nK * w));
            for (long long col = 0; col < cols; col += w) {
                const int wc = (int)std::min<long long>(w, cols - col);
                GemmDesc d7 = gemm_desc(nK, wc, nK, ctx->d_LinvK, nK, true, ctx->d_Tov + col, cols, false, tmpw, w);
                RISP_CUDA_TRY(risp_dgemm(d7, 0));
                RISP_CUDA_TRY(cudaMemcpy2DAsync(ctx->d_Tov + col, (size_t)cols * 8, tmpw, (size_t)w * 8, (size_t)wc * 8, nK, cudaMemcpyDeviceToDevice, 0));
            }
            RISP_CUDA_TRY(cudaDeviceSynchronize());
        }
    }
    RISP_CUDA_TRY(cudaDeviceSynchronize());
    if (ctx->shard_count > 1) {
        // P-sharded sigma-build: from here on this rank runs both integral passes and the pair-sparse halves
        // of the J transforms on its own pairs only -- the kept pairs of every class are dealt round robin
        for (int c = 0; c < 6; ++c) {
            std::vector<ShellPair> mine;
            for (size_t k = 0; k < pairs[c].size(); ++k)
                if ((int)(k % ctx->shard_count) == ctx->shard_rank) mine.push_back(pairs[c][k]);
            pairs[c].swap(mine);
        }
        int rc;
        if ((rc = install_pairs())) return rc;
    }
    RISP_CUDA_TRY(cudaStreamCreateWithFlags(&ctx->side, cudaStreamNonBlocking));
    for (int i = 0; i < RISP_NEV; ++i) RISP_CUDA_TRY(cudaEventCreate(&ctx->ev[i]));
    RISP_CUDA_TRY(cudaEventCreateWithFlags(&ctx->evFork, cudaEventDisableTiming));
    for (int c = 0; c < 6; ++c) {
        RISP_CUDA_TRY(cudaStreamCreateWithFlags(&ctx->cls_st[c], cudaStreamNonBlocking));
        RISP_CUDA_TRY(cudaEventCreateWithFlags(&ctx->evJoin[c], cudaEventDisableTiming));
    }
    for (int b = 0; b < 2; ++b) {
        RISP_CUDA_TRY(cudaEventCreateWithFlags(&ctx->evStage[b], cudaEventDisableTiming));
        RISP_CUDA_TRY(cudaEventCreateWithFlags(&ctx->evStageFree[b], cudaEventDisableTiming));
    }
    ctx->ev_ok = true;
    std::memset(&ctx->tim, 0, sizeof(ctx->tim));
    return RISP_OK;
}
