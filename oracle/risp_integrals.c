/*
 * ORACLE -- test infrastructure, not product code.
 *
 * Plain, slow, from-the-definition electron-repulsion integrals for TDA-risp
 * (arxiv/paper_2603_29257).  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may use anything in oracle/.
 * It shares no code, table or constant with the CUDA path.
 *
 * What it computes (Eq. 3-4; Eq. 24-26):
 *   (P|Q)      two-centre integrals over primitive s/p auxiliary Gaussians,
 *   (mu nu|P)  three-centre integrals between contracted spherical AO shells
 *              (l <= 2) and the auxiliary Gaussians,
 * each with the operator  (alpha + beta erf(omega r12)) / r12   (Eq. 25;
 * alpha=1, beta=0 is the Coulomb operator of Eq. 3/13).
 *
 * Method: McMurchie-Davidson, written out term by term:
 *   Hermite expansion coefficients E_t^{ij}, Hermite Coulomb integrals
 *   R^n_{tuv} from the Boys function F_n.  No screening unless the caller
 *   passes kab_tol > 0 (a Gaussian-product prefactor bound), no symmetry use,
 *   no blocking.  Internals run in `real` = long double (x87, 64-bit
 *   mantissa) so that the 1e-12 absolute integral tolerance is tested against
 *   something more accurate than FP64; inputs and outputs are double.
 *
 * AO conventions (the C ABI's, include/risp.h): unit-normalised real solid
 * harmonics, order s; p=(x,y,z); d=(xy,yz,z2,xz,x2-y2).  Aux functions:
 * unit-normalised Cartesian primitives s; p=(x,y,z).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef long double real;
#define EXP expl
#define SQRT sqrtl
#define ERF erfl
#define POW powl
#define FABS fabsl
static const real PI = 3.14159265358979323846264338327950288L;

#define LMAX_AO 2
#define LMAX_AUX 1
#define NMAX (2 * LMAX_AO + LMAX_AUX + 1) /* highest Boys order + 1 */

/* ---- Boys function F_n(x) = int_0^1 t^{2n} exp(-x t^2) dt, n = 0..nmax -------------
 * x < 35: ascending series at n = nmax (all terms positive), then downward recursion
 *         F_{n-1} = (2x F_n + e^-x)/(2n-1);
 * x >= 35: F_0 = sqrt(pi/x)/2 * erf(sqrt x) exactly, then upward recursion
 *         F_{n+1} = ((2n+1) F_n - e^-x)/(2x), stable for x >> n.                      */
static void boys(int nmax, real x, real *F)
{
    real ex = EXP(-x);
    if (x < 35.0L) {
        real term = 1.0L / (2 * nmax + 1), sum = term;
        for (int k = 1; k < 400; ++k) {
            term *= 2.0L * x / (2 * nmax + 2 * k + 1);
            sum += term;
            if (term < 1e-22L * sum) break;
        }
        F[nmax] = ex * sum;
        for (int n = nmax; n > 0; --n) F[n - 1] = (2.0L * x * F[n] + ex) / (2 * n - 1);
    } else {
        F[0] = 0.5L * SQRT(PI / x) * ERF(SQRT(x));
        for (int n = 0; n < nmax; ++n) F[n + 1] = ((2 * n + 1) * F[n] - ex) / (2.0L * x);
    }
}

void oracle_boys(int nmax, double x, double *F_out)
{
    real F[64];
    boys(nmax, (real)x, F);
    for (int n = 0; n <= nmax; ++n) F_out[n] = (double)F[n];
}

/* ---- Hermite Coulomb integrals R^0_{tuv}, t+u+v <= N, for the operator (ca + cb erf(w r))/r.
 * R^n_000 = kappa (-2 at)^n F_n(at |R|^2); Coulomb: at = a, kappa = 1;
 * erf(w r)/r: 1/at = 1/a + 1/w^2, kappa = sqrt(at/a).  Recursion
 * R^n_{t+1,u,v} = t R^{n+1}_{t-1,u,v} + X R^{n+1}_{t,u,v} (same for u, v).           */
#define RD (NMAX + 1)
static void hermite_R(int N, real a, const real *Rv, real ca, real cb, real w, real out[RD][RD][RD])
{
    static const int D = RD;
    real Rn[RD + 1][RD][RD][RD];
    memset(Rn, 0, sizeof(Rn));
    real r2 = Rv[0] * Rv[0] + Rv[1] * Rv[1] + Rv[2] * Rv[2];
    real F[RD + 1], G[RD + 1];
    boys(N, a * r2, F);
    real at = 0, kap = 0;
    if (cb != 0.0L) {
        at = 1.0L / (1.0L / a + 1.0L / (w * w));
        kap = SQRT(at / a);
        boys(N, at * r2, G);
    }
    for (int n = 0; n <= N; ++n) {
        real v = ca * POW(-2.0L * a, n) * F[n];
        if (cb != 0.0L) v += cb * kap * POW(-2.0L * at, n) * G[n];
        Rn[n][0][0][0] = v;
    }
    (void)D;
    for (int n = N - 1; n >= 0; --n) {
        int M = N - n;
        for (int t = 0; t <= M; ++t)
            for (int u = 0; t + u <= M; ++u)
                for (int v = 0; t + u + v <= M; ++v) {
                    if (t + u + v == 0) continue;
                    real val;
                    if (t > 0)
                        val = (t > 1 ? (t - 1) * Rn[n + 1][t - 2][u][v] : 0.0L) + Rv[0] * Rn[n + 1][t - 1][u][v];
                    else if (u > 0)
                        val = (u > 1 ? (u - 1) * Rn[n + 1][t][u - 2][v] : 0.0L) + Rv[1] * Rn[n + 1][t][u - 1][v];
                    else
                        val = (v > 1 ? (v - 1) * Rn[n + 1][t][u][v - 2] : 0.0L) + Rv[2] * Rn[n + 1][t][u][v - 1];
                    Rn[n][t][u][v] = val;
                }
    }
    for (int t = 0; t <= N; ++t)
        for (int u = 0; t + u <= N; ++u)
            for (int v = 0; t + u + v <= N; ++v) out[t][u][v] = Rn[0][t][u][v];
}

/* ---- two-centre Hermite expansion E_t^{ij}, one Cartesian direction, WITHOUT the exp(-mu Q^2) factor.
 * E_0^{00} = 1; E_t^{i+1,j} = E_{t-1}^{ij}/(2p) + PA E_t^{ij} + (t+1) E_{t+1}^{ij}; likewise j with PB.  */
#define ED (2 * LMAX_AO + 2)
static void hermite_E(int la, int lb, real p, real PA, real PB, real E[LMAX_AO + 1][LMAX_AO + 1][ED])
{
    memset(E, 0, sizeof(real) * (LMAX_AO + 1) * (LMAX_AO + 1) * ED);
    E[0][0][0] = 1.0L;
    for (int i = 0; i < la; ++i)
        for (int t = 0; t <= i + 1; ++t)
            E[i + 1][0][t] = (t > 0 ? E[i][0][t - 1] / (2 * p) : 0.0L) + PA * E[i][0][t] + (t + 1) * E[i][0][t + 1];
    for (int i = 0; i <= la; ++i)
        for (int j = 0; j < lb; ++j)
            for (int t = 0; t <= i + j + 1; ++t)
                E[i][j + 1][t] = (t > 0 ? E[i][j][t - 1] / (2 * p) : 0.0L) + PB * E[i][j][t] + (t + 1) * E[i][j][t + 1];
}

/* one-centre version: E_0^0 = 1, E_t^{l+1} = E_{t-1}^l/(2g) + (t+1) E_{t+1}^l */
static void hermite_E1(int l, real g, real E[LMAX_AUX + 1][LMAX_AUX + 2])
{
    memset(E, 0, sizeof(real) * (LMAX_AUX + 1) * (LMAX_AUX + 2));
    E[0][0] = 1.0L;
    for (int i = 0; i < l; ++i)
        for (int t = 0; t <= i + 1; ++t) E[i + 1][t] = (t > 0 ? E[i][t - 1] / (2 * g) : 0.0L) + (t + 1) * E[i][t + 1];
}

/* ---- unnormalised primitive Cartesian three-centre integral (ab|c) --------------------------------
 * (ab|c) = 2 pi^{5/2} / (p g sqrt(p+g)) exp(-mu |AB|^2)
 *          sum_{tuv} E^{ab}_{tuv} sum_{t'u'v'} (-1)^{t'+u'+v'} E^{c}_{t'u'v'} R_{t+t',u+u',v+v'}(alpha, P - C)
 * The tables (E, E^c, R, prefactor) depend only on the exponents, centres and the *total* angular momenta;
 * prim3c_eval picks one Cartesian component triple out of them.                                       */
typedef struct {
    real E[3][LMAX_AO + 1][LMAX_AO + 1][ED], Ec[3][LMAX_AUX + 1][LMAX_AUX + 2], R[RD][RD][RD], pref;
} tab3c;

static void prim3c_tables(real a, const real *A, int La, real b, const real *B, int Lb, real g, const real *C, int Lc,
                          real ca, real cb, real w, tab3c *T)
{
    real p = a + b, mu = a * b / p;
    real P[3], Rv[3], AB2 = 0;
    for (int d = 0; d < 3; ++d) {
        P[d] = (a * A[d] + b * B[d]) / p;
        Rv[d] = P[d] - C[d];
        AB2 += (A[d] - B[d]) * (A[d] - B[d]);
    }
    for (int d = 0; d < 3; ++d) {
        hermite_E(La, Lb, p, P[d] - A[d], P[d] - B[d], T->E[d]);
        hermite_E1(Lc, g, T->Ec[d]);
    }
    hermite_R(La + Lb + Lc, p * g / (p + g), Rv, ca, cb, w, T->R);
    T->pref = 2.0L * POW(PI, 2.5L) / (p * g * SQRT(p + g)) * EXP(-mu * AB2);
}

static real prim3c_eval(const tab3c *T, const int *la, const int *lb, const int *lc)
{
    real sum = 0;
    for (int t = 0; t <= la[0] + lb[0]; ++t)
        for (int u = 0; u <= la[1] + lb[1]; ++u)
            for (int v = 0; v <= la[2] + lb[2]; ++v) {
                real e = T->E[0][la[0]][lb[0]][t] * T->E[1][la[1]][lb[1]][u] * T->E[2][la[2]][lb[2]][v];
                if (e == 0.0L) continue;
                real inner = 0;
                for (int tt = 0; tt <= lc[0]; ++tt)
                    for (int uu = 0; uu <= lc[1]; ++uu)
                        for (int vv = 0; vv <= lc[2]; ++vv) {
                            real sgn = ((tt + uu + vv) & 1) ? -1.0L : 1.0L;
                            inner += sgn * T->Ec[0][lc[0]][tt] * T->Ec[1][lc[1]][uu] * T->Ec[2][lc[2]][vv] *
                                     T->R[t + tt][u + uu][v + vv];
                        }
                sum += e * inner;
            }
    return T->pref * sum;
}

static real prim3c(real a, const real *A, const int *la, real b, const real *B, const int *lb,
                   real g, const real *C, const int *lc, real ca, real cb, real w)
{
    tab3c T;
    prim3c_tables(a, A, la[0] + la[1] + la[2], b, B, lb[0] + lb[1] + lb[2], g, C, lc[0] + lc[1] + lc[2], ca, cb, w, &T);
    return prim3c_eval(&T, la, lb, lc);
}

/* ---- unnormalised primitive Cartesian two-centre integral (c|d) ----------------------------------- */
static real prim2c(real gc, const real *C, const int *lc, real gd, const real *Dv, const int *ld, real ca, real cb, real w)
{
    real Rv[3];
    for (int d = 0; d < 3; ++d) Rv[d] = C[d] - Dv[d];
    real Ec[3][LMAX_AUX + 1][LMAX_AUX + 2], Ed[3][LMAX_AUX + 1][LMAX_AUX + 2];
    for (int d = 0; d < 3; ++d) {
        hermite_E1(lc[d], gc, Ec[d]);
        hermite_E1(ld[d], gd, Ed[d]);
    }
    int N = lc[0] + lc[1] + lc[2] + ld[0] + ld[1] + ld[2];
    real R[RD][RD][RD];
    hermite_R(N, gc * gd / (gc + gd), Rv, ca, cb, w, R);
    real sum = 0;
    for (int t = 0; t <= lc[0]; ++t)
        for (int u = 0; u <= lc[1]; ++u)
            for (int v = 0; v <= lc[2]; ++v)
                for (int tt = 0; tt <= ld[0]; ++tt)
                    for (int uu = 0; uu <= ld[1]; ++uu)
                        for (int vv = 0; vv <= ld[2]; ++vv) {
                            real sgn = ((tt + uu + vv) & 1) ? -1.0L : 1.0L;
                            sum += Ec[0][lc[0]][t] * Ec[1][lc[1]][u] * Ec[2][lc[2]][v] * sgn * Ed[0][ld[0]][tt] * Ed[1][ld[1]][uu] *
                                   Ed[2][ld[2]][vv] * R[t + tt][u + uu][v + vv];
                        }
    return 2.0L * POW(PI, 2.5L) / (gc * gd * SQRT(gc + gd)) * sum;
}

double oracle_prim3c(double a, const double *A, const int *la, double b, const double *B, const int *lb,
                     double g, const double *C, const int *lc, double ca, double cb, double w)
{
    real Ar[3] = {A[0], A[1], A[2]}, Br[3] = {B[0], B[1], B[2]}, Cr[3] = {C[0], C[1], C[2]};
    return (double)prim3c(a, Ar, la, b, Br, lb, g, Cr, lc, ca, cb, w);
}

double oracle_prim2c(double gc, const double *C, const int *lc, double gd, const double *D, const int *ld,
                     double ca, double cb, double w)
{
    real Cr[3] = {C[0], C[1], C[2]}, Dr[3] = {D[0], D[1], D[2]};
    return (double)prim2c(gc, Cr, lc, gd, Dr, ld, ca, cb, w);
}

/* ---- normalisation and spherical components --------------------------- */
static const int CART[3][6][3] = {
    {{0, 0, 0}},
    {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}},
    {{2, 0, 0}, {1, 1, 0}, {1, 0, 1}, {0, 2, 0}, {0, 1, 1}, {0, 0, 2}}};
static const int NCART[3] = {1, 3, 6};

static real gamma_half(int l) /* Gamma(l + 3/2) */
{
    real g = SQRT(PI) / 2;
    for (int k = 0; k < l; ++k) g *= (k + 1.5L);
    return g;
}
static real radial_norm(real a, int l) { return SQRT(2.0L * POW(2.0L * a, l + 1.5L) / gamma_half(l)); }

/* angular factors: rows = spherical component, cols = Cartesian monomial in CART order */
static void sph_matrix(int l, real M[5][6])
{
    memset(M, 0, sizeof(real) * 30);
    if (l == 0) M[0][0] = 1.0L / SQRT(4 * PI);
    else if (l == 1) for (int k = 0; k < 3; ++k) M[k][k] = SQRT(3.0L / (4 * PI));
    else {
        real a = SQRT(15.0L / (4 * PI)), b = SQRT(5.0L / (16 * PI)), c = SQRT(15.0L / (16 * PI));
        M[0][1] = a;                              /* xy        */
        M[1][4] = a;                              /* yz        */
        M[2][5] = 2 * b; M[2][0] = -b; M[2][3] = -b; /* 2zz-xx-yy */
        M[3][2] = a;                              /* xz        */
        M[4][0] = c; M[4][3] = -c;                /* xx-yy     */
    }
}

/* contraction coefficients times primitive radial norms, shell rescaled to unit norm */
static void shell_coefs(int l, int np, const double *ex, const double *cf, real *out)
{
    real s = 0;
    for (int k = 0; k < np; ++k)
        for (int q = 0; q < np; ++q)
            s += (real)cf[k] * cf[q] * radial_norm(ex[k], l) * radial_norm(ex[q], l) * gamma_half(l) /
                 (2.0L * POW((real)ex[k] + ex[q], l + 1.5L));
    for (int k = 0; k < np; ++k) out[k] = (real)cf[k] * radial_norm(ex[k], l) / SQRT(s);
}

static real aux_norm(real g, int l)
{
    real ns = POW(2.0L * g / PI, 0.75L);
    return l == 0 ? ns : ns * 2.0L * SQRT(g);
}

typedef struct {
    int natm; const double *xyz;
    int nshl; const int *shl_atom, *shl_l, *shl_nprim, *shl_poff; const double *prim_exp, *prim_coef;
    int naux; const int *aux_atom, *aux_l; const double *aux_exp;
} basis_t;

/* AO overlap matrix S[nao][nao] -- used only to pin the normalisation conventions */
void oracle_overlap(int natm, const double *xyz, int nshl, const int *shl_atom, const int *shl_l, const int *shl_nprim,
                    const int *shl_poff, const double *prim_exp, const double *prim_coef, double *S)
{
    int *off = malloc(sizeof(int) * (nshl + 1));
    off[0] = 0;
    for (int s = 0; s < nshl; ++s) off[s + 1] = off[s] + 2 * shl_l[s] + 1;
    int nao = off[nshl];
    (void)natm;
    for (int sa = 0; sa < nshl; ++sa)
        for (int sb = 0; sb < nshl; ++sb) {
            int la = shl_l[sa], lb = shl_l[sb];
            real A[3], B[3], ca[16], cb[16], Ma[5][6], Mb[5][6];
            for (int d = 0; d < 3; ++d) { A[d] = xyz[3 * shl_atom[sa] + d]; B[d] = xyz[3 * shl_atom[sb] + d]; }
            shell_coefs(la, shl_nprim[sa], prim_exp + shl_poff[sa], prim_coef + shl_poff[sa], ca);
            shell_coefs(lb, shl_nprim[sb], prim_exp + shl_poff[sb], prim_coef + shl_poff[sb], cb);
            sph_matrix(la, Ma); sph_matrix(lb, Mb);
            real cart[6][6];
            memset(cart, 0, sizeof(cart));
            for (int ka = 0; ka < shl_nprim[sa]; ++ka)
                for (int kb = 0; kb < shl_nprim[sb]; ++kb) {
                    real a = prim_exp[shl_poff[sa] + ka], b = prim_exp[shl_poff[sb] + kb], p = a + b, AB2 = 0;
                    real E[3][LMAX_AO + 1][LMAX_AO + 1][ED];
                    for (int d = 0; d < 3; ++d) {
                        real Pd = (a * A[d] + b * B[d]) / p;
                        hermite_E(la, lb, p, Pd - A[d], Pd - B[d], E[d]);
                        AB2 += (A[d] - B[d]) * (A[d] - B[d]);
                    }
                    real pre = POW(PI / p, 1.5L) * EXP(-a * b / p * AB2) * ca[ka] * cb[kb];
                    for (int x = 0; x < NCART[la]; ++x)
                        for (int y = 0; y < NCART[lb]; ++y)
                            cart[x][y] += pre * E[0][CART[la][x][0]][CART[lb][y][0]][0] * E[1][CART[la][x][1]][CART[lb][y][1]][0] *
                                          E[2][CART[la][x][2]][CART[lb][y][2]][0];
                }
            for (int i = 0; i < 2 * la + 1; ++i)
                for (int j = 0; j < 2 * lb + 1; ++j) {
                    real v = 0;
                    for (int x = 0; x < NCART[la]; ++x)
                        for (int y = 0; y < NCART[lb]; ++y) v += Ma[i][x] * Mb[j][y] * cart[x][y];
                    S[(size_t)(off[sa] + i) * nao + off[sb] + j] = (double)v;
                }
        }
    free(off);
}

/* (P|Q) over the listed aux shells: out[nf][nf], nf = sum over listed shells of (1 or 3) */
void oracle_int2c(const double *xyz, int nsel, const int *sel, const int *aux_atom, const int *aux_l, const double *aux_exp,
                  double ca, double cb, double w, double *out)
{
    int *off = malloc(sizeof(int) * (nsel + 1));
    off[0] = 0;
    for (int s = 0; s < nsel; ++s) off[s + 1] = off[s] + NCART[aux_l[sel[s]]];
    int nf = off[nsel];
    for (int s = 0; s < nsel; ++s)
        for (int q = 0; q < nsel; ++q) {
            int ps = sel[s], pq = sel[q];
            real C[3], Dv[3];
            for (int d = 0; d < 3; ++d) { C[d] = xyz[3 * aux_atom[ps] + d]; Dv[d] = xyz[3 * aux_atom[pq] + d]; }
            real gs = aux_exp[ps], gq = aux_exp[pq];
            for (int x = 0; x < NCART[aux_l[ps]]; ++x)
                for (int y = 0; y < NCART[aux_l[pq]]; ++y)
                    out[(size_t)(off[s] + x) * nf + off[q] + y] =
                        (double)(aux_norm(gs, aux_l[ps]) * aux_norm(gq, aux_l[pq]) *
                                 prim2c(gs, C, CART[aux_l[ps]][x], gq, Dv, CART[aux_l[pq]][y], ca, cb, w));
        }
    free(off);
}

/* (mu nu|P) for the listed aux shells: out[nf][nao][nao].
 * full_square != 0: every ordered shell pair is computed on its own (used to pin (mu nu|P) = (nu mu|P));
 * otherwise shell pairs sa >= sb are computed and mirrored.
 * kab_tol > 0: skip a primitive pair whose Gaussian-product prefactor exp(-mu |AB|^2) is below kab_tol
 * (reading G14: conservative distance bound, only for the largest oracle cases). */
void oracle_int3c(const double *xyz, int nshl, const int *shl_atom, const int *shl_l, const int *shl_nprim, const int *shl_poff,
                  const double *prim_exp, const double *prim_coef, int nsel, const int *sel, const int *aux_atom,
                  const int *aux_l, const double *aux_exp, double ca, double cb, double w, int full_square, double kab_tol,
                  double *out)
{
    int *off = malloc(sizeof(int) * (nshl + 1));
    off[0] = 0;
    for (int s = 0; s < nshl; ++s) off[s + 1] = off[s] + 2 * shl_l[s] + 1;
    int nao = off[nshl];
    int *aoff = malloc(sizeof(int) * (nsel + 1));
    aoff[0] = 0;
    for (int s = 0; s < nsel; ++s) aoff[s + 1] = aoff[s] + NCART[aux_l[sel[s]]];
    size_t nn = (size_t)nao * nao;
    memset(out, 0, sizeof(double) * nn * aoff[nsel]);
#pragma omp parallel for schedule(dynamic, 1)
    for (int sa = 0; sa < nshl; ++sa)
        for (int sb = 0; sb < (full_square ? nshl : sa + 1); ++sb) {
            int la = shl_l[sa], lb = shl_l[sb];
            real A[3], B[3], ca_[16], cb_[16], Ma[5][6], Mb[5][6], AB2 = 0;
            for (int d = 0; d < 3; ++d) {
                A[d] = xyz[3 * shl_atom[sa] + d]; B[d] = xyz[3 * shl_atom[sb] + d];
                AB2 += (A[d] - B[d]) * (A[d] - B[d]);
            }
            shell_coefs(la, shl_nprim[sa], prim_exp + shl_poff[sa], prim_coef + shl_poff[sa], ca_);
            shell_coefs(lb, shl_nprim[sb], prim_exp + shl_poff[sb], prim_coef + shl_poff[sb], cb_);
            sph_matrix(la, Ma); sph_matrix(lb, Mb);
            for (int q = 0; q < nsel; ++q) {
                int P = sel[q], lc = aux_l[P];
                real g = aux_exp[P], Cc[3];
                for (int d = 0; d < 3; ++d) Cc[d] = xyz[3 * aux_atom[P] + d];
                real cart[6][6][3];
                memset(cart, 0, sizeof(cart));
                for (int ka = 0; ka < shl_nprim[sa]; ++ka)
                    for (int kb = 0; kb < shl_nprim[sb]; ++kb) {
                        real a = prim_exp[shl_poff[sa] + ka], b = prim_exp[shl_poff[sb] + kb];
                        if (kab_tol > 0 && EXP(-a * b / (a + b) * AB2) < kab_tol) continue;
                        tab3c T;
                        prim3c_tables(a, A, la, b, B, lb, g, Cc, lc, ca, cb, w, &T);
                        for (int x = 0; x < NCART[la]; ++x)
                            for (int y = 0; y < NCART[lb]; ++y)
                                for (int z = 0; z < NCART[lc]; ++z)
                                    cart[x][y][z] += ca_[ka] * cb_[kb] * prim3c_eval(&T, CART[la][x], CART[lb][y], CART[lc][z]);
                    }
                for (int z = 0; z < NCART[lc]; ++z)
                    for (int i = 0; i < 2 * la + 1; ++i)
                        for (int j = 0; j < 2 * lb + 1; ++j) {
                            real v = 0;
                            for (int x = 0; x < NCART[la]; ++x)
                                for (int y = 0; y < NCART[lb]; ++y) v += Ma[i][x] * Mb[j][y] * cart[x][y][z];
                            v *= aux_norm(g, lc);
                            double *o = out + nn * (aoff[q] + z);
                            o[(size_t)(off[sa] + i) * nao + off[sb] + j] = (double)v;
                            if (!full_square) o[(size_t)(off[sb] + j) * nao + off[sa] + i] = (double)v;
                        }
            }
        }
    free(off);
    free(aoff);
}
