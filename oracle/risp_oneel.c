/*
 * ORACLE -- test infrastructure, not product code.
 *
 * One-electron integrals for the transition properties of TDA-risp (arxiv/paper_2603_29257, Eq. 5-8):
 *   dipole length         <mu| (r - O)_k |nu>              k = x, y, z      (enters mu_0n, Eq. 7)
 *   angular momentum      <mu| ((r - O) x nabla)_k |nu>    k = x, y, z      (enters m_0n, Eq. 8)
 * over the same contracted, unit-normalised real-solid-harmonic AO shells as oracle/risp_integrals.c (conventions of
 * include/risp.h), from the textbook McMurchie-Davidson Hermite expansion, written out term by term in long double:
 *   1D overlap   S_ij = E_0^{ij} sqrt(pi/p)
 *   1D moment    M_ij = (E_1^{ij} + (P - O) E_0^{ij}) sqrt(pi/p)          [x - O = (x - P) + (P - O), Hermite Lambda_1 = 2p (x-P) Lambda_0]
 *   1D gradient  D_ij = j S_{i,j-1} - 2 b S_{i,j+1}                        [d/dx acts on the ket Gaussian x_B^j exp(-b x_B^2)]
 * and the three-dimensional integrals are products of these, e.g. ((r-O) x nabla)_x = (y-O_y) d/dz - (z-O_z) d/dy:
 *   <a|L_x|b> = S^x (M^y D^z - D^y M^z).
 * Only tests/, __graft_entry__.smoke() and bench.py's CPU legs may use anything in oracle/.  Shares nothing with the CUDA path
 * (which uses the Obara-Saika overlap recursion and takes the gradient through the centre derivative).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef long double real;
static const real PI = 3.14159265358979323846264338327950288L;

#define LMAX 2
#define JD (LMAX + 2)            /* ket index runs to l + 1 */
#define TD (2 * LMAX + 3)

static const int CART[3][6][3] = {
    {{0, 0, 0}},
    {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}},
    {{2, 0, 0}, {1, 1, 0}, {1, 0, 1}, {0, 2, 0}, {0, 1, 1}, {0, 0, 2}}};
static const int NCART[3] = {1, 3, 6};

static real gamma_half(int l)
{
    real g = sqrtl(PI) / 2;
    for (int k = 0; k < l; ++k) g *= (k + 1.5L);
    return g;
}
static real radial_norm(real a, int l) { return sqrtl(2.0L * powl(2.0L * a, l + 1.5L) / gamma_half(l)); }

static void sph_matrix(int l, real M[5][6])
{
    memset(M, 0, sizeof(real) * 30);
    if (l == 0) M[0][0] = 1.0L / sqrtl(4 * PI);
    else if (l == 1) for (int k = 0; k < 3; ++k) M[k][k] = sqrtl(3.0L / (4 * PI));
    else {
        real a = sqrtl(15.0L / (4 * PI)), b = sqrtl(5.0L / (16 * PI)), c = sqrtl(15.0L / (16 * PI));
        M[0][1] = a; M[1][4] = a; M[2][5] = 2 * b; M[2][0] = -b; M[2][3] = -b; M[3][2] = a; M[4][0] = c; M[4][3] = -c;
    }
}

static void shell_coefs(int l, int np, const double *ex, const double *cf, real *out)
{
    real s = 0;
    for (int k = 0; k < np; ++k)
        for (int q = 0; q < np; ++q)
            s += (real)cf[k] * cf[q] * radial_norm(ex[k], l) * radial_norm(ex[q], l) * gamma_half(l) / (2.0L * powl((real)ex[k] + ex[q], l + 1.5L));
    for (int k = 0; k < np; ++k) out[k] = (real)cf[k] * radial_norm(ex[k], l) / sqrtl(s);
}

/* E_t^{ij}, i <= LMAX, j <= LMAX + 1, without the exp(-mu Q^2) factor */
static void hermite_E(real p, real PA, real PB, real E[LMAX + 1][JD][TD])
{
    memset(E, 0, sizeof(real) * (LMAX + 1) * JD * TD);
    E[0][0][0] = 1.0L;
    for (int i = 0; i < LMAX; ++i)
        for (int t = 0; t <= i + 1; ++t)
            E[i + 1][0][t] = (t > 0 ? E[i][0][t - 1] / (2 * p) : 0.0L) + PA * E[i][0][t] + (t + 1) * E[i][0][t + 1];
    for (int i = 0; i <= LMAX; ++i)
        for (int j = 0; j + 1 < JD; ++j)
            for (int t = 0; t <= i + j + 1; ++t)
                E[i][j + 1][t] = (t > 0 ? E[i][j][t - 1] / (2 * p) : 0.0L) + PB * E[i][j][t] + (t + 1) * E[i][j][t + 1];
}

/* out[6][nao][nao]: components 0-2 = <mu|(r-O)_k|nu>, 3-5 = <mu|((r-O) x nabla)_k|nu> */
void oracle_oneel(const double *xyz, int nshl, const int *shl_atom, const int *shl_l, const int *shl_nprim, const int *shl_poff,
                  const double *prim_exp, const double *prim_coef, const double *origin, double *out)
{
    int *off = malloc(sizeof(int) * (nshl + 1));
    off[0] = 0;
    for (int s = 0; s < nshl; ++s) off[s + 1] = off[s] + 2 * shl_l[s] + 1;
    const int nao = off[nshl];
    const size_t nn = (size_t)nao * nao;
    memset(out, 0, sizeof(double) * 6 * nn);
#pragma omp parallel for schedule(dynamic, 1)
    for (int sa = 0; sa < nshl; ++sa)
        for (int sb = 0; sb < nshl; ++sb) {
            const int la = shl_l[sa], lb = shl_l[sb];
            real A[3], B[3], ca[16], cb[16], Ma[5][6], Mb[5][6], AB2 = 0;
            for (int d = 0; d < 3; ++d) {
                A[d] = xyz[3 * shl_atom[sa] + d]; B[d] = xyz[3 * shl_atom[sb] + d];
                AB2 += (A[d] - B[d]) * (A[d] - B[d]);
            }
            shell_coefs(la, shl_nprim[sa], prim_exp + shl_poff[sa], prim_coef + shl_poff[sa], ca);
            shell_coefs(lb, shl_nprim[sb], prim_exp + shl_poff[sb], prim_coef + shl_poff[sb], cb);
            sph_matrix(la, Ma); sph_matrix(lb, Mb);
            real cart[6][6][6];
            memset(cart, 0, sizeof(cart));
            for (int ka = 0; ka < shl_nprim[sa]; ++ka)
                for (int kb = 0; kb < shl_nprim[sb]; ++kb) {
                    const real a = prim_exp[shl_poff[sa] + ka], b = prim_exp[shl_poff[sb] + kb], p = a + b;
                    const real pre = expl(-a * b / p * AB2) * ca[ka] * cb[kb];
                    real S[3][LMAX + 1][JD], M[3][LMAX + 1][JD], D[3][LMAX + 1][LMAX + 1];
                    for (int d = 0; d < 3; ++d) {
                        const real Pd = (a * A[d] + b * B[d]) / p;
                        real E[LMAX + 1][JD][TD];
                        hermite_E(p, Pd - A[d], Pd - B[d], E);
                        const real rt = sqrtl(PI / p);
                        for (int i = 0; i <= LMAX; ++i)
                            for (int j = 0; j < JD; ++j) {
                                S[d][i][j] = E[i][j][0] * rt;
                                M[d][i][j] = (E[i][j][1] + (Pd - (real)origin[d]) * E[i][j][0]) * rt;
                            }
                        for (int i = 0; i <= LMAX; ++i)
                            for (int j = 0; j <= LMAX; ++j) D[d][i][j] = (j > 0 ? j * S[d][i][j - 1] : 0.0L) - 2 * b * S[d][i][j + 1];
                    }
                    for (int x = 0; x < NCART[la]; ++x)
                        for (int y = 0; y < NCART[lb]; ++y) {
                            const int *u = CART[la][x], *v = CART[lb][y];
                            const real Sx = S[0][u[0]][v[0]], Sy = S[1][u[1]][v[1]], Sz = S[2][u[2]][v[2]];
                            const real Mx = M[0][u[0]][v[0]], My = M[1][u[1]][v[1]], Mz = M[2][u[2]][v[2]];
                            const real Dx = D[0][u[0]][v[0]], Dy = D[1][u[1]][v[1]], Dz = D[2][u[2]][v[2]];
                            cart[0][x][y] += pre * Mx * Sy * Sz;
                            cart[1][x][y] += pre * Sx * My * Sz;
                            cart[2][x][y] += pre * Sx * Sy * Mz;
                            cart[3][x][y] += pre * Sx * (My * Dz - Dy * Mz);      /* y d/dz - z d/dy */
                            cart[4][x][y] += pre * Sy * (Mz * Dx - Dz * Mx);      /* z d/dx - x d/dz */
                            cart[5][x][y] += pre * Sz * (Mx * Dy - Dx * My);      /* x d/dy - y d/dx */
                        }
                }
            for (int c = 0; c < 6; ++c)
                for (int i = 0; i < 2 * la + 1; ++i)
                    for (int j = 0; j < 2 * lb + 1; ++j) {
                        real v = 0;
                        for (int x = 0; x < NCART[la]; ++x)
                            for (int y = 0; y < NCART[lb]; ++y) v += Ma[i][x] * Mb[j][y] * cart[c][x][y];
                        out[c * nn + (size_t)(off[sa] + i) * nao + off[sb] + j] = (double)v;
                    }
        }
    free(off);
}
