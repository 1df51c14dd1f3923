// eri.cuh -- device-side three-centre integral engine (FP64, sm_100a).
//
// Computes (mu nu|P) between contracted AO shell pairs (l <= 2) and primitive s / p auxiliary Gaussians that
// share one exponent per centre (Eq. 4), for the operator (ca + cb erf(w r))/r (Eq. 25,
// PAPER.md:177; ca=1, cb=0 is the Coulomb operator of Eq. 13-16).
//
// Algorithm: Obara-Saika / Head-Gordon-Pople.  For every primitive pair the vertical recursion builds
//   [e 0|0]^(m),  e = la .. la+lb (all angular momentum on centre A), from the Boys function F_m(rho |PC|^2);
// the p-type auxiliary components follow from one more recursion step on the auxiliary centre,
//   [e 0|1_i] = (W-C)_i [e 0|0]^(1) + e_i / (2(p+g)) [e-1_i 0|0]^(1);
// primitives are summed (contraction), and the horizontal recursion (closed form: binomial expansion of
// (x-B)^b = ((x-A) + (A-B))^b) plus the Cartesian->real-solid-harmonic transform turn the "e0" intermediates
// into (mu nu|.  The hot J passes never leave the e0 representation: the density is transformed *into* it once
// per shell pair (adjoint of HRR+spherical transform) and U is transformed back once.
// This is deliberately a different algorithm from the oracle's McMurchie-Davidson scheme.
#pragma once
#include <cuda_runtime.h>

namespace risp_eri {

// ----------------------------------------------------------------------------- Cartesian component indexing
__host__ __device__ constexpr int ncart(int n) { return (n + 1) * (n + 2) / 2; }
__host__ __device__ constexpr int coff(int n) { return n * (n + 1) * (n + 2) / 6; }            // # components of degree < n
__host__ __device__ constexpr int cidx(int ex, int ey, int ez) { return coff(ex + ey + ez) + (ey + ez) * (ey + ez + 1) / 2 + ez; }
// e0 components of a pair class (la >= lb): degrees la .. la+lb
__host__ __device__ constexpr int ne_of(int la, int lb) { return coff(la + lb + 1) - coff(la); }

// ----------------------------------------------------------------------------- Boys function
// Table: F_k(x_i), x_i = i*BOYS_DX, i = 0..BOYS_NX-1, k = 0..BOYS_NK-1 (built on the host in setup.cu).
constexpr double BOYS_DX = 0.1;
constexpr int BOYS_NX = 401;           // x in [0, 40]
constexpr int BOYS_NK = 14;            // orders 0..13: up to m = 6 with an 8-term Taylor expansion
constexpr double BOYS_XMAX = 40.0;

// F_0..F_M at x.  x < 40: 8-term Taylor series of F_M AND of F_{M+1} about the nearest grid point (two independent Horner chains
// over the same table row), e^-x from the recurrence itself, e^-x = (2M+1) F_M - 2x F_{M+1} -- no exp() call, no MUFU, no
// integer scaling work -- then the downward recursion F_{m-1} = (2x F_m + e^-x)/(2m-1) (every term positive).  The absolute
// error of that e^-x is ~1e-16 (2M+1) F_M, far below the 2x F_m it is added to.  x >= 40: F_0 = sqrt(pi/x)/2 and the upward
// recursion (e^-x < 5e-18 is dropped).
template <int M>
__device__ __forceinline__ void boys(double x, const double *__restrict__ tab, double (&F)[M + 1])
{
    if (x < BOYS_XMAX) {
        int i = (int)(x * (1.0 / BOYS_DX) + 0.5);
        double d = (double)i * BOYS_DX - x;                 // -(x - x_i)
        const double *t = tab + i * BOYS_NK + M;
        double t8 = M > 0 ? __ldg(t + 8) : 0.0;
        double f = __ldg(t + 7) * (1.0 / 5040.0), g = t8 * (1.0 / 5040.0);
        double c6 = __ldg(t + 6), c5 = __ldg(t + 5), c4 = __ldg(t + 4), c3 = __ldg(t + 3), c2 = __ldg(t + 2), c1 = __ldg(t + 1), c0 = __ldg(t);
        f = fma(f, d, c6 * (1.0 / 720.0));
        f = fma(f, d, c5 * (1.0 / 120.0));
        f = fma(f, d, c4 * (1.0 / 24.0));
        f = fma(f, d, c3 * (1.0 / 6.0));
        f = fma(f, d, c2 * 0.5);
        f = fma(f, d, c1);
        f = fma(f, d, c0);
        F[M] = f;
        if (M > 0) {
            g = fma(g, d, __ldg(t + 7) * (1.0 / 720.0));
            g = fma(g, d, c6 * (1.0 / 120.0));
            g = fma(g, d, c5 * (1.0 / 24.0));
            g = fma(g, d, c4 * (1.0 / 6.0));
            g = fma(g, d, c3 * 0.5);
            g = fma(g, d, c2);
            g = fma(g, d, c1);                                  // F_{M+1}(x)
            const double x2 = 2.0 * x, ex = fma(-x2, g, (double)(2 * M + 1) * f);
#pragma unroll
            for (int m = M; m > 0; --m) F[m - 1] = fma(x2, F[m], ex) * (1.0 / (2 * m - 1));
        }
    } else {
        double ix = 1.0 / x;
        F[0] = 0.88622692545275801365 * sqrt(ix);          // sqrt(pi)/2
#pragma unroll
        for (int m = 0; m < M; ++m) F[m + 1] = F[m] * (0.5 * (2 * m + 1)) * ix;
    }
}

// ----------------------------------------------------------------------------- records
struct PrimPair {        // one primitive pair of a shell pair
    double p;            // a + b
    double Px, Py, Pz;   // (a A + b B)/p
    double cc;           // d_a d_b exp(-a b/p |AB|^2) * 2 pi^{5/2} / p   (d = contraction coef * radial norm)
    double hp;           // 1 / (2p), precomputed: the recursion then needs no FP64 division
};
struct ShellPair {       // l(A) >= l(B)
    double Ax, Ay, Az;
    double ABx, ABy, ABz;  // A - B
    int aoA, aoB;          // first AO of each shell
    int ppoff, npp;        // primitive-pair range
    int shA, shB;
    int pad0, pad1;
};
struct AuxCentre {       // s and p functions sharing one exponent on one atom
    double x, y, z, g;
    double ns, np;       // normalisation of the s and of the p functions
    int qs, qp;          // function index of s (or -1) and of p_x (or -1) in the target aux set
    double ig;           // 1 / g
};
struct OpParams { double ca, cb, w2; };   // operator (ca + cb erf(w r))/r, w2 = w*w

// ----------------------------------------------------------------------------- vertical recursion + emission, one primitive pair
// v[cidx(e)][m] = [e0|0]^(m) for deg(e) <= L, m <= MTOP - deg(e), built level by level; the e0 integrals of a level are emitted
// as soon as the level is complete, so that only the two levels below the current one are alive (the (dd| class otherwise keeps
// all 105 intermediates in registers and spills).  sink(e_local, c, value): c = 0 (s), 1..3 (p_x, p_y, p_z); e_local runs over
// degrees LA..LA+LB in cidx order.  Values include the auxiliary normalisation.
template <int LA, int LB, bool HASP, bool ERF, class Sink>
__device__ __forceinline__ void eri_e0_prim(const PrimPair &pp, double Ax, double Ay, double Az, const AuxCentre &ax,
                                            const OpParams &op, const double *__restrict__ boys_tab, Sink &&sink)
{
    constexpr int L = LA + LB, MTOP = L + (HASP ? 1 : 0);
    double v[coff(L + 1)][MTOP + 1];
    const double p = pp.p, g = ax.g;
    const double q = p + g, rsq = rsqrt(q), iq = rsq * rsq;     // 1/(p+g) from the reciprocal square root the prefactor needs anyway
    const double rho = p * g * iq;
    const double PCx = pp.Px - ax.x, PCy = pp.Py - ax.y, PCz = pp.Pz - ax.z;
    const double T = rho * (PCx * PCx + PCy * PCy + PCz * PCz);
    const double pref = pp.cc * rsq * ax.ig;                // cc carries 2 pi^{5/2}/p
    {
        double F[MTOP + 1];
        boys<MTOP>(T, boys_tab, F);
        if (ERF) {
            // erf(w r)/r: [0]^(m) -> (rho~/rho)^{m+1/2} F_m(rho~ |PC|^2), rho~ = rho w^2/(rho + w^2)
            double k2 = op.w2 / (rho + op.w2);
            double G[MTOP + 1];
            if (op.cb != 0.0) boys<MTOP>(k2 * T, boys_tab, G);
            double kf = op.cb * sqrt(k2);
#pragma unroll
            for (int m = 0; m <= MTOP; ++m) {
                F[m] = op.ca * F[m] + (op.cb != 0.0 ? kf * G[m] : 0.0);
                kf *= k2;
            }
        }
#pragma unroll
        for (int m = 0; m <= MTOP; ++m) v[0][m] = pref * F[m];
    }
    const double PA[3] = {pp.Px - Ax, pp.Py - Ay, pp.Pz - Az};
    const double c2 = g * iq;                                // rho / p
    const double WP[3] = {-c2 * PCx, -c2 * PCy, -c2 * PCz};  // W - P
    const double c1 = pp.hp;
    const double pq = p * iq;
    const double WC[3] = {pq * PCx, pq * PCy, pq * PCz};     // W - C
    const double c3 = 0.5 * iq;
#pragma unroll
    for (int n = 0; n <= L; ++n) {
        if (n > 0) {
#pragma unroll
            for (int ex = n; ex >= 0; --ex) {
#pragma unroll
                for (int ey = n - ex; ey >= 0; --ey) {
                    const int ez = n - ex - ey;
                    const int dir = ex > 0 ? 0 : (ey > 0 ? 1 : 2);
                    const int fx = ex - (dir == 0), fy = ey - (dir == 1), fz = ez - (dir == 2);
                    const int ei = dir == 0 ? fx : (dir == 1 ? fy : fz);
                    const int i1 = cidx(fx, fy, fz);
                    // levels that are only emitted need m = 0 (s) and m = 1 (p) -- MTOP - n covers exactly that at n = L
#pragma unroll
                    for (int m = 0; m <= MTOP - n; ++m) {
                        double val = fma(PA[dir], v[i1][m], WP[dir] * v[i1][m + 1]);
                        if (ei > 0) {
                            const int i2 = cidx(fx - (dir == 0), fy - (dir == 1), fz - (dir == 2));
                            val = fma((double)ei * c1, fma(-c2, v[i2][m + 1], v[i2][m]), val);
                        }
                        v[cidx(ex, ey, ez)][m] = val;
                    }
                }
            }
        }
        if (n >= LA) {
#pragma unroll
            for (int ex = n; ex >= 0; --ex) {
#pragma unroll
                for (int ey = n - ex; ey >= 0; --ey) {
                    const int ez = n - ex - ey;
                    const int id = cidx(ex, ey, ez);
                    const int el = id - coff(LA);
                    sink(el, 0, ax.ns * v[id][0]);
                    if (HASP) {
                        const int e3[3] = {ex, ey, ez};
#pragma unroll
                        for (int d = 0; d < 3; ++d) {
                            double val = WC[d] * v[id][1];
                            if (e3[d] > 0) val = fma((double)e3[d] * c3, v[cidx(ex - (d == 0), ey - (d == 1), ez - (d == 2))][1], val);
                            sink(el, 1 + d, ax.np * val);
                        }
                    }
                }
            }
        }
    }
}

// ----------------------------------------------------------------------------- HRR + spherical transform
// Angular factors of the unit-normalised real solid harmonics (include/risp.h AO order).
__device__ __forceinline__ constexpr double sph_coef(int l, int i, int c)
{
    // l = 0: 1/sqrt(4 pi); l = 1: sqrt(3/4pi) delta_ic; l = 2 rows (xy, yz, z2, xz, x2-y2) over (xx,xy,xz,yy,yz,zz)
    const double S0 = 0.28209479177387814, P0 = 0.48860251190291992, DA = 1.0925484305920792, DB = 0.31539156525252005,
                 DC = 0.54627421529603959;
    if (l == 0) return S0;
    if (l == 1) return i == c ? P0 : 0.0;
    if (i == 0) return c == 1 ? DA : 0.0;
    if (i == 1) return c == 4 ? DA : 0.0;
    if (i == 2) return c == 5 ? 2.0 * DB : ((c == 0 || c == 3) ? -DB : 0.0);
    if (i == 3) return c == 2 ? DA : 0.0;
    return c == 0 ? DC : (c == 3 ? -DC : 0.0);
}

// Enumerate cart(a,b) = sum_k coef * e0[a + k]:  f(ia, ib, e_local, coef)
template <int LA, int LB, class F>
__device__ __forceinline__ void hrr_terms(double ABx, double ABy, double ABz, F &&f)
{
    const double pw[3][3] = {{1.0, ABx, ABx * ABx}, {1.0, ABy, ABy * ABy}, {1.0, ABz, ABz * ABz}};
    constexpr int binom[3][3] = {{1, 0, 0}, {1, 1, 0}, {1, 2, 1}};
#pragma unroll
    for (int ax = LA; ax >= 0; --ax)
#pragma unroll
        for (int ay = LA - ax; ay >= 0; --ay) {
            const int az = LA - ax - ay;
            const int ia = cidx(ax, ay, az) - coff(LA);
#pragma unroll
            for (int bx = LB; bx >= 0; --bx)
#pragma unroll
                for (int by = LB - bx; by >= 0; --by) {
                    const int bz = LB - bx - by;
                    const int ib = cidx(bx, by, bz) - coff(LB);
#pragma unroll
                    for (int kx = 0; kx <= bx; ++kx)
#pragma unroll
                        for (int ky = 0; ky <= by; ++ky)
#pragma unroll
                            for (int kz = 0; kz <= bz; ++kz) {
                                const double coef = (double)(binom[bx][kx] * binom[by][ky] * binom[bz][kz]) * pw[0][bx - kx] *
                                                    pw[1][by - ky] * pw[2][bz - kz];
                                f(ia, ib, cidx(ax + kx, ay + ky, az + kz) - coff(LA), coef);
                            }
                }
        }
}

// e0[ne] -> spherical block out[(2LA+1)][(2LB+1)]
template <int LA, int LB>
__device__ __forceinline__ void e0_to_sph(const double (&e0)[ne_of(LA, LB)], double ABx, double ABy, double ABz,
                                          double (&out)[2 * LA + 1][2 * LB + 1])
{
    double cart[ncart(LA)][ncart(LB)];
#pragma unroll
    for (int i = 0; i < ncart(LA); ++i)
#pragma unroll
        for (int j = 0; j < ncart(LB); ++j) cart[i][j] = 0.0;
    hrr_terms<LA, LB>(ABx, ABy, ABz, [&](int ia, int ib, int e, double coef) { cart[ia][ib] = fma(coef, e0[e], cart[ia][ib]); });
#pragma unroll
    for (int i = 0; i < 2 * LA + 1; ++i)
#pragma unroll
        for (int j = 0; j < 2 * LB + 1; ++j) {
            double s = 0.0;
#pragma unroll
            for (int a = 0; a < ncart(LA); ++a)
#pragma unroll
                for (int b = 0; b < ncart(LB); ++b) {
                    const double c = sph_coef(LA, i, a) * sph_coef(LB, j, b);
                    if (c != 0.0) s = fma(c, cart[a][b], s);
                }
            out[i][j] = s;
        }
}

// adjoint: spherical block d[(2LA+1)][(2LB+1)] -> e0-space dbar[ne]  (sum_{ij} d_ij (ij|P) = sum_e dbar_e [e0|P])
template <int LA, int LB>
__device__ __forceinline__ void sph_to_e0_adjoint(const double (&d)[2 * LA + 1][2 * LB + 1], double ABx, double ABy, double ABz,
                                                  double (&dbar)[ne_of(LA, LB)])
{
    double cart[ncart(LA)][ncart(LB)];
#pragma unroll
    for (int a = 0; a < ncart(LA); ++a)
#pragma unroll
        for (int b = 0; b < ncart(LB); ++b) {
            double s = 0.0;
#pragma unroll
            for (int i = 0; i < 2 * LA + 1; ++i)
#pragma unroll
                for (int j = 0; j < 2 * LB + 1; ++j) {
                    const double c = sph_coef(LA, i, a) * sph_coef(LB, j, b);
                    if (c != 0.0) s = fma(c, d[i][j], s);
                }
            cart[a][b] = s;
        }
#pragma unroll
    for (int e = 0; e < ne_of(LA, LB); ++e) dbar[e] = 0.0;
    hrr_terms<LA, LB>(ABx, ABy, ABz, [&](int ia, int ib, int e, double coef) { dbar[e] = fma(coef, cart[ia][ib], dbar[e]); });
}

}  // namespace risp_eri
