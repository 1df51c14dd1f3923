"""More pins for the oracle ("Oracle (c)"): the normalisation of the p-type auxiliary functions, the
conditioning of the metrics, the RI invariance under a re-mix of the auxiliary functions (SURVEY 8(c).4,
pin I6), invariance of A under a rigid motion of the molecule, and the `kab_tol` screening branch against the unscreened
path (reading G14).  CPU only."""
import math
import os

import numpy as np
import pytest
from scipy.special import erf

from oracle import risp_oracle as ro
from workloads import make_system, trial_vectors

GOLD = os.path.join(os.path.dirname(__file__), "golden")
BOHR_ANG = 0.529177210903
G_C = 0.2 / (4 / 3.25) ** 2          # 0.13203125 bohr^-2


def _gold(name):
    out = {}
    for line in open(os.path.join(GOLD, name)):
        line = line.split("#")[0].split()
        if line:
            out[line[0]] = float(line[1])
    return out


def _aux_only_system(xyz_bohr, aux_atom, aux_l, aux_exp, alpha=0.16, beta=0.84, omega=0.2):
    """The smallest dict `Oracle` accepts: the aux shells that matter plus one dummy s AO shell."""
    n = len(xyz_bohr)
    return dict(natm=n, xyz_bohr=np.asarray(xyz_bohr, dtype=float), Z=np.full(n, 6, dtype=np.int32), nshl=1,
                shl_atom=np.array([0], dtype=np.int32), shl_l=np.array([0], dtype=np.int32), shl_nprim=np.array([1], dtype=np.int32),
                shl_poff=np.array([0], dtype=np.int32), prim_exp=np.array([1.0]), prim_coef=np.array([1.0]),
                naux=len(aux_l), aux_atom=np.asarray(aux_atom, dtype=np.int32), aux_l=np.asarray(aux_l, dtype=np.int32),
                aux_exp=np.asarray(aux_exp, dtype=float), aux_in_K=(np.asarray(aux_l) == 0).astype(np.uint8),
                nao=1, nocc=1, nvir=1, C=np.ones((1, 2)), eps=np.array([-1.0, 1.0]), alpha=alpha, beta=beta, omega=omega, cutoff_ev=0.0)


# ------------------------------------------------------------------ aux_norm(l = 1)
def test_p_aux_function_is_unit_normalised():
    """N_p^2 = (normalised (p|p)) / (unnormalised primitive (p|p)) taken from the oracle; <p|p> = N_p^2 int x^2 e^{-2 g r^2} = 1 by
    Gauss-Hermite quadrature of the defining integral."""
    g = 0.37
    o = ro.Oracle(_aux_only_system([[0.1, 0.2, -0.3]], [0, 0], [0, 1], [g, g]))
    M = o.int2c(o.selJ)                                                 # functions: s, px, py, pz
    x, w = np.polynomial.hermite.hermgauss(40)                          # int f(t) e^{-t^2} dt
    for k in range(3):
        lk = [0, 0, 0]; lk[k] = 1
        raw = ro.prim2c(g, o.xyz[0], lk, g, o.xyz[0], lk)
        Np2 = M[1 + k, 1 + k] / raw
        # int x^2 e^{-2 g r^2} d3r with t = sqrt(2g) x per axis
        one_d = float(np.sum(w)) / math.sqrt(2 * g)
        x2 = float(np.sum(w * x * x)) / (2 * g) ** 1.5
        assert Np2 * x2 * one_d * one_d == pytest.approx(1.0, rel=1e-13)
    raw_s = ro.prim2c(g, o.xyz[0], [0, 0, 0], g, o.xyz[0], [0, 0, 0])
    one_d = float(np.sum(w)) / math.sqrt(2 * g)
    assert M[0, 0] / raw_s * one_d ** 3 == pytest.approx(1.0, rel=1e-13)


def test_one_centre_pp_closed_form():
    """(p_x|p_x) = 4 pi/(3 g) for the unit-normalised function (derivation in tests/golden/aux_p_norm.txt), both operators."""
    gold = _gold("aux_p_norm.txt")
    assert gold["pp_coulomb"] == pytest.approx(4 * math.pi / (3 * G_C), rel=1e-15)
    ac = G_C / 2; ae = 1 / (2 / G_C + 1 / 0.04)
    assert gold["pp_rsh"] == pytest.approx(4 * math.pi / (3 * G_C) * (0.16 + 0.84 * (ae / ac) ** 1.5), rel=1e-14)
    o = ro.Oracle(_aux_only_system([[0.4, -1.0, 2.0]], [0, 0], [0, 1], [G_C, G_C]))
    for key, op in (("pp_coulomb", (1.0, 0.0, 0.0)), ("pp_rsh", (0.16, 0.84, 0.2))):
        M = o.int2c(o.selJ, *op)
        for k in range(3):
            assert M[1 + k, 1 + k] == pytest.approx(gold[key], rel=1e-14)
        off = M - np.diag(np.diag(M))
        assert np.abs(off).max() < 1e-14                                # (s|p) and (p_x|p_y) vanish on one centre


def test_normalised_pp_by_quadrature_of_the_definition():
    """Two-centre (p_i|p_j) of NORMALISED functions = int rho_i(r) V_j(r) dr with the closed-form potential of a p Gaussian,
    Gauss-Hermite product grid, norms typed out here (N_p = (2g/pi)^(3/4) 2 sqrt g)."""
    gc, gd = 0.21, 0.34
    Cc, Dd = np.array([0.3, -0.2, 0.5]), np.array([-0.9, 0.8, 1.4])
    o = ro.Oracle(_aux_only_system([Cc, Dd], [0, 1], [1, 1], [gc, gd]))
    n = 44
    x, wq = np.polynomial.hermite.hermgauss(n)
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij")
    W = (wq[:, None, None] * wq[None, :, None] * wq[None, None, :]).reshape(-1) / gc ** 1.5
    pts = np.stack([X.reshape(-1), Y.reshape(-1), Z.reshape(-1)], axis=1) / math.sqrt(gc) + Cc[None]
    Np = lambda g: (2 * g / math.pi) ** 0.75 * 2 * math.sqrt(g)
    for op in ((1.0, 0.0, 0.0), (0.16, 0.84, 0.2)):
        M = o.int2c(o.selJ, *op)
        for i in range(3):
            for j in range(3):
                d = pts - Dd[None, :]
                R = np.linalg.norm(d, axis=1)
                V = np.zeros(len(pts))
                for coef, s2 in ((op[0], gd), (op[1], gd * op[2] ** 2 / (gd + op[2] ** 2) if op[1] else 0.0)):
                    if coef == 0:
                        continue
                    s = math.sqrt(s2)
                    fp = 2 * s / math.sqrt(math.pi) * np.exp(-s2 * R * R) / R - erf(s * R) / (R * R)
                    V += coef * (math.pi / gd) ** 1.5 / (2 * gd) * fp * (-d[:, j] / R)
                ref = Np(gc) * Np(gd) * float(np.sum(W * (pts[:, i] - Cc[i]) * V))
                assert M[i, 3 + j] == pytest.approx(ref, rel=1e-9, abs=1e-11)


def test_contracted_ss_p_element(sys1):
    """A contracted, normalised (s s|p_k) element re-assembled from pinned primitive integrals and norms typed out here."""
    o = ro.Oracle(sys1)
    from workloads.generate import normalised_coefs, _radial_norm
    sa, sb = 0, 2
    assert o.shl_l[sa] == 0 and o.shl_l[sb] == 0
    P = int(np.nonzero(o.aux_l == 1)[0][1]); g = o.aux_exp[P]; C = o.xyz[o.aux_atom[P]]
    for op in ((1.0, 0.0, 0.0), (0.16, 0.84, 0.2)):
        I = o.int3c([P], *op)
        ea = o.pe[o.shl_poff[sa]:o.shl_poff[sa] + o.shl_nprim[sa]]; eb = o.pe[o.shl_poff[sb]:o.shl_poff[sb] + o.shl_nprim[sb]]
        ca = normalised_coefs(0, ea, o.pc[o.shl_poff[sa]:o.shl_poff[sa] + o.shl_nprim[sa]]) * _radial_norm(ea, 0)
        cb = normalised_coefs(0, eb, o.pc[o.shl_poff[sb]:o.shl_poff[sb] + o.shl_nprim[sb]]) * _radial_norm(eb, 0)
        for k in range(3):
            lk = [0, 0, 0]; lk[k] = 1
            tot = 0.0
            for q, a in enumerate(ea):
                for r, b in enumerate(eb):
                    tot += ca[q] * cb[r] * ro.prim3c(a, o.xyz[o.shl_atom[sa]], [0, 0, 0], b, o.xyz[o.shl_atom[sb]], [0, 0, 0], g, C, lk, *op)
            tot *= (1 / math.sqrt(4 * math.pi)) ** 2 * (2 * g / math.pi) ** 0.75 * 2 * math.sqrt(g)
            assert I[k, 0, 2] == pytest.approx(tot, rel=1e-13, abs=1e-15)


# ------------------------------------------------------------------ C6 zig-zag chain
def test_metric_condition_numbers_c6_chain():
    """24x24 s+p Coulomb metric: lambda_min 0.0871, lambda_max 404.5, cond 4.64e3; s-only cond 59.5 (Coulomb), 176.5 (RSH);
    s+p RSH cond 1.93e4 -- SURVEY App. B.3 (computed there with mpmath, three significant digits printed)."""
    d = 1.54 / BOHR_ANG
    h = math.radians(109.47) / 2
    xyz = np.array([[k * d * math.sin(h), (k % 2) * d * math.cos(h), 0.0] for k in range(6)])
    aux_atom = np.repeat(np.arange(6), 2); aux_l = np.tile([0, 1], 6)
    o = ro.Oracle(_aux_only_system(xyz, aux_atom, aux_l, np.full(12, G_C)))
    MJ = o.int2c(o.selJ)
    w = np.linalg.eigvalsh(MJ)
    assert MJ.shape == (24, 24) and w[0] > 0
    assert w[0] == pytest.approx(0.0871, rel=6e-3)
    assert w[-1] == pytest.approx(404.5, rel=2e-3)
    assert w[-1] / w[0] == pytest.approx(4.64e3, rel=6e-3)
    ws = np.linalg.eigvalsh(o.int2c(o.selK))
    assert ws[-1] / ws[0] == pytest.approx(59.5, rel=5e-3)
    wr = np.linalg.eigvalsh(o.int2c(o.selK, 0.16, 0.84, 0.2))
    assert wr[-1] / wr[0] == pytest.approx(176.5, rel=5e-3)
    wj = np.linalg.eigvalsh(o.int2c(o.selJ, 0.16, 0.84, 0.2))
    assert wj[0] > 0 and wj[-1] / wj[0] == pytest.approx(1.93e4, rel=6e-3)


# ------------------------------------------------------------------ I6: re-mix of the auxiliary functions
def test_sigma_invariant_under_aux_remix(sys_small_rsh, oracle_small_rsh):
    """RI depends only on the span of the aux set: scale every aux function by a random factor and rotate every p shell by a
    random orthogonal 3x3 (in the 3c AND the 2c integrals) -- sigma, J and K must not move."""
    X = trial_vectors(sys_small_rsh, 3)
    ref = oracle_small_rsh.sigma(X, parts=True)
    o = ro.Oracle(sys_small_rsh)
    rng = np.random.default_rng(77)
    blocks = []
    for l in o.aux_l:
        if l == 0:
            blocks.append(np.array([[rng.uniform(0.3, 3.0) * rng.choice([-1.0, 1.0])]]))
        else:
            Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
            blocks.append(Q * rng.uniform(0.3, 3.0))

    def mix_matrix(sel):
        nf = sum(b.shape[0] for b in (blocks[s] for s in sel))
        T = np.zeros((nf, nf)); f = 0
        for s in sel:
            b = blocks[s]; T[f:f + len(b), f:f + len(b)] = b; f += len(b)
        return T

    int3c0, int2c0 = o.int3c, o.int2c
    o.int3c = lambda sel, *a, **k: np.einsum('pq,qmn->pmn', mix_matrix(list(sel)), int3c0(sel, *a, **k))
    o.int2c = lambda sel, *a, **k: mix_matrix(list(sel)) @ int2c0(sel, *a, **k) @ mix_matrix(list(sel)).T
    got = o.sigma(X, parts=True)
    assert np.abs(o.MJ - oracle_small_rsh.MJ).max() > 0.1              # the mixed metric really is another matrix
    for a, b, name in zip(got, ref, ("sigma", "diag", "J", "K")):
        assert np.linalg.norm(a - b) <= 1e-11 * np.linalg.norm(b), name


# ------------------------------------------------------------------ rigid motion of the whole molecule
def _ylm(l, u):
    """Unit-normalised real solid harmonics in the ABI order (include/risp.h) at the points u[n][3]."""
    x, y, z = u[:, 0], u[:, 1], u[:, 2]
    if l == 0:
        return np.full((len(u), 1), 1 / math.sqrt(4 * math.pi))
    if l == 1:
        return math.sqrt(3 / (4 * math.pi)) * np.stack([x, y, z], axis=1)
    return np.stack([math.sqrt(15 / (4 * math.pi)) * x * y, math.sqrt(15 / (4 * math.pi)) * y * z,
                     math.sqrt(5 / (16 * math.pi)) * (2 * z * z - x * x - y * y), math.sqrt(15 / (4 * math.pi)) * x * z,
                     math.sqrt(15 / (16 * math.pi)) * (x * x - y * y)], axis=1)


def test_A_invariant_under_rigid_motion(sys_small_rsh, oracle_small_rsh):
    """Rotate and translate the molecule and rotate the MO coefficients with it: every element of A (hence every eigenvalue)
    must stay put.  Sensitive to any slip in the p / d component order, signs or norms of AO and aux functions."""
    s = sys_small_rsh
    rng = np.random.default_rng(2024)
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(Q) < 0:
        Q[:, 0] = -Q[:, 0]
    u = rng.normal(size=(40, 3))
    Dt = {}
    for l in (0, 1, 2):                                                 # Y(Q^T u) = Y(u) D^T
        Dt[l] = np.linalg.lstsq(_ylm(l, u), _ylm(l, u @ Q), rcond=None)[0]
    C2 = np.array(s["C"], dtype=float).copy()
    off = 0
    for l in np.asarray(s["shl_l"]):
        nf = 2 * int(l) + 1
        C2[off:off + nf] = Dt[int(l)] @ C2[off:off + nf]
        off += nf
    s2 = dict(s); s2["xyz_bohr"] = np.asarray(s["xyz_bohr"]) @ Q.T + np.array([1.5, -2.0, 0.7]); s2["C"] = C2
    A1 = oracle_small_rsh.full_A()
    A2 = ro.Oracle(s2).full_A()
    assert np.abs(C2 - s["C"]).max() > 1e-2
    assert np.abs(A1 - A2).max() < 2e-12
    w1, w2 = np.linalg.eigvalsh(A1)[:8], np.linalg.eigvalsh(A2)[:8]
    assert np.abs(w1 - w2).max() < 1e-12


# ------------------------------------------------------------------ kab_tol (reading G14: conservative screen for the largest oracle cases)
def test_kab_tol_screen_against_unscreened_path():
    """The oracle's primitive-pair screen exp(-mu |AB|^2) < kab_tol, at the value the 300-atom tests use (1e-20), changes no
    integral of the 100-atom system by more than 1e-15 (tolerance of the method: 1e-12); an absurd threshold does, i.e. the
    branch under test is live."""
    s = make_system(2)
    sel = [0, 1, 38, 39, 60, 61]                                        # s and p shells on three atoms along the chain
    for op in ((1.0, 0.0, 0.0), (0.16, 0.84, 0.2)):
        I0 = ro.Oracle(s).int3c(sel, *op)
        I1 = ro.Oracle(s, kab_tol=1e-20).int3c(sel, *op)
        assert np.abs(I1 - I0).max() <= 1e-15
        I2 = ro.Oracle(s, kab_tol=1e-2).int3c(sel, *op)
        assert np.abs(I2 - I0).max() > 1e-6
