"""Pins for oracle/risp_integrals.c -- the oracle is checked against things other than itself:
closed forms, quadrature of the defining integrals, derivative identities, printed values
(tests/golden/), invariances.  CPU only."""
import math
import os

import numpy as np
import pytest
from scipy.special import erf

from oracle import risp_oracle as ro

GOLD = os.path.join(os.path.dirname(__file__), "golden")
A0, a0 = np.array([0.1, -0.3, 0.2]), 0.8
B0, b0 = np.array([0.9, 0.4, -0.5]), 1.3
C0, g0 = np.array([-0.7, 1.1, 0.6]), 0.17


def _gold(name):
    rows = []
    for line in open(os.path.join(GOLD, name)):
        line = line.split("#")[0].split()
        if line:
            rows.append(line)
    return rows


# ------------------------------------------------------------------ Boys function (Eq. 3 needs it)
@pytest.mark.parametrize("x", [1e-9, 0.003, 0.5, 3.7, 12.0, 34.9, 35.0, 36.2, 80.0, 400.0])
def test_boys_closed_forms(x):
    F = ro.boys(6, x)
    assert F[0] == pytest.approx(0.5 * math.sqrt(math.pi / x) * erf(math.sqrt(x)), rel=2e-15)
    for n in range(6, 0, -1):                                        # F_{n-1} = (2x F_n + e^-x)/(2n-1)
        assert F[n - 1] == pytest.approx((2 * x * F[n] + math.exp(-x)) / (2 * n - 1), rel=1e-14)


def test_boys_at_zero():
    F = ro.boys(6, 0.0)
    for n in range(7):
        assert F[n] == pytest.approx(1.0 / (2 * n + 1), rel=1e-15)


@pytest.mark.parametrize("x", [0.2, 5.0, 20.0, 34.0, 36.0, 60.0])
def test_boys_quadrature(x):
    t, w = np.polynomial.legendre.leggauss(200)
    t = 0.5 * (t + 1); w = 0.5 * w
    F = ro.boys(6, x)
    for n in range(7):
        assert F[n] == pytest.approx(float(np.sum(w * t ** (2 * n) * np.exp(-x * t * t))), rel=1e-13)


def test_boys_golden():
    for r in _gold("boys_and_prim3c.txt"):
        if r[0] == "boys":
            n, x, v = int(r[1]), float(r[2]), float(r[3])
            assert ro.boys(n, x)[n] == pytest.approx(v, rel=2e-15)


# ------------------------------------------------------------------ primitive integrals
def test_prim3c_golden():
    for r in _gold("boys_and_prim3c.txt"):
        if r[0] == "prim3c":
            la, lb, lc = ([int(c) for c in s] for s in r[1:4])
            assert ro.prim3c(a0, A0, la, b0, B0, lb, g0, C0, lc) == pytest.approx(float(r[4]), rel=3e-15)
            assert ro.prim3c(a0, A0, la, b0, B0, lb, g0, C0, lc, 0.0, 1.0, 0.2) == pytest.approx(float(r[5]), rel=3e-15)


def _sss_closed(a, A, b, B, g, C, ca, cb, w):
    """(s_a s_b|s_c) = 2 pi^{5/2}/(p g sqrt(p+g)) e^{-mu AB^2} [ca F0(al R^2) + cb sqrt(at/al) F0(at R^2)]."""
    p = a + b; mu = a * b / p
    P = (a * A + b * B) / p
    R2 = float(np.sum((P - C) ** 2)); AB2 = float(np.sum((A - B) ** 2))
    al = p * g / (p + g)
    F0 = lambda x: 1.0 if x == 0 else 0.5 * math.sqrt(math.pi / x) * erf(math.sqrt(x))
    v = ca * F0(al * R2)
    if cb:
        at = 1.0 / (1.0 / al + 1.0 / (w * w))
        v += cb * math.sqrt(at / al) * F0(at * R2)
    return 2 * math.pi ** 2.5 / (p * g * math.sqrt(p + g)) * math.exp(-mu * AB2) * v


@pytest.mark.parametrize("op", [(1.0, 0.0, 0.0), (0.0, 1.0, 0.2), (0.16, 0.84, 0.2), (0.3, 0.5, 1.7)])
def test_sss_closed_form(op):
    z = [0, 0, 0]
    rng = np.random.default_rng(5)
    for _ in range(20):
        A, B, C = rng.normal(size=(3, 3)) * 2
        a, b, g = rng.uniform(0.1, 5.0, size=3)
        assert ro.prim3c(a, A, z, b, B, z, g, C, z, *op) == pytest.approx(_sss_closed(a, A, b, B, g, C, *op), rel=1e-13)


def _potential(lc, g, C, pts, ca, cb, w):
    """V(r) = int G_c(r') (ca + cb erf(w|r-r'|))/|r-r'| dr' for an unnormalised s or p_x/y/z aux Gaussian (closed form)."""
    d = pts - C[None, :]
    R = np.linalg.norm(d, axis=1)
    out = np.zeros(len(pts))
    for coef, s2 in ((ca, g), (cb, g * w * w / (g + w * w) if cb else 0.0)):
        if coef == 0:
            continue
        s = math.sqrt(s2)
        f = erf(s * R) / R
        if sum(lc) == 0:
            out += coef * (math.pi / g) ** 1.5 * f
        else:                                                          # x e^{-g r^2} = (1/2g) d/dC_x e^{-g r^2}
            k = lc.index(1)
            fp = 2 * s / math.sqrt(math.pi) * np.exp(-s2 * R * R) / R - erf(s * R) / (R * R)
            out += coef * (math.pi / g) ** 1.5 / (2 * g) * fp * (-d[:, k] / R)
    return out


CASES = [([0, 0, 0], [0, 0, 0]), ([1, 0, 0], [0, 0, 0]), ([0, 1, 0], [0, 0, 1]), ([2, 0, 0], [0, 0, 0]), ([1, 1, 0], [0, 1, 0]),
         ([0, 0, 2], [1, 0, 0]), ([1, 0, 1], [0, 2, 0]), ([2, 0, 0], [0, 1, 1]), ([0, 1, 1], [1, 0, 1])]


@pytest.mark.parametrize("la,lb", CASES)
@pytest.mark.parametrize("lc", [[0, 0, 0], [1, 0, 0], [0, 1, 0], [0, 0, 1]])
@pytest.mark.parametrize("op", [(1.0, 0.0, 0.0), (0.16, 0.84, 0.2)])
def test_prim3c_vs_quadrature_of_definition(la, lb, lc, op):
    """(ab|c) = int rho_ab(r) V_c(r) dr, Gauss-Hermite product grid on the pair Gaussian."""
    n = 48
    x, wq = np.polynomial.hermite.hermgauss(n)
    p = a0 + b0
    P = (a0 * A0 + b0 * B0) / p
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij")
    W = (wq[:, None, None] * wq[None, :, None] * wq[None, None, :]).reshape(-1) / p ** 1.5
    pts = np.stack([X.reshape(-1), Y.reshape(-1), Z.reshape(-1)], axis=1) / math.sqrt(p) + P[None]
    poly = np.ones(len(pts))
    for k in range(3):
        poly *= (pts[:, k] - A0[k]) ** la[k] * (pts[:, k] - B0[k]) ** lb[k]
    pref = math.exp(-a0 * b0 / p * float(np.sum((A0 - B0) ** 2)))
    ref = pref * float(np.sum(W * poly * _potential(lc, g0, C0, pts, *op)))
    got = ro.prim3c(a0, A0, la, b0, B0, lb, g0, C0, lc, *op)
    assert got == pytest.approx(ref, rel=1e-9, abs=1e-11)


def test_p_and_d_by_derivative_identity():
    """x e^{-a r^2} = (1/2a) d/dA_x e^{-a r^2}: central differences of the lower class."""
    h = 1e-4
    z = [0, 0, 0]
    for k in range(3):
        e = np.zeros(3); e[k] = h
        lk = [0, 0, 0]; lk[k] = 1
        for op in ((1.0, 0.0, 0.0), (0.16, 0.84, 0.2)):
            fd = (ro.prim3c(a0, A0 + e, z, b0, B0, z, g0, C0, z, *op) - ro.prim3c(a0, A0 - e, z, b0, B0, z, g0, C0, z, *op)) / (2 * h)
            assert ro.prim3c(a0, A0, lk, b0, B0, z, g0, C0, z, *op) == pytest.approx(fd / (2 * a0), rel=1e-7)
            fd = (ro.prim3c(a0, A0, z, b0, B0, z, g0, C0 + e, z, *op) - ro.prim3c(a0, A0, z, b0, B0, z, g0, C0 - e, z, *op)) / (2 * h)
            assert ro.prim3c(a0, A0, z, b0, B0, z, g0, C0, lk, *op) == pytest.approx(fd / (2 * g0), rel=1e-7)
            # x^2 e^{-b r^2} = (1/2b) d/dB_x (x e^{-b r^2}) + (1/2b) e^{-b r^2}
            l2 = [0, 0, 0]; l2[k] = 2
            fd = (ro.prim3c(a0, A0, z, b0, B0 + e, lk, g0, C0, z, *op) - ro.prim3c(a0, A0, z, b0, B0 - e, lk, g0, C0, z, *op)) / (2 * h)
            want = fd / (2 * b0) + ro.prim3c(a0, A0, z, b0, B0, z, g0, C0, z, *op) / (2 * b0)
            assert ro.prim3c(a0, A0, z, b0, B0, l2, g0, C0, z, *op) == pytest.approx(want, rel=1e-7)


def test_3c_reduces_to_2c():
    """Two s primitives on one centre are one s primitive: (s_a s_b|P) = (s_{a+b}|P)."""
    for lc in ([0, 0, 0], [0, 1, 0]):
        for op in ((1.0, 0.0, 0.0), (0.16, 0.84, 0.2)):
            v3 = ro.prim3c(a0, A0, [0, 0, 0], b0, A0, [0, 0, 0], g0, C0, lc, *op)
            v2 = ro.prim2c(a0 + b0, A0, [0, 0, 0], g0, C0, lc, *op)
            assert v3 == pytest.approx(v2, rel=1e-14)


def test_2c_symmetric_and_pp_by_derivative():
    h = 1e-4
    for op in ((1.0, 0.0, 0.0), (0.16, 0.84, 0.2)):
        for lc in ([1, 0, 0], [0, 0, 1]):
            for ld in ([0, 1, 0], [0, 0, 1]):
                v = ro.prim2c(g0, C0, lc, 0.3, B0, ld, *op)
                assert v == pytest.approx(ro.prim2c(0.3, B0, ld, g0, C0, lc, *op), rel=1e-14)
                e = np.zeros(3); e[ld.index(1)] = h
                fd = (ro.prim2c(g0, C0, lc, 0.3, B0 + e, [0, 0, 0], *op) - ro.prim2c(g0, C0, lc, 0.3, B0 - e, [0, 0, 0], *op)) / (2 * h)
                assert v == pytest.approx(fd / (2 * 0.3), rel=1e-7)


def test_metric_diagonal_closed_form(sys1):
    """Normalised s: (P|P) = 4 pi/g (Coulomb), (4 pi/g)[alpha + beta sqrt(a_eff/a_c)] (RSH); golden numbers from SURVEY B.3."""
    gold = {r[0]: float(r[1]) for r in _gold("metric_c6.txt")}
    g = 0.2 / (4 / 3.25) ** 2
    assert g == pytest.approx(0.13203125)
    o = ro.Oracle(sys1)
    s_sel = [int(o.selK[0])]
    assert o.aux_exp[s_sel[0]] == pytest.approx(g)
    assert o.int2c(s_sel)[0, 0] == pytest.approx(gold["ss_coulomb"], rel=1e-14)
    assert o.int2c(s_sel, 0.16, 0.84, 0.2)[0, 0] == pytest.approx(gold["ss_rsh"], rel=1e-14)
    assert gold["ss_coulomb"] == pytest.approx(4 * math.pi / g, rel=1e-15)
    ac = g / 2; ae = 1 / (2 / g + 1 / 0.04)
    assert gold["ss_rsh"] == pytest.approx(4 * math.pi / g * (0.16 + 0.84 * math.sqrt(ae / ac)), rel=1e-14)


# ------------------------------------------------------------------ contracted, spherical, normalised
def test_overlap_normalisation_and_generator_agreement(sys1):
    """S_mumu = 1, components of one shell are orthonormal, and the MOs the generator made (with its own
    overlap code) are orthonormal under the oracle's S: two independent codings of the AO conventions agree."""
    o = ro.Oracle(sys1)
    S = o.overlap()
    assert np.allclose(np.diag(S), 1.0, atol=1e-14)
    off = 0
    for l in o.shl_l:
        nf = 2 * l + 1
        assert np.allclose(S[off:off + nf, off:off + nf], np.eye(nf), atol=1e-14)
        off += nf
    assert np.abs(sys1["C"].T @ S @ sys1["C"] - np.eye(o.nao)).max() < 1e-11


def test_int3c_symmetry_translation_rotation(sys1):
    o = ro.Oracle(sys1)
    sel = o.selJ[:4]
    full = o.int3c(sel, full_square=True)
    assert np.abs(full - full.transpose(0, 2, 1)).max() < 1e-14          # (mu nu|P) = (nu mu|P), both computed
    assert np.abs(full - o.int3c(sel)).max() < 1e-15
    # rigid motion: every shell-triple block keeps its Frobenius norm; s-type blocks keep their values
    rng = np.random.default_rng(3)
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    s2 = dict(sys1); s2["xyz_bohr"] = sys1["xyz_bohr"] @ Q.T + np.array([3.0, -1.0, 2.5])
    o2 = ro.Oracle(s2)
    for op in ((1.0, 0.0, 0.0), (0.16, 0.84, 0.2)):
        I1, I2 = o.int3c(sel, *op), o2.int3c(sel, *op)
        aoff = np.concatenate([[0], np.cumsum(2 * o.aux_l[sel] + 1)])
        soff = np.concatenate([[0], np.cumsum(2 * o.shl_l + 1)])
        for q in range(len(sel)):
            for sa in range(0, o.nshl, 5):
                for sb in range(0, o.nshl, 7):
                    b1 = I1[aoff[q]:aoff[q + 1], soff[sa]:soff[sa + 1], soff[sb]:soff[sb + 1]]
                    b2 = I2[aoff[q]:aoff[q + 1], soff[sa]:soff[sa + 1], soff[sb]:soff[sb + 1]]
                    assert np.linalg.norm(b1) == pytest.approx(np.linalg.norm(b2), rel=1e-11, abs=1e-13)
                    if b1.size == 1:
                        assert b1.item() == pytest.approx(b2.item(), rel=1e-11, abs=1e-13)


def test_contracted_sss_against_closed_form(sys1):
    """A contracted normalised (s s|s) element re-assembled in Python from the closed form."""
    o = ro.Oracle(sys1)
    from workloads.generate import normalised_coefs, _radial_norm
    sa, sb = 0, 1                                                      # carbon s1 (5 primitives), s2
    assert o.shl_l[sa] == 0 and o.shl_l[sb] == 0
    P = int(o.selK[2]); g = o.aux_exp[P]; C = o.xyz[o.aux_atom[P]]
    I = o.int3c([P], 0.16, 0.84, 0.2)
    tot = 0.0
    ea = o.pe[o.shl_poff[sa]:o.shl_poff[sa] + o.shl_nprim[sa]]; eb = o.pe[o.shl_poff[sb]:o.shl_poff[sb] + o.shl_nprim[sb]]
    ca = normalised_coefs(0, ea, o.pc[o.shl_poff[sa]:o.shl_poff[sa] + o.shl_nprim[sa]]) * _radial_norm(ea, 0)
    cb = normalised_coefs(0, eb, o.pc[o.shl_poff[sb]:o.shl_poff[sb] + o.shl_nprim[sb]]) * _radial_norm(eb, 0)
    for k, a in enumerate(ea):
        for q, b in enumerate(eb):
            tot += ca[k] * cb[q] * _sss_closed(a, o.xyz[o.shl_atom[sa]], b, o.xyz[o.shl_atom[sb]], g, C, 0.16, 0.84, 0.2)
    tot *= (1 / math.sqrt(4 * math.pi)) ** 2 * (2 * g / math.pi) ** 0.75
    assert I[0, 0, 1] == pytest.approx(tot, rel=1e-13)
