"""Pins for oracle/risp_oneel.c and oracle/risp_properties.py (transition dipoles, oscillator and rotatory strengths, Eq. 5-8,
PAPER.md:73-84): quadrature of the defining integrals with an AO evaluator written here, a closed form, hermiticity, the
origin-shift rules, and the behaviour of f and R under rigid motions and reflections.  CPU only."""
import math

import numpy as np
import pytest

from oracle import risp_oracle as ro
from oracle import risp_properties as rp
from workloads import make_system, trial_vectors
from workloads.generate import normalised_coefs, _radial_norm


def _solid(l, u):
    """unit-normalised real solid harmonics r^l Y_lm in the ABI order (include/risp.h) at the points u[n][3]"""
    x, y, z = u[:, 0], u[:, 1], u[:, 2]
    if l == 0:
        return np.full((len(u), 1), 1 / math.sqrt(4 * math.pi))
    if l == 1:
        return math.sqrt(3 / (4 * math.pi)) * np.stack([x, y, z], axis=1)
    return np.stack([math.sqrt(15 / (4 * math.pi)) * x * y, math.sqrt(15 / (4 * math.pi)) * y * z,
                     math.sqrt(5 / (16 * math.pi)) * (2 * z * z - x * x - y * y), math.sqrt(15 / (4 * math.pi)) * x * z,
                     math.sqrt(15 / (16 * math.pi)) * (x * x - y * y)], axis=1)


def _prim_and_grad(l, a, centre, pts):
    """S_lm(r - A) exp(-a |r - A|^2) and its gradient [n][2l+1][3]; the gradient of the (at most quadratic) polynomial by central
    differences, which are exact for quadratics"""
    u = pts - centre[None]
    g = np.exp(-a * np.sum(u * u, axis=1))
    S = _solid(l, u)
    h = 1e-3
    dS = np.stack([(_solid(l, u + h * np.eye(3)[k][None]) - _solid(l, u - h * np.eye(3)[k][None])) / (2 * h) for k in range(3)], axis=2)
    val = S * g[:, None]
    grad = (dS - 2 * a * u[:, None, :] * S[:, :, None]) * g[:, None, None]
    return val, grad


def _quadrature_block(s, sa, sb, origin, n=26):
    """<mu|(r-O)_k|nu> and <mu|((r-O) x nabla)_k|nu> for the shell pair (sa, sb): Gauss-Hermite product grid per primitive pair"""
    x, w = np.polynomial.hermite.hermgauss(n)
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij")
    W0 = (w[:, None, None] * w[None, :, None] * w[None, None, :]).reshape(-1)
    P0 = np.stack([X.reshape(-1), Y.reshape(-1), Z.reshape(-1)], axis=1)
    la, lb = int(s["shl_l"][sa]), int(s["shl_l"][sb])
    A = s["xyz_bohr"][s["shl_atom"][sa]]; B = s["xyz_bohr"][s["shl_atom"][sb]]
    out = np.zeros((6, 2 * la + 1, 2 * lb + 1))

    def prims(sh, l):
        o, k = int(s["shl_poff"][sh]), int(s["shl_nprim"][sh])
        e = np.asarray(s["prim_exp"][o:o + k]); c = np.asarray(s["prim_coef"][o:o + k])
        return e, normalised_coefs(l, e, c) * _radial_norm(e, l)

    ea, da = prims(sa, la); eb, db = prims(sb, lb)
    for a, ca in zip(ea, da):
        for b, cb in zip(eb, db):
            p = a + b
            P = (a * A + b * B) / p
            pts = P0 / math.sqrt(p) + P[None]
            # weight function of the grid is exp(-p |r - P|^2); the integrand carries exp(-a rA^2 - b rB^2) = K exp(-p rP^2)
            Wt = W0 / p ** 1.5 * np.exp(p * np.sum((pts - P[None]) ** 2, axis=1))
            va, _ = _prim_and_grad(la, a, A, pts)
            vb, gb = _prim_and_grad(lb, b, B, pts)
            r = pts - np.asarray(origin)[None]
            for k in range(3):
                out[k] += ca * cb * np.einsum('n,ni,nj->ij', Wt * r[:, k], va, vb)
            L = np.stack([r[:, 1, None] * gb[:, :, 2] - r[:, 2, None] * gb[:, :, 1],
                          r[:, 2, None] * gb[:, :, 0] - r[:, 0, None] * gb[:, :, 2],
                          r[:, 0, None] * gb[:, :, 1] - r[:, 1, None] * gb[:, :, 0]], axis=0)
            for k in range(3):
                out[3 + k] += ca * cb * np.einsum('n,ni,nj->ij', Wt, va, L[k])
    return out


@pytest.fixture(scope="module")
def small():
    return make_system(3, counts=(6, 4, 1, 1))


def test_oneel_against_quadrature_of_the_definition(small):
    s = small
    origin = (0.3, -0.8, 1.1)
    ao = rp.oneel_ao(s, origin)
    soff = np.concatenate([[0], np.cumsum(2 * np.asarray(s["shl_l"]) + 1)])
    by_l = {l: np.nonzero(np.asarray(s["shl_l"]) == l)[0] for l in (0, 1, 2)}
    rng = np.random.default_rng(8)
    for la in (0, 1, 2):
        for lb in (0, 1, 2):
            for _ in range(2):
                sa, sb = int(rng.choice(by_l[la])), int(rng.choice(by_l[lb]))
                ref = _quadrature_block(s, sa, sb, origin)
                got = ao[:, soff[sa]:soff[sa + 1], soff[sb]:soff[sb + 1]]
                assert np.abs(got - ref).max() < 2e-10 * max(1.0, np.abs(ref).max()), (la, lb, sa, sb)


def test_same_centre_s_px_closed_form():
    """normalised s and p_x Gaussians with one exponent on one centre: <s|x|p_x> = 1/(2 sqrt a), <s|d/dx|p_x> = sqrt a"""
    a = 0.73
    s = dict(natm=1, xyz_bohr=np.array([[0.2, 0.1, -0.4]]), Z=np.array([6], dtype=np.int32), nshl=2, shl_atom=np.array([0, 0], dtype=np.int32),
             shl_l=np.array([0, 1], dtype=np.int32), shl_nprim=np.array([1, 1], dtype=np.int32), shl_poff=np.array([0, 1], dtype=np.int32),
             prim_exp=np.array([a, a]), prim_coef=np.array([1.0, 1.0]), nao=4)
    ao = rp.oneel_ao(s, origin=s["xyz_bohr"][0])
    for k in range(3):
        assert ao[k, 0, 1 + k] == pytest.approx(1 / (2 * math.sqrt(a)), rel=1e-14)
        assert ao[k, 1 + k, 0] == pytest.approx(1 / (2 * math.sqrt(a)), rel=1e-14)
    # L_z p_x = (x d/dy - y d/dx) x f(r) = -y f(r) = -p_y:  <p_y|L_z|p_x> = -1, <p_x|L_z|p_y> = +1
    assert ao[5, 2, 1] == pytest.approx(-1.0, rel=1e-14) and ao[5, 1, 2] == pytest.approx(1.0, rel=1e-14)
    assert abs(ao[5, 1, 1]) < 1e-15 and abs(ao[3, 0, 0]) < 1e-15


def test_hermiticity_and_origin_shift(small):
    s = small
    a0 = rp.oneel_ao(s)
    assert np.abs(a0[:3] - a0[:3].transpose(0, 2, 1)).max() < 1e-13          # r is symmetric
    assert np.abs(a0[3:] + a0[3:].transpose(0, 2, 1)).max() < 1e-13          # r x nabla is real antisymmetric
    S = ro.Oracle(s).overlap()
    O = np.array([1.3, -0.4, 2.2])
    a1 = rp.oneel_ao(s, O)
    for k in range(3):
        assert np.abs(a1[k] - (a0[k] - O[k] * S)).max() < 1e-12               # (r - O)_k = r_k - O_k
    # (r - O) x nabla = r x nabla - O x nabla: the gradient matrices obtained from two different components must agree
    dz_a = -(rp.oneel_ao(s, (0, 1, 0))[3] - a0[3])                            # L_x = y dz - z dy, shift O_y = 1 removes dz
    dz_b = rp.oneel_ao(s, (1, 0, 0))[4] - a0[4]                               # L_y = z dx - x dz, shift O_x = 1 adds dz
    assert np.abs(dz_a - dz_b).max() < 1e-12 and np.abs(dz_a + dz_a.T).max() < 1e-12
    want = a0[3] - (O[1] * dz_a - O[2] * (rp.oneel_ao(s, (0, 0, 1))[3] - a0[3]))
    assert np.abs(a1[3] - want).max() < 1e-11


def _rotate_system(s, Q, shift):
    u = np.random.default_rng(5).normal(size=(40, 3))
    C2 = np.array(s["C"], dtype=float).copy()
    off = 0
    for l in np.asarray(s["shl_l"]):
        nf = 2 * int(l) + 1
        Dt = np.linalg.lstsq(_solid(int(l), u), _solid(int(l), u @ Q), rcond=None)[0]
        C2[off:off + nf] = Dt @ C2[off:off + nf]
        off += nf
    s2 = dict(s); s2["xyz_bohr"] = np.asarray(s["xyz_bohr"]) @ Q.T + shift; s2["C"] = C2
    return s2


def test_strengths_under_rigid_motion_and_reflection(small):
    """mu and m rotate like vectors, so f (Eq. 5) and R (Eq. 6) are invariant under a rigid rotation; a reflection keeps f and
    flips the sign of the rotatory strength (a pseudoscalar); mu does not depend on the gauge origin for orthonormal MOs."""
    s = small
    X = trial_vectors(s, 4)
    omega = np.array([0.1, 0.12, 0.15, 0.2])
    mu, m = rp.transition_moments(s, X)
    f, R = rp.strengths(omega, mu, m)
    assert np.all(f > 0) and np.abs(R).max() > 1e-6
    rng = np.random.default_rng(31)
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(Q) < 0:
        Q[:, 0] = -Q[:, 0]
    mu2, m2 = rp.transition_moments(_rotate_system(s, Q, np.zeros(3)), X)
    assert np.abs(mu2 - mu @ Q.T).max() < 1e-11 and np.abs(m2 - m @ Q.T).max() < 1e-11
    f2, R2 = rp.strengths(omega, mu2, m2)
    assert np.abs(f2 - f).max() < 1e-12 and np.abs(R2 - R).max() < 1e-12
    M = np.diag([1.0, 1.0, -1.0])                                              # mirror z -> -z
    mu3, m3 = rp.transition_moments(_rotate_system(s, M, np.zeros(3)), X)
    f3, R3 = rp.strengths(omega, mu3, m3)
    assert np.abs(f3 - f).max() < 1e-12 and np.abs(R3 + R).max() < 1e-12
    mu4, _ = rp.transition_moments(s, X, origin=(5.0, -3.0, 1.0))
    assert np.abs(mu4 - mu).max() < 1e-9                                        # <i|a> = 0: C^T S C = 1 to 1e-11 in the generator
    # Eq. 5-6 written out for one state
    assert f[1] == pytest.approx(2 / 3 * omega[1] * float(mu[1] @ mu[1]), rel=1e-14)
    assert R[2] == pytest.approx(0.5 * float(mu[2] @ m[2]), rel=1e-14)
    mu1, _ = rp.transition_moments(s, X, scale=1.0)
    assert np.abs(mu1 * math.sqrt(2.0) - mu).max() < 1e-14                      # reading G24: closed-shell singlet factor
