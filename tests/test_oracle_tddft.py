"""Pins for oracle/risp_tddft.py (full TDDFT-risp, Eq. 1-2): the symplectic eigenproblem solved by two independent
library routes, elements of B assembled by hand from AO integrals, sigma products against the explicit matrices, the pure-Coulomb
reduction, and the TDA upper bound.  CPU only."""
import numpy as np
import pytest

from oracle.risp_tddft import TddftOracle
from workloads import trial_vectors


@pytest.fixture(scope="module")
def td(sys_small_rsh):
    o = TddftOracle(sys_small_rsh)
    o.build()
    return o


def test_B_symmetric_and_elements_from_the_definition(td):
    o = td
    B = o.full_B()
    assert np.abs(B - B.T).max() < 1e-13
    I3 = o.int3c(o.selJ); I3K = o.int3c(o.selK, o.alpha, o.beta, o.omega)
    MJi = np.linalg.inv(o.int2c(o.selJ)); MKi = np.linalg.inv(o.int2c(o.selK, o.alpha, o.beta, o.omega))
    C = o.C; no = o.nocc
    rng = np.random.default_rng(4)
    occK, virK = set(o.occK.tolist()), set(o.virK.tolist())
    for t in range(8):
        i, j = (int(rng.choice(o.occK)), int(rng.choice(o.occK))) if t < 5 else (int(rng.integers(no)), int(rng.integers(no)))
        a, b = (int(rng.choice(o.virK)), int(rng.choice(o.virK))) if t < 5 else (int(rng.integers(o.nvir)), int(rng.integers(o.nvir)))
        ia = np.einsum('pmn,m,n->p', I3, C[:, i], C[:, no + a]); jb = np.einsum('pmn,m,n->p', I3, C[:, j], C[:, no + b])
        want = 2 * ia @ MJi @ jb
        if i in occK and j in occK and a in virK and b in virK:
            ib = np.einsum('pmn,m,n->p', I3K, C[:, i], C[:, no + b]); ja = np.einsum('pmn,m,n->p', I3K, C[:, j], C[:, no + a])
            want -= ib @ MKi @ ja
        assert B[i * o.nvir + a, j * o.nvir + b] == pytest.approx(want, rel=1e-10, abs=1e-13)


def test_sigma_pm_against_explicit_matrices(td, sys_small_rsh):
    o = td
    X = trial_vectors(sys_small_rsh, 3)
    sp, sm = o.sigma_pm(X)
    A, B = o.full_A(), o.full_B()
    x = X.reshape(3, -1).T
    assert np.linalg.norm((A + B) @ x - sp.reshape(3, -1).T) / np.linalg.norm(sp) < 1e-13
    assert np.linalg.norm((A - B) @ x - sm.reshape(3, -1).T) / np.linalg.norm(sm) < 1e-13
    mask = np.ones_like(X, dtype=bool); mask[np.ix_(np.arange(3), o.occK, o.virK)] = False
    assert np.all(o.exchange2(X)[mask] == 0.0) and np.linalg.norm(o.exchange2(X)) > 0


def test_symplectic_eigenvalues_two_routes_and_tda_bound(td):
    """Omega from (A-B)^(1/2)(A+B)(A-B)^(1/2) equals the positive eigenvalues of the non-symmetric matrix [[A, B], [-B, -A]] of Eq. 1
    (LAPACK geev); X, Y satisfy Eq. 1 and X^T X - Y^T Y = 1; each TDDFT root lies below the corresponding TDA root."""
    o = td
    A, B = o.full_A(), o.full_B()
    n = 6
    om, X, Y = o.tddft_eigenvalues(n)
    dim = A.shape[0]
    big = np.block([[A, B], [-B, -A]])
    ev = np.linalg.eigvals(big)
    assert np.abs(ev.imag).max() < 1e-9
    pos = np.sort(ev.real[ev.real > 0])
    assert np.abs(pos[:n] - om).max() < 1e-9
    x, y = X.reshape(n, dim).T, Y.reshape(n, dim).T
    assert np.abs(A @ x + B @ y - x * om[None]).max() < 1e-10 and np.abs(B @ x + A @ y + y * om[None]).max() < 1e-10
    assert np.abs(np.einsum('dk,dk->k', x, x) - np.einsum('dk,dk->k', y, y) - 1.0).max() < 1e-10
    tda = np.linalg.eigvalsh(A)[:n]
    assert np.all(om <= tda + 1e-12) and np.all(om > 0)


def test_pure_coulomb_reduction(sys_small_rsh):
    """alpha = beta = 0: A - B = Delta is diagonal and Omega^2 = eig(Delta^(1/2) (Delta + 4 J) Delta^(1/2)) -- the textbook RPA form."""
    s = dict(sys_small_rsh); s.update(alpha=0.0, beta=0.0)
    o = TddftOracle(s)
    om, _, _ = o.tddft_eigenvalues(5)
    Bm = o.BiaW.reshape(o.BiaW.shape[0], -1)
    d = o.delta.reshape(-1)
    H = np.sqrt(d)[:, None] * (np.diag(d) + 4 * Bm.T @ Bm) * np.sqrt(d)[None, :]
    assert np.abs(np.sqrt(np.linalg.eigvalsh(H)[:5]) - om).max() < 1e-11
    assert np.abs(o.full_B() - 2 * Bm.T @ Bm).max() < 1e-13
