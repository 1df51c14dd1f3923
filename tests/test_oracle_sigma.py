"""Pins for oracle/risp_oracle.py (sigma-build, explicit A, Davidson) -- invariants, limits, brute force.  CPU only."""
import numpy as np
import pytest

from oracle.risp_oracle import Oracle, HARTREE_EV
from workloads import trial_vectors, make_system


def test_metrics_positive_definite(oracle1, oracle_small_rsh):
    for o in (oracle1, oracle_small_rsh):
        for M in (o.MJ, o.MK):
            assert np.abs(M - M.T).max() < 1e-13
            assert np.linalg.eigvalsh(M)[0] > 0
    assert oracle1.MJ.shape[0] == 4 * oracle1.MK.shape[0]              # N_auxJ = 4 N_auxK


def test_J_ao_direct_equals_mo_route(sys1, oracle1):
    """Eq. 11-17 (on-the-fly order) reproduce J from the explicit (ia|P) tensor."""
    X = trial_vectors(sys1)
    J_mo = oracle1.coulomb(X)
    J_ao = oracle1.coulomb_ao_direct(X)
    assert np.linalg.norm(J_ao - J_mo) / np.linalg.norm(J_mo) < 1e-11
    # and J is what Eq. 13 says: sum_jb sum_PQ (ia|P) (P|Q)^-1 (Q|jb) X_jb with the plain inverse
    B = oracle1.Bia.reshape(oracle1.Bia.shape[0], -1)
    J_inv = (B.T @ np.linalg.inv(oracle1.MJ) @ B @ X.reshape(X.shape[0], -1).T).T.reshape(X.shape)
    assert np.linalg.norm(J_inv - J_mo) / np.linalg.norm(J_mo) < 1e-11


def test_K_metric_placement(oracle_small_rsh, sys_small_rsh):
    """Eq. 20-21 as printed (whole inverse metric on T_ij, reading G3) equals the symmetric whitening the oracle uses."""
    o = oracle_small_rsh
    X = trial_vectors(sys_small_rsh, 3)
    K = o.exchange(X)
    Tij = np.einsum('qij,qp->pij', o.Bij, np.linalg.inv(o.MK))          # Eq. 20
    Tab = o.Bab                                                         # Eq. 21
    Xw = X[:, o.occK][:, :, o.virK]
    M = np.einsum('pab,mjb->pmja', Tab, Xw)                             # Eq. 22
    Kw = np.einsum('pij,pmja->mia', Tij, M)                             # Eq. 23
    K2 = np.zeros_like(X); K2[np.ix_(np.arange(3), o.occK, o.virK)] = Kw
    assert np.linalg.norm(K2 - K) / np.linalg.norm(K) < 1e-11
    assert len(o.occK) < o.nocc and len(o.virK) < o.nvir                # the window really truncates here
    mask = np.ones_like(K, dtype=bool); mask[np.ix_(np.arange(3), o.occK, o.virK)] = False
    assert np.all(K[mask] == 0.0)                                       # reading G7: K is zero outside the window


@pytest.mark.parametrize("which", ["tiny", "rsh"])
def test_A_symmetric_and_matches_sigma(which, sys1, oracle1, sys_small_rsh, oracle_small_rsh):
    s, o = (sys1, oracle1) if which == "tiny" else (sys_small_rsh, oracle_small_rsh)
    A = o.full_A()
    assert np.abs(A - A.T).max() < 1e-13
    X = trial_vectors(s, 4)
    sig = o.sigma(X)
    assert np.linalg.norm(A @ X.reshape(4, -1).T - sig.reshape(4, -1).T) / np.linalg.norm(sig) < 1e-13
    # sigma of a unit vector is a column of A
    dim = o.nocc * o.nvir
    for jb in (0, dim // 3, dim - 1):
        e = np.zeros((1, dim)); e[0, jb] = 1.0
        assert np.abs(o.sigma(e.reshape(1, o.nocc, o.nvir)).reshape(-1) - A[:, jb]).max() < 1e-13


def test_A_elements_from_the_definition(oracle1):
    """A few elements of Eq. 10 assembled by hand from AO integrals and the plain inverse metrics."""
    o = oracle1
    I3 = o.int3c(o.selJ); I3K = o.int3c(o.selK, o.alpha, o.beta, o.omega)
    MJi = np.linalg.inv(o.int2c(o.selJ)); MKi = np.linalg.inv(o.int2c(o.selK, o.alpha, o.beta, o.omega))
    A = o.full_A()
    C = o.C; no = o.nocc
    rng = np.random.default_rng(11)
    for _ in range(6):
        i, j = rng.integers(no, size=2); a, b = rng.integers(o.nvir, size=2)
        ia = np.einsum('pmn,m,n->p', I3, C[:, i], C[:, no + a]); jb = np.einsum('pmn,m,n->p', I3, C[:, j], C[:, no + b])
        ij = np.einsum('pmn,m,n->p', I3K, C[:, i], C[:, j]); ab = np.einsum('pmn,m,n->p', I3K, C[:, no + a], C[:, no + b])
        want = 2 * ia @ MJi @ jb - ij @ MKi @ ab
        if i == j and a == b:
            want += o.eps[no + a] - o.eps[i]
        assert A[i * o.nvir + a, j * o.nvir + b] == pytest.approx(want, rel=1e-10, abs=1e-13)


def test_cutoff_limits(sys_small_rsh):
    """cutoff = +inf reproduces the untruncated K; a cutoff below every |eps| empties the window, K = 0."""
    X = trial_vectors(sys_small_rsh, 2)
    s_inf = dict(sys_small_rsh); s_inf["cutoff_ev"] = float("inf")
    s_big = dict(sys_small_rsh); s_big["cutoff_ev"] = 1e6
    K_inf, K_big = Oracle(s_inf).exchange(X), Oracle(s_big).exchange(X)
    assert np.array_equal(K_inf, K_big) and np.linalg.norm(K_inf) > 0
    s_0 = dict(sys_small_rsh); s_0["cutoff_ev"] = 0.5 * float(np.min(np.abs(sys_small_rsh["eps"]))) * HARTREE_EV
    o0 = Oracle(s_0)
    assert len(o0.occK) == 0 or len(o0.virK) == 0
    assert np.all(o0.exchange(X) == 0.0)
    # a window that keeps everything by energy equals no truncation
    K_cut = Oracle(sys_small_rsh).exchange(X)
    assert np.linalg.norm(K_cut - K_inf) > 1e-6 * np.linalg.norm(K_inf)   # 40 eV does cut in this system


def test_operator_limits(sys_small_rsh):
    """beta = 0 is the global hybrid; omega -> large makes J^ -> (alpha+beta)/r."""
    X = trial_vectors(sys_small_rsh, 2)
    s_a = dict(sys_small_rsh); s_a.update(alpha=1.0, beta=0.0, omega=0.0)
    s_b = dict(sys_small_rsh); s_b.update(alpha=0.16, beta=0.84, omega=1e3)
    Ka, Kb = Oracle(s_a).exchange(X), Oracle(s_b).exchange(X)
    assert np.linalg.norm(Ka - Kb) / np.linalg.norm(Ka) < 1e-5
    s_c = dict(sys_small_rsh); s_c.update(alpha=0.25, beta=0.0, omega=0.7)
    Kc = Oracle(s_c).exchange(X)
    assert np.linalg.norm(Kc - 0.25 * Ka) / np.linalg.norm(Kc) < 1e-12   # K is linear in a_x: c_x (ij|ab) of Eq. 10


def test_2J_positive_semidefinite(sys1):
    s = dict(sys1); s.update(alpha=0.0, beta=0.0)
    o = Oracle(s)
    w = np.linalg.eigvalsh(o.full_A())
    assert w[0] >= o.delta.min() - 1e-12


def _jacobi_eigvals(A, sweeps=30):
    A = A.copy(); n = len(A)
    for _ in range(sweeps):
        for p in range(n - 1):
            for q in range(p + 1, n):
                if abs(A[p, q]) < 1e-300:
                    continue
                th = 0.5 * np.arctan2(2 * A[p, q], A[q, q] - A[p, p])
                c, s = np.cos(th), np.sin(th)
                R = np.eye(n); R[p, p] = c; R[q, q] = c; R[p, q] = s; R[q, p] = -s
                A = R.T @ A @ R
    return np.sort(np.diag(A))


def test_dense_eigensolver_against_jacobi():
    rng = np.random.default_rng(2)
    M = rng.normal(size=(30, 30)); M = M + M.T
    assert np.abs(np.linalg.eigvalsh(M) - _jacobi_eigvals(M)).max() < 1e-11


@pytest.mark.parametrize("which", ["tiny", "rsh"])
def test_davidson_roots_equal_brute_force(which, oracle1, oracle_small_rsh):
    o = oracle1 if which == "tiny" else oracle_small_rsh
    n = 5
    w = np.linalg.eigvalsh(o.full_A())[:n]
    th, X, info = o.davidson(n, n_guess=n if which == "tiny" else None, tol=1e-8)
    assert info["converged"]
    assert np.abs(th - w).max() < 1e-10
    sig = o.sigma(X)
    assert np.abs(np.linalg.norm((sig - th[:, None, None] * X).reshape(n, -1), axis=1)).max() < 1e-7


def test_davidson_restart_path(oracle1):
    w = np.linalg.eigvalsh(oracle1.full_A())[:3]
    th, X, info = oracle1.davidson(3, tol=1e-8, max_sub=30, max_iter=300)
    assert info["restarts"] > 0 and info["converged"]
    assert np.abs(th - w).max() < 1e-10


def test_generator_shapes_and_determinism():
    s = make_system(1); s2 = make_system(1)
    assert (s["nao"], s["nocc"], s["nvir"], s["natm"]) == (154, 25, 129, 20)
    assert np.array_equal(s["C"], s2["C"]) and np.array_equal(s["xyz_bohr"], s2["xyz_bohr"])
    assert np.all(np.diff(s["eps"][:25]) >= 0) and np.all(np.diff(s["eps"][25:]) >= 0)
    assert not np.any(np.asarray(s["Z"])[s["aux_atom"]] == 1)          # hydrogen-free aux basis
    X = trial_vectors(s)
    G = X.reshape(5, -1) @ X.reshape(5, -1).T
    assert np.abs(G - np.eye(5)).max() < 1e-13
