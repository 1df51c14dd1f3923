"""GPU parity of full TDDFT-risp (Eq. 1-2) against oracle/risp_tddft.py: (A+B) X and (A-B) X element by element,
the whitened T_ia^P' through the (ib|ja) term, and the excitation energies of risp_tddft_solve against the dense symplectic
eigenvalues; restart path; error paths."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
HARTREE_EV = 27.211386245988
FLAG_TDDFT = 8


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    return torch


def _rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


@pytest.fixture(scope="module")
def td_rsh(torch_cuda, sys_small_rsh):
    from paper_2603_29257_b200 import setup
    from oracle.risp_tddft import TddftOracle
    o = TddftOracle(sys_small_rsh)
    o.build()
    c = setup(sys_small_rsh, flags=FLAG_TDDFT)
    yield sys_small_rsh, o, c
    c.close()


@pytest.mark.parametrize("m", [1, 5, 32, 40])
def test_sigma_plus_minus(m, torch_cuda, td_rsh):
    torch = torch_cuda
    from workloads import trial_vectors
    s, o, c = td_rsh
    X = trial_vectors(s, m)
    sp_ref, sm_ref = o.sigma_pm(X)
    sp, sm = c.matvec_tddft(torch.from_numpy(X).cuda())
    assert _rel(sp.cpu().numpy(), sp_ref) <= 1e-10 and _rel(sm.cpu().numpy(), sm_ref) <= 1e-10
    # the exchange pieces separately (the diagonal dominates the norms): K2 = ((A-B) - (A+B))/2 + 2 J ... via the TDA sigma
    sig = c.matvec(torch.from_numpy(X).cuda()).cpu().numpy()          # Delta X + 2 J - K1
    K2 = 0.5 * (sm.cpu().numpy() - sp.cpu().numpy()) + 2.0 * o.coulomb(X)
    assert _rel(K2, o.exchange2(X)) <= 1e-9
    assert _rel(0.5 * (sp.cpu().numpy() + sm.cpu().numpy()), sig) <= 1e-12                            # (A+B + A-B)/2 = A, the TDA operator
    assert _rel(0.5 * (sp.cpu().numpy() + sm.cpu().numpy()), o.delta[None] * X + 2 * o.coulomb(X) - o.exchange(X)) <= 1e-10


def test_sigma_plus_minus_small_chunks_and_tiny_system(torch_cuda, td_rsh, sys1):
    """forced small work-space plans (the (ib|ja) contraction in several aux chunks), and a global hybrid without window (cfg 1)"""
    torch = torch_cuda
    from paper_2603_29257_b200 import setup
    from oracle.risp_tddft import TddftOracle
    from workloads import trial_vectors
    s, o, c = td_rsh
    X = trial_vectors(s, 4)
    sp_ref, sm_ref = o.sigma_pm(X)
    try:
        c.force_plan(2, 24, 1)
        sp, sm = c.matvec_tddft(torch.from_numpy(X).cuda())
        assert _rel(sp.cpu().numpy(), sp_ref) <= 1e-10 and _rel(sm.cpu().numpy(), sm_ref) <= 1e-10
    finally:
        c.force_plan(0, 0, 0)
    o1 = TddftOracle(sys1)
    c1 = setup(sys1, flags=FLAG_TDDFT)
    try:
        X1 = trial_vectors(sys1, 3)
        sp_ref, sm_ref = o1.sigma_pm(X1)
        sp, sm = c1.matvec_tddft(torch.from_numpy(X1).cuda())
        assert _rel(sp.cpu().numpy(), sp_ref) <= 1e-10 and _rel(sm.cpu().numpy(), sm_ref) <= 1e-10
        w, _, _ = o1.tddft_eigenvalues(5)
        omega, Xv, Yv, info = c1.tddft_solve(5, tol=1e-8, n_guess=10, want_vectors=True)
        assert info["converged"] == 1 and np.abs(omega - w).max() * HARTREE_EV <= 1e-6
    finally:
        c1.close()


def test_tddft_roots_and_vectors(torch_cuda, td_rsh):
    torch = torch_cuda
    s, o, c = td_rsh
    n = 6
    w, Xr, Yr = o.tddft_eigenvalues(n)
    omega, X, Y, info = c.tddft_solve(n, tol=1e-8, want_vectors=True)
    assert info["converged"] == 1
    assert np.abs(omega - w).max() * HARTREE_EV <= 1e-6
    x, y = X.cpu().numpy(), Y.cpu().numpy()
    nrm = np.einsum('kia,kia->k', x, x) - np.einsum('kia,kia->k', y, y)
    assert np.abs(nrm - 1.0).max() < 1e-8
    # Eq. 1 with the oracle's matrices: (A+B)(X+Y) = Omega (X-Y), (A-B)(X-Y) = Omega (X+Y)
    sp, _ = o.sigma_pm(x + y)
    _, sm = o.sigma_pm(x - y)
    assert np.linalg.norm((sp - omega[:, None, None] * (x - y)).reshape(n, -1), axis=1).max() < 1e-7
    assert np.linalg.norm((sm - omega[:, None, None] * (x + y)).reshape(n, -1), axis=1).max() < 1e-7
    # below the TDA roots of the same context
    om_tda, _, _ = c.tda_solve(n, tol=1e-8)
    assert np.all(omega <= om_tda + 1e-10)
    # restart path
    omega2, _, _, info2 = c.tddft_solve(3, tol=1e-8, max_sub=18, max_iter=400)
    assert info2["converged"] == 1 and info2["restarts"] > 0
    assert np.abs(omega2 - w[:3]).max() * HARTREE_EV <= 1e-6


def test_tddft_needs_the_setup_flag_and_reports_oom(torch_cuda, sys_small_rsh, td_rsh):
    torch = torch_cuda
    from paper_2603_29257_b200 import setup, RispError
    c = setup(sys_small_rsh)
    try:
        X = torch.zeros((1, c.nocc, c.nvir), dtype=torch.float64, device="cuda")
        with pytest.raises(RispError) as e:
            c.matvec_tddft(X)
        assert e.value.code == -1
        with pytest.raises(RispError):
            c.tddft_solve(2)
    finally:
        c.close()
    _, _, c2 = td_rsh
    c2.tddft_solve(2, tol=1e-6)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    with pytest.raises(RispError) as e:
        c2.tddft_solve(2, device_budget_bytes=4096)
    assert e.value.code == -2
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
