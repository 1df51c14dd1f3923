"""GPU parity of risp_transition_properties (Eq. 5-8) against oracle/risp_properties.py: the six one-electron AO
matrices element by element on the kept shell pairs, then mu, m, f and R for random vectors and for the solver's own roots."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
HARTREE_EV = 27.211386245988


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    return torch


@pytest.mark.parametrize("which", ["tiny", "rsh"])
def test_oneel_ao_matrices(which, torch_cuda, sys1, sys_small_rsh):
    from paper_2603_29257_b200 import setup
    from oracle.risp_properties import oneel_ao
    s = sys1 if which == "tiny" else sys_small_rsh
    origin = (0.4, -1.2, 0.9)
    c = setup(s)
    try:
        got = c.oneel_ao(origin)
        ref = oneel_ao(s, origin)
        kept = np.zeros((s["nshl"], s["nshl"]), dtype=bool)
        pr = c.stage("PAIRS")
        kept[pr[:, 0], pr[:, 1]] = True; kept[pr[:, 1], pr[:, 0]] = True
        nf = 2 * np.asarray(s["shl_l"]) + 1
        mask = np.repeat(np.repeat(kept, nf, axis=0), nf, axis=1)
        assert np.abs(got - ref)[:, mask].max() <= 1e-12 * max(1.0, np.abs(ref).max())      # values reach |r - O| ~ 20 bohr
        assert np.abs(ref[:, ~mask]).max() < 1e-10 if (~mask).any() else True      # what the pair screen drops is negligible here too
        assert np.abs(got[:, ~mask]).max() == 0.0 if (~mask).any() else True
    finally:
        c.close()


@pytest.mark.parametrize("which", ["tiny", "rsh"])
def test_transition_moments_and_strengths(which, torch_cuda, sys1, sys_small_rsh):
    torch = torch_cuda
    from paper_2603_29257_b200 import setup
    from oracle.risp_properties import transition_moments, strengths
    from workloads import trial_vectors
    s = sys1 if which == "tiny" else sys_small_rsh
    c = setup(s)
    try:
        n = 7
        X = trial_vectors(s, n)
        omega = np.linspace(0.1, 0.3, n)
        for origin, scale in ((None, 0.0), ((1.0, -2.0, 0.5), 1.0)):
            mu, m, f, R = c.transition_properties(torch.from_numpy(X).cuda(), omega, origin=origin, scale=scale)
            mu_r, m_r = transition_moments(s, X, origin=(0, 0, 0) if origin is None else origin, scale=np.sqrt(2.0) if scale == 0.0 else scale)
            f_r, R_r = strengths(omega, mu_r, m_r)
            assert np.abs(mu - mu_r).max() <= 1e-10 * max(1.0, np.abs(mu_r).max())
            assert np.abs(m - m_r).max() <= 1e-10 * max(1.0, np.abs(m_r).max())
            assert np.abs(f - f_r).max() <= 1e-10 * max(1.0, np.abs(f_r).max())
            assert np.abs(R - R_r).max() <= 1e-10 * max(1.0, np.abs(R_r).max())
        # the solver's own roots -> spectrum; vectors are defined up to a sign, f and R are not
        omega, Xr, info = c.tda_solve(5, tol=1e-8, n_guess=5 if which == "tiny" else 0, want_vectors=True)
        mu, m, f, R = c.transition_properties(Xr, omega)
        mu_r, m_r = transition_moments(s, Xr.cpu().numpy())
        f_r, R_r = strengths(omega, mu_r, m_r)
        assert np.abs(f - f_r).max() <= 1e-10 and np.abs(R - R_r).max() <= 1e-10 and np.all(f >= 0)
    finally:
        c.close()


def test_transition_properties_many_states_and_host_vectors(torch_cuda, sys_small_rsh):
    """more states than one contraction chunk (64), and the Ritz vectors of risp_tda_solve delivered to HOST memory"""
    torch = torch_cuda
    from paper_2603_29257_b200 import setup
    from oracle.risp_properties import transition_moments
    from workloads import trial_vectors
    s = sys_small_rsh
    c = setup(s)
    try:
        X = trial_vectors(s, 70)
        mu, m, f, R = c.transition_properties(torch.from_numpy(X).cuda(), np.ones(70))
        mu_r, m_r = transition_moments(s, X)
        assert np.abs(mu - mu_r).max() <= 1e-10 and np.abs(m - m_r).max() <= 1e-10
        om_d, X_d, _ = c.tda_solve(4, tol=1e-8, want_vectors=True, max_block=3)
        om_h, X_h, _ = c.tda_solve(4, tol=1e-8, want_vectors=True, max_block=3, flags=16)
        assert isinstance(X_h, np.ndarray) and np.array_equal(X_h, X_d.cpu().numpy()) and np.array_equal(om_d, om_h)
    finally:
        c.close()
