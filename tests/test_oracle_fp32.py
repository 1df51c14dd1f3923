"""Pins for oracle/risp_fp32.py (the paper's single-precision mode of Eq. 22-23): the binary32 contraction
lies inside the textbook forward error bound of an inner product around the FP64 exchange, is exact where binary32 arithmetic is
exact (small dyadic inputs), is not the FP64 result in disguise, and vanishes outside the exchange window.  CPU only."""
import numpy as np
import pytest

from oracle.risp_oracle import Oracle
from oracle.risp_fp32 import exchange_fp32, exchange_error_bound, U32
from workloads import trial_vectors


@pytest.fixture(scope="module")
def orc(sys_small_rsh):
    o = Oracle(sys_small_rsh)
    o.build()
    return o


def test_inside_the_forward_error_bound_and_not_fp64(orc, sys_small_rsh):
    X = trial_vectors(sys_small_rsh, 4)
    K64, K32 = orc.exchange(X), exchange_fp32(orc, X)
    bound = exchange_error_bound(orc, X)
    err = np.abs(K32 - K64)
    assert np.all(err <= bound + 1e-300)
    rel = np.linalg.norm(K32 - K64) / np.linalg.norm(K64)
    assert 1e-9 < rel < 1e-5            # really rounded to binary32 (an FP64 copy would give 0), and no worse than a few thousand ulps
    mask = np.ones_like(X, dtype=bool); mask[np.ix_(np.arange(4), orc.occK, orc.virK)] = False
    assert np.all(K32[mask] == 0.0)


def test_exact_on_small_dyadic_inputs(orc):
    """Integers below 2^6 times a power of two: every product and partial sum of Eq. 22-23 stays below 2^24 in units of the common
    scale, so binary32 commits no rounding and the two precisions must agree bit for bit."""
    rng = np.random.default_rng(11)
    o = orc
    keepij, keepab = o.BijW, o.BabW
    try:
        nP = min(4, keepij.shape[0])
        o.BijW = rng.integers(-3, 4, size=(nP,) + keepij.shape[1:]).astype(np.float64) * 2.0 ** -3
        o.BabW = rng.integers(-3, 4, size=(nP,) + keepab.shape[1:]).astype(np.float64) * 2.0 ** -5
        for P in range(nP):
            o.BijW[P] = np.tril(o.BijW[P]) + np.tril(o.BijW[P], -1).T
            o.BabW[P] = np.tril(o.BabW[P]) + np.tril(o.BabW[P], -1).T
        X = rng.integers(-3, 4, size=(2, o.nocc, o.nvir)).astype(np.float64) * 2.0 ** -2
        K64, K32 = o.exchange(X), exchange_fp32(o, X)
        assert np.abs(K64).max() > 0
        assert np.array_equal(K64, K32)
    finally:
        o.BijW, o.BabW = keepij, keepab


def test_bound_scales_with_unit_roundoff(orc, sys_small_rsh):
    X = trial_vectors(sys_small_rsh, 2)
    b = exchange_error_bound(orc, X)
    n = len(orc.virK) + len(orc.occK) + orc.BijW.shape[0] + 3
    ref = np.zeros_like(X)
    Xw = np.abs(X[:, orc.occK][:, :, orc.virK])
    acc = np.zeros_like(Xw)
    for P in range(orc.BijW.shape[0]):
        acc += np.einsum('ij,mjb,ab->mia', np.abs(orc.BijW[P]), Xw, np.abs(orc.BabW[P]))
    ref[np.ix_(np.arange(2), orc.occK, orc.virK)] = acc
    assert np.allclose(b, ref * n * U32 / (1 - n * U32), rtol=1e-12, atol=0)
