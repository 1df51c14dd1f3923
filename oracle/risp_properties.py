"""ORACLE -- test infrastructure, not product code.

Transition properties of TDA-risp excited states (arxiv/paper_2603_29257 Eq. 5-8), plain numpy on top of the
one-electron integrals of oracle/risp_oneel.c:

    mu_0n = scale * sum_ia r_ia X_nia                         (Eq. 7 with Y = 0, "in TDA one sets Y = 0")
    m_0n  = scale * sum_ia (r x nabla)_ia X_nia               (Eq. 8 with Y = 0)
    f_0n  = 2/3 Omega_n mu_0n . mu_0n                         (Eq. 5)
    R_0n  = 1/2 mu_0n . m_0n                                  (Eq. 6)

`scale` is DESIGN.md reading G24: the paper prints no spin factor; for a closed-shell singlet and <X|X> = 1 (what
risp_tda_solve returns) the moments carry sqrt(2), which is the default here and in the CUDA path.
Only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import this module.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None
_D, _I = ctypes.c_double, ctypes.c_int


def build_lib(force: bool = False) -> str:
    src = os.path.join(_HERE, "risp_oneel.c")
    so = os.path.join(_HERE, "librisp_oracle_oneel.so")
    if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", so, src, "-lm"])
    return so


def _lib():
    global _LIB
    if _LIB is None:
        _LIB = ctypes.CDLL(build_lib())
    return _LIB


def _p(a, t):
    return a.ctypes.data_as(ctypes.POINTER(t))


def oneel_ao(sys: dict, origin=(0.0, 0.0, 0.0)) -> np.ndarray:
    """[6][nao][nao]: <mu|(r-O)_k|nu> (k = x, y, z), then <mu|((r-O) x nabla)_k|nu>."""
    f64 = lambda k: np.ascontiguousarray(sys[k], dtype=np.float64)
    i32 = lambda k: np.ascontiguousarray(sys[k], dtype=np.int32)
    xyz, pe, pc = f64("xyz_bohr"), f64("prim_exp"), f64("prim_coef")
    sa, sl, sn, so = i32("shl_atom"), i32("shl_l"), i32("shl_nprim"), i32("shl_poff")
    nao = int(sys["nao"])
    out = np.zeros((6, nao, nao))
    org = np.ascontiguousarray(origin, dtype=np.float64)
    _lib().oracle_oneel(_p(xyz, _D), _I(len(sl)), _p(sa, _I), _p(sl, _I), _p(sn, _I), _p(so, _I), _p(pe, _D), _p(pc, _D), _p(org, _D), _p(out, _D))
    return out


def transition_moments(sys: dict, X: np.ndarray, origin=(0.0, 0.0, 0.0), scale: float = np.sqrt(2.0)):
    """mu[n][3], m[n][3] of Eq. 7-8 (TDA) for the vectors X[n][nocc][nvir]."""
    nocc = int(sys["nocc"])
    C = np.asarray(sys["C"], dtype=np.float64)
    Co, Cv = C[:, :nocc], C[:, nocc:]
    ao = oneel_ao(sys, origin)
    mo = np.array([Co.T @ ao[c] @ Cv for c in range(6)])                   # r_ia, (r x nabla)_ia
    mu = scale * np.einsum('cia,nia->nc', mo[:3], X)
    m = scale * np.einsum('cia,nia->nc', mo[3:], X)
    return mu, m


def strengths(omega: np.ndarray, mu: np.ndarray, m: np.ndarray):
    """oscillator strengths f_0n (Eq. 5) and rotatory strengths R_0n (Eq. 6)."""
    f = 2.0 / 3.0 * np.asarray(omega) * np.einsum('nc,nc->n', mu, mu)
    R = 0.5 * np.einsum('nc,nc->n', mu, m)
    return f, R
