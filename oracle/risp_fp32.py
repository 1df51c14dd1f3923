"""ORACLE -- test infrastructure, not product code.

The single-precision mode of the paper (arxiv/paper_2603_29257: "all quantities after the integral evaluation are
kept in single precision") for the exchange contractions Eq. 22-23, written out on top of
oracle/risp_oracle.py:

    M^P_mja = sum_b T_ab^P X_mjb        (Eq. 22)      K_mia = sum_P sum_j T_ij^P M^P_mja        (Eq. 23)

with T_ij^P, T_ab^P and X rounded to IEEE binary32 and both contractions carried out in binary32 (numpy float32 matmul), the
sum over P in binary32 too -- the plain definition of "the contractions in FP32", no blocking or compensation.  It is the
yardstick the FP32 mode of the CUDA path is judged by: that path must lie as close to the FP64 exchange as this does (its
error bound is derived in DESIGN.md, "FP32 mode").

`exchange_error_bound` is the standard forward bound of a floating-point inner product (Higham, Accuracy and Stability of
Numerical Algorithms, Sec. 3.1: |fl(x.y) - x.y| <= gamma_n |x|.|y|, gamma_n = n u / (1 - n u)) applied to the two nested
contractions and the input rounding, evaluated in FP64 with absolute values.

Only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import this module.
"""
from __future__ import annotations

import numpy as np

U32 = 2.0 ** -24          # unit roundoff of binary32


def exchange_fp32(o, X):
    """K (Eq. 22-23) with T, X and every product/sum in binary32; o is a built oracle.risp_oracle.Oracle. Returns float64 storage."""
    o.build()
    X = np.asarray(X, dtype=np.float64)
    K = np.zeros_like(X)
    if not o.has_K:
        return K
    Xw = X[:, o.occK][:, :, o.virK].astype(np.float32)
    Kw = np.zeros(Xw.shape, dtype=np.float32)
    for P in range(o.BijW.shape[0]):
        Tab = o.BabW[P].astype(np.float32)
        Tij = o.BijW[P].astype(np.float32)
        M = Xw @ Tab.T                                # Eq. 22 in binary32
        Kw = Kw + Tij[None] @ M                       # Eq. 23 in binary32, P summed in binary32
    K[np.ix_(np.arange(X.shape[0]), o.occK, o.virK)] = Kw.astype(np.float64)
    return K


def exchange_error_bound(o, X):
    """Elementwise bound on |exchange_fp32 - exchange|: the nested inner products have nv + no*nP + nP terms and three rounded
    inputs, so |dK| <= gamma_(nv + no + nP + 3) * sum_P |T_ij^P| (|X| |T_ab^P|^T)  (first order in u, constant rounded up)."""
    o.build()
    X = np.asarray(X, dtype=np.float64)
    B = np.zeros_like(X)
    if not o.has_K:
        return B
    Xw = np.abs(X[:, o.occK][:, :, o.virK])
    Bw = np.zeros_like(Xw)
    for P in range(o.BijW.shape[0]):
        Bw += np.abs(o.BijW[P])[None] @ (Xw @ np.abs(o.BabW[P]).T)
    n = len(o.virK) + len(o.occK) + o.BijW.shape[0] + 3
    g = n * U32 / (1.0 - n * U32)
    B[np.ix_(np.arange(X.shape[0]), o.occK, o.virK)] = g * Bw
    return B
