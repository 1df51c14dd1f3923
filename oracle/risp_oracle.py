"""ORACLE -- test infrastructure, not product code.

Plain CPU FP64 implementation of what the TDA-risp sigma-build computes
(arxiv/paper_2603_29257), written from the paper's equations.  Only tests/,
`__graft_entry__.smoke()` and bench.py's cpu_baseline / `--impl reference` legs
may import this module.  It shares nothing with the CUDA path
(`paper_2603_29257_b200/`): the integrals come from oracle/risp_integrals.c
(McMurchie-Davidson, long-double internals), everything else is numpy.

The method has an exact definition: TDA-risp
*defines* the matrix

    A[ia,jb] = d_ij d_ab (e_a - e_i) + 2 (ia|jb)_RI-J - (ij|J^|ab)_RI-K [i,j in occK'; a,b in virK']

(Eq. 10 with Eq. 3 and Eq. 19-21, 26 substituted; window PAPER.md:136)
and the oracle is that definition written out:

  * `full_A`           -- A formed explicitly (tiny systems), `eigh` for the roots;
  * `sigma`            -- sigma = A X by the MO route with explicit (ia|P), (ij|P), (ab|P);
  * `coulomb_ao_direct`-- Eq. 11-17 literally (D, R, R~, U, J), to pin J_AO = J_MO;
  * `davidson`         -- a standard Davidson (reading G16) on `sigma`.

Pins: tests/test_oracle_*.py (closed forms, quadrature of the definition, invariants,
limits, brute force).  No function here is parity-unpinned.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

HARTREE_EV = 27.211386245988           # CODATA 2018; the window decision depends on it

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None


def build_lib(force: bool = False) -> str:
    """Compile oracle/risp_integrals.c -> oracle/librisp_oracle.so (gcc -O2 -fopenmp)."""
    src = os.path.join(_HERE, "risp_integrals.c")
    so = os.path.join(_HERE, "librisp_oracle.so")
    if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", so, src, "-lm"])
    return so


def _lib():
    global _LIB
    if _LIB is None:
        _LIB = ctypes.CDLL(build_lib())
        _LIB.oracle_prim3c.restype = ctypes.c_double
        _LIB.oracle_prim2c.restype = ctypes.c_double
    return _LIB


def _p(a, t):
    return a.ctypes.data_as(ctypes.POINTER(t))


_D, _I = ctypes.c_double, ctypes.c_int


def boys(nmax: int, x: float) -> np.ndarray:
    out = np.zeros(nmax + 1)
    _lib().oracle_boys(_I(nmax), _D(x), _p(out, _D))
    return out


def prim3c(a, A, la, b, B, lb, g, C, lc, ca=1.0, cb=0.0, w=0.0) -> float:
    """Unnormalised primitive Cartesian (ab|c), operator (ca + cb erf(w r))/r."""
    A, B, C = (np.ascontiguousarray(v, dtype=np.float64) for v in (A, B, C))
    la, lb, lc = (np.ascontiguousarray(v, dtype=np.int32) for v in (la, lb, lc))
    return _lib().oracle_prim3c(_D(a), _p(A, _D), _p(la, _I), _D(b), _p(B, _D), _p(lb, _I), _D(g), _p(C, _D), _p(lc, _I),
                                _D(ca), _D(cb), _D(w))


def prim2c(gc, C, lc, gd, D, ld, ca=1.0, cb=0.0, w=0.0) -> float:
    C, D = (np.ascontiguousarray(v, dtype=np.float64) for v in (C, D))
    lc, ld = (np.ascontiguousarray(v, dtype=np.int32) for v in (lc, ld))
    return _lib().oracle_prim2c(_D(gc), _p(C, _D), _p(lc, _I), _D(gd), _p(D, _D), _p(ld, _I), _D(ca), _D(cb), _D(w))


class Oracle:
    """CPU oracle for one system (dict with the fields of `risp_system`, include/risp.h)."""

    def __init__(self, sys: dict, kab_tol: float = 0.0):
        self.s = sys
        self.kab_tol = float(kab_tol)
        f64 = lambda k: np.ascontiguousarray(sys[k], dtype=np.float64)
        i32 = lambda k: np.ascontiguousarray(sys[k], dtype=np.int32)
        self.xyz, self.pe, self.pc, self.aux_exp = f64("xyz_bohr"), f64("prim_exp"), f64("prim_coef"), f64("aux_exp")
        self.shl_atom, self.shl_l, self.shl_nprim, self.shl_poff = i32("shl_atom"), i32("shl_l"), i32("shl_nprim"), i32("shl_poff")
        self.aux_atom, self.aux_l = i32("aux_atom"), i32("aux_l")
        self.nshl, self.naux_shl = len(self.shl_l), len(self.aux_l)
        self.nao, self.nocc, self.nvir = int(sys["nao"]), int(sys["nocc"]), int(sys["nvir"])
        self.C = f64("C"); self.eps = f64("eps")
        self.Co, self.Cv = self.C[:, :self.nocc], self.C[:, self.nocc:]
        self.alpha, self.beta, self.omega = float(sys["alpha"]), float(sys["beta"]), float(sys["omega"])
        self.selJ = np.arange(self.naux_shl, dtype=np.int32)                       # J: all aux shells
        self.selK = np.nonzero(np.asarray(sys["aux_in_K"]))[0].astype(np.int32)    # K: the s shells
        self.delta = self.eps[None, self.nocc:] - self.eps[:self.nocc, None]       # (e_a - e_i), Eq. 10
        self.window()
        self._built = False

    # ------------------------------------------------------------------ integrals
    def overlap(self) -> np.ndarray:
        S = np.zeros((self.nao, self.nao))
        _lib().oracle_overlap(_I(self.s["natm"]), _p(self.xyz, _D), _I(self.nshl), _p(self.shl_atom, _I), _p(self.shl_l, _I),
                              _p(self.shl_nprim, _I), _p(self.shl_poff, _I), _p(self.pe, _D), _p(self.pc, _D), _p(S, _D))
        return S

    def nfun(self, sel) -> int:
        return int(np.sum(2 * self.aux_l[np.asarray(sel)] + 1))

    def int2c(self, sel, ca=1.0, cb=0.0, w=0.0) -> np.ndarray:
        sel = np.ascontiguousarray(sel, dtype=np.int32)
        nf = self.nfun(sel)
        out = np.zeros((nf, nf))
        _lib().oracle_int2c(_p(self.xyz, _D), _I(len(sel)), _p(sel, _I), _p(self.aux_atom, _I), _p(self.aux_l, _I),
                            _p(self.aux_exp, _D), _D(ca), _D(cb), _D(w), _p(out, _D))
        return out

    def int3c(self, sel, ca=1.0, cb=0.0, w=0.0, full_square=False) -> np.ndarray:
        """(mu nu|P) for the aux shells `sel`: [nfun(sel)][nao][nao]."""
        sel = np.ascontiguousarray(sel, dtype=np.int32)
        out = np.zeros((self.nfun(sel), self.nao, self.nao))
        _lib().oracle_int3c(_p(self.xyz, _D), _I(self.nshl), _p(self.shl_atom, _I), _p(self.shl_l, _I), _p(self.shl_nprim, _I),
                            _p(self.shl_poff, _I), _p(self.pe, _D), _p(self.pc, _D), _I(len(sel)), _p(sel, _I),
                            _p(self.aux_atom, _I), _p(self.aux_l, _I), _p(self.aux_exp, _D), _D(ca), _D(cb), _D(w),
                            _I(1 if full_square else 0), _D(self.kab_tol), _p(out, _D))
        return out

    # ------------------------------------------------------------------ window
    def window(self, cutoff_ev=None):
        """occK' = {i: e_i > -cut}, virK' = {a: e_a < +cut}; cut <= 0 or inf: no truncation."""
        cut = self.s["cutoff_ev"] if cutoff_ev is None else cutoff_ev
        e_ev = self.eps * HARTREE_EV
        if cut is None or cut <= 0 or not np.isfinite(cut):
            self.occK = np.arange(self.nocc); self.virK = np.arange(self.nvir)
        else:
            self.occK = np.nonzero(e_ev[:self.nocc] > -cut)[0]
            self.virK = np.nonzero(e_ev[self.nocc:] < cut)[0]
        self._built = False
        return self.occK, self.virK

    # ------------------------------------------------------------------ MO three-index tensors
    def build(self, chunk_shells: int = 8):
        if self._built:
            return
        from scipy.linalg import cholesky, solve_triangular
        # J: (ia|P) over ALL occ/virt, Coulomb operator and Coulomb metric
        Bia = np.zeros((self.nfun(self.selJ), self.nocc, self.nvir))
        f0 = 0
        for s0 in range(0, len(self.selJ), chunk_shells):
            sel = self.selJ[s0:s0 + chunk_shells]
            I3 = self.int3c(sel)
            for q in range(I3.shape[0]):
                Bia[f0 + q] = self.Co.T @ I3[q] @ self.Cv
            f0 += I3.shape[0]
        self.MJ = self.int2c(self.selJ)
        self.LJ = cholesky(self.MJ, lower=True)
        self.Bia = Bia
        self.BiaW = solve_triangular(self.LJ, Bia.reshape(Bia.shape[0], -1), lower=True).reshape(Bia.shape)
        # K: (ij|J^|P), (ab|J^|P) over the window, operator J^ in 3c AND 2c integrals (Eq. 26)
        Cok, Cvk = self.Co[:, self.occK], self.Cv[:, self.virK]
        nK = self.nfun(self.selK)
        Bij = np.zeros((nK, len(self.occK), len(self.occK))); Bab = np.zeros((nK, len(self.virK), len(self.virK)))
        f0 = 0
        for s0 in range(0, len(self.selK), chunk_shells):
            sel = self.selK[s0:s0 + chunk_shells]
            I3 = self.int3c(sel, self.alpha, self.beta, self.omega)
            for q in range(I3.shape[0]):
                Bij[f0 + q] = Cok.T @ I3[q] @ Cok
                Bab[f0 + q] = Cvk.T @ I3[q] @ Cvk
            f0 += I3.shape[0]
        self.Bij, self.Bab = Bij, Bab
        self.has_K = (self.alpha != 0.0 or self.beta != 0.0) and nK > 0 and len(self.occK) > 0 and len(self.virK) > 0
        if self.has_K:
            self.MK = self.int2c(self.selK, self.alpha, self.beta, self.omega)
            self.LK = cholesky(self.MK, lower=True)
            self.BijW = solve_triangular(self.LK, Bij.reshape(nK, -1), lower=True).reshape(Bij.shape)
            self.BabW = solve_triangular(self.LK, Bab.reshape(nK, -1), lower=True).reshape(Bab.shape)
        self._built = True

    # ------------------------------------------------------------------ sigma = A X, MO route
    def coulomb(self, X):
        """J_mia = sum_jb (ia|jb)_RI X_mjb, Eq. 3/13 with explicit (ia|P)."""
        self.build()
        m = X.shape[0]
        B = self.BiaW.reshape(self.BiaW.shape[0], -1)
        return (B.T @ (B @ X.reshape(m, -1).T)).T.reshape(X.shape)

    def exchange(self, X):
        """K_mia = sum_jb sum_PQ (ij|P)(P|Q)^-1(Q|ab) X_mjb on the window (Eq. 18-21, 26); zero outside."""
        self.build()
        K = np.zeros_like(X)
        if not self.has_K:
            return K
        Xw = X[:, self.occK][:, :, self.virK]
        Kw = np.zeros_like(Xw)
        for P in range(self.BijW.shape[0]):
            M = Xw @ self.BabW[P].T                      # M^P_mja = sum_b T_ab^P X_mjb        (Eq. 22)
            Kw += self.BijW[P][None] @ M                 # K_mia  += sum_j T_ij^P M^P_mja      (Eq. 23)
        K[np.ix_(np.arange(X.shape[0]), self.occK, self.virK)] = Kw
        return K

    def sigma(self, X, parts: bool = False):
        """sigma_m = A X_m = Delta*X + 2 J - K (Eq. 10).  X: [m][nocc][nvir]."""
        X = np.asarray(X, dtype=np.float64)
        dg = self.delta[None] * X
        J = self.coulomb(X)
        K = self.exchange(X)
        sig = dg + 2.0 * J - K
        return (sig, dg, J, K) if parts else sig

    def full_A(self) -> np.ndarray:
        """The explicit (nocc*nvir)^2 matrix of Eq. 10 (tiny systems only)."""
        self.build()
        dim = self.nocc * self.nvir
        B = self.BiaW.reshape(self.BiaW.shape[0], dim)
        A = np.diag(self.delta.reshape(-1)) + 2.0 * (B.T @ B)
        if self.has_K:
            Kfull = np.einsum('pij,pab->iajb', self.BijW, self.BabW)
            A4 = A.reshape(self.nocc, self.nvir, self.nocc, self.nvir)
            A4[np.ix_(self.occK, self.virK, self.occK, self.virK)] -= Kfull
        return A

    # ------------------------------------------------------------------ Eq. 11-17 literally
    def coulomb_ao_direct(self, X):
        """J by the paper's on-the-fly order: D (Eq. 12), R (Eq. 14), R~ (Eq. 15), U (Eq. 16), J (Eq. 17)."""
        m = X.shape[0]
        I3 = self.int3c(self.selJ)                                    # (Q|kappa lambda), all pairs, no screening
        MJ = self.int2c(self.selJ)
        J = np.zeros_like(X)
        stages = []
        for k in range(m):
            D = self.Co @ X[k] @ self.Cv.T                             # Eq. 12 (reading G1: sum over j, b)
            R = np.einsum('qkl,kl->q', I3, D)                          # Eq. 14
            Rt = np.linalg.solve(MJ, R)                                # Eq. 15
            U = np.einsum('pmn,p->mn', I3, Rt)                         # Eq. 16
            J[k] = self.Co.T @ U @ self.Cv                             # Eq. 17
            stages.append((D, R, Rt, U))
        self.ao_stages = stages
        return J

    # ------------------------------------------------------------------ Davidson (reading G16)
    def davidson(self, nroots, n_guess=None, tol=1e-8, max_iter=100, max_sub=None, sigma_fn=None, log=None):
        """Standard Davidson for the lowest `nroots` eigenpairs of A.  Returns (omega[nroots], X[nroots][nocc][nvir], info)."""
        sigma_fn = self.sigma if sigma_fn is None else sigma_fn
        dim = self.nocc * self.nvir
        n_guess = min(dim, 2 * nroots if n_guess is None else n_guess)
        max_sub = 20 * nroots if max_sub is None else max_sub
        dflat = self.delta.reshape(-1)
        order = np.argsort(dflat, kind="stable")[:n_guess]
        V = np.zeros((n_guess, dim)); V[np.arange(n_guess), order] = 1.0
        W = sigma_fn(V.reshape(-1, self.nocc, self.nvir)).reshape(-1, dim)
        n_sigma, restarts = n_guess, 0
        for it in range(1, max_iter + 1):
            G = V @ W.T; G = 0.5 * (G + G.T)
            th, y = np.linalg.eigh(G)
            th, y = th[:nroots], y[:, :nroots]
            Xr = y.T @ V; AX = y.T @ W
            res = AX - th[:, None] * Xr
            rn = np.linalg.norm(res, axis=1)
            if log is not None:
                log.append((it, V.shape[0], th.copy(), rn.copy()))
            if np.all(rn < tol):
                return th, Xr.reshape(nroots, self.nocc, self.nvir), dict(iterations=it, n_sigma=n_sigma, restarts=restarts, resid=rn, converged=True)
            new = []
            for j in range(nroots):
                if rn[j] < tol:
                    continue
                den = th[j] - dflat
                den = np.where(np.abs(den) < 1e-8, np.where(den < 0, -1e-8, 1e-8), den)
                new.append(res[j] / den)
            if V.shape[0] + len(new) > max_sub:                         # restart from the Ritz vectors (G17)
                V, W = Xr.copy(), AX.copy(); restarts += 1
            T = np.array(new)
            kept = []
            for t in T:
                t = t / np.linalg.norm(t)
                for _ in range(2):                                      # two passes of classical Gram-Schmidt
                    t = t - V.T @ (V @ t)
                    for k in kept:
                        t = t - k * (k @ t)
                nt = np.linalg.norm(t)
                if nt > 1e-8:
                    kept.append(t / nt)
            if not kept:
                break
            Vn = np.array(kept)
            Wn = sigma_fn(Vn.reshape(-1, self.nocc, self.nvir)).reshape(-1, dim)
            n_sigma += len(kept)
            V = np.vstack([V, Vn]); W = np.vstack([W, Wn])
        return th, Xr.reshape(nroots, self.nocc, self.nvir), dict(iterations=max_iter, n_sigma=n_sigma, restarts=restarts, resid=rn, converged=False)
