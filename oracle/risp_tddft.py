"""ORACLE -- test infrastructure, not product code.

Full TDDFT-risp (arxiv/paper_2603_29257 Eq. 1-2) on top of oracle/risp_oracle.py: the matrices

    (A+B)[ia,jb] = d_ij d_ab (e_a - e_i) + 4 (ia|jb)_RI-J - [(ij|J^|ab) + (ib|J^|ja)]_RI-K [i,j in occK'; a,b in virK']
    (A-B)[ia,jb] = d_ij d_ab (e_a - e_i)                  - [(ij|J^|ab) - (ib|J^|ja)]_RI-K [window]

written out explicitly on tiny systems, their products with trial vectors by the MO route (explicit (ia|J^|P) over the window:
the tensor T_ia^P' that "is required only in the full TDDFT formalism"), and the excitation energies as the
positive eigenvalues of the symplectic problem Eq. 1.

Readings: G25 -- Eq. 2a prints "2(ia|jb)" for A+B, which is at odds with Eq. 10 (A has 2(ia|jb)) and Eq. 2b (A-B has
no Coulomb term, so B has 2(ia|jb) too): A+B carries 4(ia|jb).  The XC kernel is dropped.  The (ib|ja) term is
truncated to the same exchange window and uses the same K auxiliary set and operator J^ as (ij|ab).
Only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import this module.
"""
from __future__ import annotations

import numpy as np

from .risp_oracle import Oracle


class TddftOracle(Oracle):
    def build(self, chunk_shells: int = 8):
        if self._built:
            return
        super().build(chunk_shells)
        from scipy.linalg import solve_triangular
        self.BovW = None
        if self.has_K:
            # (ia|J^|P) over the window, whitened with the Cholesky factor of the K metric like (ij|P), (ab|P)
            Cok, Cvk = self.Co[:, self.occK], self.Cv[:, self.virK]
            nK = self.nfun(self.selK)
            Bov = np.zeros((nK, len(self.occK), len(self.virK)))
            f0 = 0
            for s0 in range(0, len(self.selK), chunk_shells):
                I3 = self.int3c(self.selK[s0:s0 + chunk_shells], self.alpha, self.beta, self.omega)
                for q in range(I3.shape[0]):
                    Bov[f0 + q] = Cok.T @ I3[q] @ Cvk
                f0 += I3.shape[0]
            self.Bov = Bov
            self.BovW = solve_triangular(self.LK, Bov.reshape(nK, -1), lower=True).reshape(Bov.shape)

    def exchange2(self, X):
        """K2_mia = sum_jb (ib|J^|ja)_RI X_mjb on the window; zero outside."""
        self.build()
        K = np.zeros_like(X)
        if not self.has_K:
            return K
        Xw = X[:, self.occK][:, :, self.virK]
        Kw = np.zeros_like(Xw)
        for P in range(self.BovW.shape[0]):
            N = np.einsum('ja,mjb->mab', self.BovW[P], Xw)          # N^P_mab = sum_j T_ja^P X_mjb
            Kw += np.einsum('ib,mab->mia', self.BovW[P], N)         # K2_mia += sum_b T_ib^P N^P_mab
        K[np.ix_(np.arange(X.shape[0]), self.occK, self.virK)] = Kw
        return K

    def sigma_pm(self, X):
        """((A+B) X, (A-B) X) for X[m][nocc][nvir]."""
        X = np.asarray(X, dtype=np.float64)
        dg = self.delta[None] * X
        J, K1, K2 = self.coulomb(X), self.exchange(X), self.exchange2(X)
        return dg + 4.0 * J - K1 - K2, dg - K1 + K2

    def full_B(self) -> np.ndarray:
        """B[ia,jb] = 2 (ia|jb) - (ib|J^|ja) [window], the matrix that couples X and Y in Eq. 1 (tiny systems only)."""
        self.build()
        dim = self.nocc * self.nvir
        Bm = self.BiaW.reshape(self.BiaW.shape[0], dim)
        B = 2.0 * (Bm.T @ Bm)
        if self.has_K:
            K2 = np.einsum('pib,pja->iajb', self.BovW, self.BovW)
            B4 = B.reshape(self.nocc, self.nvir, self.nocc, self.nvir)
            B4[np.ix_(self.occK, self.virK, self.occK, self.virK)] -= K2
        return B

    def tddft_eigenvalues(self, n=None):
        """Excitation energies of Eq. 1: Omega^2 are the eigenvalues of (A-B)^(1/2) (A+B) (A-B)^(1/2) (both matrices positive definite
        for a stable reference).  Returns Omega ascending, and the normalised X, Y (X^T X - Y^T Y = 1) as [n][nocc][nvir]."""
        A, B = self.full_A(), self.full_B()
        P, M = A + B, A - B
        w, U = np.linalg.eigh(M)
        if w[0] <= 0:
            raise ValueError("A - B is not positive definite")
        Mh = (U * np.sqrt(w)) @ U.T
        w2, Z = np.linalg.eigh(Mh @ P @ Mh)
        om = np.sqrt(w2)
        n = len(om) if n is None else n
        Zs = Z[:, :n] / np.sqrt(om[:n])[None, :]
        XpY = Mh @ Zs                                                  # |X+Y>, normalised so that <X+Y|X-Y> = 1
        XmY = (P @ XpY) / om[:n][None, :]
        Xv, Yv = 0.5 * (XpY + XmY), 0.5 * (XpY - XmY)
        return om[:n], Xv.T.reshape(n, self.nocc, self.nvir), Yv.T.reshape(n, self.nocc, self.nvir)
