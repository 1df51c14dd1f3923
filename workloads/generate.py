"""Seeded synthetic systems with the shapes of the paper's workloads.

The paper measures on EXTEST42 and on named 660-3145 atom systems with the
def2-SVP / def2-TZVP basis sets.  None of those
structures or basis-set tables is reproduced here: the generators below only
take their *shapes* (element mix, def2-SVP shell structure, pair sparsity,
window ratios, RSH parameters), as laid out in BASELINE.json `configs` and
DESIGN.md "Input recipe".

This module holds no arithmetic of the method (no ERI, no sigma, no eigen
solve).  The only integrals it evaluates are AO *overlaps*, which the method
itself never sees: they are needed to make the synthetic MO coefficients
orthonormal, C = S^-1/2 Q.

AO conventions (part of the C ABI, include/risp.h): real solid harmonics,
unit-normalised, order s; p = (x, y, z); d = (xy, yz, z2, xz, x2-y2).
"""
from __future__ import annotations

import math
import numpy as np

BASE_SEED = 260329257
HARTREE_EV = 27.211386245988
BOHR_ANG = 0.529177210903

CONFIG_NAMES = {
    1: "cfg1-C6H14-20atoms",
    2: "cfg2-C40H60-100atoms",
    3: "cfg3-cluster-300atoms",
    4: "cfg4-cluster-1000atoms",
    5: "cfg5-cluster-3000atoms",
}

# atoms (H, C, N, O), batch m, nroots, f_v (share of virtuals inside the window)
_CFG = {
    1: dict(counts=(14, 6, 0, 0), m=5, nroots=5, fv=None),
    2: dict(counts=(60, 40, 0, 0), m=30, nroots=15, fv=0.65),
    3: dict(counts=(147, 96, 27, 30), m=30, nroots=15, fv=0.65),
    4: dict(counts=(490, 320, 90, 100), m=30, nroots=15, fv=0.65),
    # f_v of config 5 is sized for THIS pool's boxes (180 GB HBM + 206 GB host RAM): 0.12 keeps the packed
    # K tensors (~156 GB) inside HBM + pinned host memory next to X, sigma and the work space; SURVEY proposed 0.20 for a 600 GB host
    5: dict(counts=(1470, 960, 270, 300), m=30, nroots=15, fv=0.12),
}


def _seed(cfg: int, item: int, base: int = BASE_SEED) -> np.random.Generator:
    return np.random.default_rng(base + 1000 * cfg + item)


# ----------------------------------------------------------------------------- geometry
_TET = math.radians(109.4712206)


def _alkane(rng):
    """All-trans C6H14, planar zig-zag carbon chain (BASELINE.json configs[0])."""
    cc, ch = 1.54, 1.09
    h = _TET / 2
    nC = 6
    Cpos = np.array([[k * cc * math.sin(h), (k % 2) * cc * math.cos(h), 0.0] for k in range(-1, nC + 1)])
    xyz, Z = [], []
    for k in range(1, nC + 1):
        xyz.append(Cpos[k]); Z.append(6)
    for k in range(1, nC + 1):
        c = Cpos[k]
        out = -1.0 if (k - 1) % 2 == 0 else 1.0          # away from both neighbours
        for sz in (1.0, -1.0):
            d = np.array([0.0, out * math.cos(h), sz * math.sin(h)])
            xyz.append(c + ch * d); Z.append(1)
        if k == 1 or k == nC:                              # terminal: H along the missing C-C bond
            nb = Cpos[k - 1] if k == 1 else Cpos[k + 1]
            d = (nb - c) / np.linalg.norm(nb - c)
            xyz.append(c + ch * d); Z.append(1)
    xyz = np.array(xyz) + rng.normal(0.0, 0.02, size=(len(xyz), 3))
    return xyz, np.array(Z, dtype=np.int32)


def _polyene(rng):
    """Planar C40 zig-zag backbone, alternating 1.34/1.46 A, 120 deg; 60 H (configs[1])."""
    nC, ch = 40, 1.09
    ang = math.radians(30.0)
    pos = [np.zeros(3)]
    for k in range(1, nC):
        L = 1.34 if k % 2 == 1 else 1.46
        sgn = 1.0 if k % 2 == 1 else -1.0
        pos.append(pos[-1] + L * np.array([math.cos(ang), sgn * math.sin(ang), 0.0]))
    pos = np.array(pos)
    sp3 = set(range(1, 37, 2))                              # 18 interior carbons carry two H
    xyz, Z = [p for p in pos], [6] * nC
    for k in range(nC):
        c = pos[k]
        if 0 < k < nC - 1:
            u = (pos[k - 1] - c) / np.linalg.norm(pos[k - 1] - c)
            v = (pos[k + 1] - c) / np.linalg.norm(pos[k + 1] - c)
            out = -(u + v); out /= np.linalg.norm(out)
            if k in sp3:
                hh = _TET / 2
                for sz in (1.0, -1.0):
                    xyz.append(c + ch * (math.cos(hh) * out + sz * math.sin(hh) * np.array([0, 0, 1.0]))); Z.append(1)
            else:
                xyz.append(c + ch * out); Z.append(1)
        else:
            nb = pos[1] if k == 0 else pos[nC - 2]
            u = (nb - c) / np.linalg.norm(nb - c)
            for s in (1.0, -1.0):                           # two in-plane H at +-120 deg from the bond
                a = s * math.radians(120.0)
                d = np.array([u[0] * math.cos(a) - u[1] * math.sin(a), u[0] * math.sin(a) + u[1] * math.cos(a), 0.0])
                xyz.append(c + ch * d); Z.append(1)
    xyz = np.array(xyz)
    assert len(xyz) == 100
    xyz = xyz + rng.normal(0.0, 0.02, size=xyz.shape)
    return xyz, np.array(Z, dtype=np.int32)


def _cluster(rng, counts):
    """Protein-like cluster: Poisson-disk heavy atoms in a ball, H hung on random heavy atoms."""
    nH, nC, nN, nO = counts
    nheavy = nC + nN + nO
    radius = (3.0 * nheavy / (4.0 * math.pi * 0.05)) ** (1.0 / 3.0)
    pts = np.zeros((0, 3))
    while len(pts) < nheavy:
        cand = rng.uniform(-radius, radius, size=3)
        if cand @ cand > radius * radius:
            continue
        if len(pts) and np.min(np.sum((pts - cand) ** 2, axis=1)) < 1.3 ** 2:
            continue
        pts = np.vstack([pts, cand])
    labels = np.array([6] * nC + [7] * nN + [8] * nO)
    rng.shuffle(labels)
    hs = np.zeros((0, 3))
    while len(hs) < nH:
        k = int(rng.integers(nheavy))
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        cand = pts[k] + 1.09 * d
        d2 = np.sum((pts - cand) ** 2, axis=1); d2[k] = 1e9
        if np.min(d2) < 1.5 ** 2:
            continue
        if len(hs) and np.min(np.sum((hs - cand) ** 2, axis=1)) < 1.5 ** 2:
            continue
        hs = np.vstack([hs, cand])
    xyz = np.vstack([pts, hs])
    Z = np.concatenate([labels, np.ones(nH, dtype=int)]).astype(np.int32)
    return xyz, Z


# ----------------------------------------------------------------------------- basis
def _element_basis(rng):
    """def2-SVP *shape* with synthetic exponents: heavy 3s2p1d, H 2s1p (DESIGN.md recipe)."""
    basis = {}
    for Z in (1, 6, 7, 8):
        shells = []
        if Z == 1:
            raw = [(0, [3.24, 1.08, 0.36]), (0, [0.12]), (1, [0.8])]
        else:
            lam = (Z / 6.0) ** 2
            t = 1000.0 * math.sqrt(Z / 6.0)
            raw = [(0, [t * 3.0 ** (-k) for k in range(5)]), (0, [0.39 * lam]), (0, [0.13 * lam]),
                   (1, [4.05 * lam, 1.35 * lam, 0.45 * lam]), (1, [0.15 * lam]), (2, [0.8 * lam])]
        for l, exps in raw:
            e = np.array(exps) * np.exp(rng.normal(0.0, 0.05, size=len(exps)))
            c = rng.uniform(0.2, 1.0, size=len(exps)) if len(exps) > 1 else np.ones(1)
            shells.append((l, e, c))
        basis[Z] = shells
    return basis


# stand-in radii R_A = n^2/Z_eff bohr (Slater screening); NOT the paper's table (ref. 18), G10
_AUX_RADIUS = {6: 4.0 / 3.25, 7: 4.0 / 3.90, 8: 4.0 / 4.55}
THETA = 0.2


def _radial_norm(a, l):
    return np.sqrt(2.0 * (2.0 * a) ** (l + 1.5) / math.gamma(l + 1.5))


def normalised_coefs(l, exps, coefs):
    """Coefficients of unit-normalised primitives, rescaled so the contracted shell has unit norm."""
    N = _radial_norm(exps, l)
    s = 0.0
    for k in range(len(exps)):
        for kk in range(len(exps)):
            s += coefs[k] * coefs[kk] * N[k] * N[kk] * math.gamma(l + 1.5) / (2.0 * (exps[k] + exps[kk]) ** (l + 1.5))
    return coefs / math.sqrt(s)


_CART = {0: [(0, 0, 0)], 1: [(1, 0, 0), (0, 1, 0), (0, 0, 1)],
         2: [(2, 0, 0), (1, 1, 0), (1, 0, 1), (0, 2, 0), (0, 1, 1), (0, 0, 2)]}


def _sph_matrix(l):
    """rows: spherical components, cols: Cartesian monomials in _CART order (angular factor only)."""
    if l == 0:
        return np.array([[1.0 / math.sqrt(4 * math.pi)]])
    if l == 1:
        return math.sqrt(3.0 / (4 * math.pi)) * np.eye(3)
    a = math.sqrt(15.0 / (4 * math.pi)); b = math.sqrt(5.0 / (16 * math.pi)); c = math.sqrt(15.0 / (16 * math.pi))
    M = np.zeros((5, 6))
    M[0, 1] = a                                  # xy
    M[1, 4] = a                                  # yz
    M[2, 5] = 2 * b; M[2, 0] = -b; M[2, 3] = -b  # 2zz - xx - yy
    M[3, 2] = a                                  # xz
    M[4, 0] = c; M[4, 3] = -c                    # xx - yy
    return M


def _overlap(xyz, shl_atom, shl_l, shl_nprim, shl_poff, prim_exp, prim_coef):
    """AO overlap matrix (generator-only; the sigma-build never uses S)."""
    nshl = len(shl_l)
    nf = np.array([2 * l + 1 for l in shl_l])
    off = np.concatenate([[0], np.cumsum(nf)])
    nao = int(off[-1])
    S = np.zeros((nao, nao))
    groups = {}
    for s in range(nshl):
        groups.setdefault((int(shl_l[s]), int(shl_nprim[s])), []).append(s)
    gdata = {}
    for (l, k), idx in groups.items():
        idx = np.array(idx)
        ex = np.array([prim_exp[shl_poff[s]:shl_poff[s] + k] for s in idx])
        cf = np.array([normalised_coefs(l, prim_exp[shl_poff[s]:shl_poff[s] + k], prim_coef[shl_poff[s]:shl_poff[s] + k])
                       * _radial_norm(prim_exp[shl_poff[s]:shl_poff[s] + k], l) for s in idx])
        gdata[(l, k)] = (idx, xyz[shl_atom[idx]], ex, cf)
    keys = sorted(gdata)

    def block(ka, kb, s0, chunk):
        la, lb = ka[0], kb[0]
        ia, A, ea, ca = gdata[ka]
        ib, B, eb, cb = gdata[kb]
        sl = slice(s0, s0 + chunk)
        a = ea[sl][:, None, :, None]; b = eb[None, :, None, :]
        p = a + b
        Ax = A[sl][:, None, None, None, :]; Bx = B[None, :, None, None, :]
        P = (a[..., None] * Ax + b[..., None] * Bx) / p[..., None]
        PA = P - Ax; PB = P - Bx
        AB2 = np.sum((A[sl][:, None, :] - B[None, :, :]) ** 2, axis=-1)[:, :, None, None]
        s1 = {}
        s1[(0, 0)] = np.ones_like(PA)
        for i in range(la + 1):
            for j in range(lb + 1):
                if i == 0 and j == 0:
                    continue
                if i > 0:
                    v = PA * s1[(i - 1, j)]
                    if i > 1: v = v + (i - 1) / (2 * p[..., None]) * s1[(i - 2, j)]
                    if j > 0: v = v + j / (2 * p[..., None]) * s1[(i - 1, j - 1)]
                else:
                    v = PB * s1[(i, j - 1)]
                    if j > 1: v = v + (j - 1) / (2 * p[..., None]) * s1[(i, j - 2)]
                s1[(i, j)] = v
        pref = (math.pi / p) ** 1.5 * np.exp(-a * b / p * AB2) * ca[sl][:, None, :, None] * cb[None, :, None, :]
        cartA, cartB = _CART[la], _CART[lb]
        blk = np.zeros((P.shape[0], P.shape[1], len(cartA), len(cartB)))
        for x, ca_ in enumerate(cartA):
            for y, cb_ in enumerate(cartB):
                t = pref * s1[(ca_[0], cb_[0])][..., 0] * s1[(ca_[1], cb_[1])][..., 1] * s1[(ca_[2], cb_[2])][..., 2]
                blk[:, :, x, y] = t.sum(axis=(2, 3))
        blk = np.einsum('sx,abxy,ty->abst', _sph_matrix(la), blk, _sph_matrix(lb))
        rows = (off[ia[sl]][:, None] + np.arange(2 * la + 1)[None, :])
        cols = (off[ib][:, None] + np.arange(2 * lb + 1)[None, :])
        S[rows[:, None, :, None], cols[None, :, None, :]] = blk      # disjoint blocks: safe from several threads

    tasks = []
    for ka in keys:
        for kb in keys:
            chunk = max(1, int(2e6 // max(1, len(gdata[kb][0]) * ka[1] * kb[1])))
            for s0 in range(0, len(gdata[ka][0]), chunk):
                tasks.append((ka, kb, s0, chunk))
    if nshl > 2000:
        import os
        from concurrent.futures import ThreadPoolExecutor
        with ThreadPoolExecutor(max_workers=min(32, os.cpu_count() or 1)) as ex:
            list(ex.map(lambda t: block(*t), tasks))
    else:
        for t in tasks:
            block(*t)
    return S


# ----------------------------------------------------------------------------- driver
def _torch_cuda():
    try:
        import torch
        return torch if torch.cuda.is_available() else None
    except Exception:
        return None


def _chol_blocked(torch, A, nb=4096):
    """Lower Cholesky factor of a (device) SPD matrix with panel-sized library calls only (in place on a copy)."""
    n = A.shape[0]
    L = A.clone()
    for k in range(0, n, nb):
        e = min(n, k + nb)
        L[k:e, k:e] = torch.linalg.cholesky(L[k:e, k:e])
        if e < n:
            # L21 = A21 L11^-T ; A22 -= L21 L21^T
            L[e:, k:e] = torch.linalg.solve_triangular(L[k:e, k:e], L[e:, k:e].T, upper=False).T
            L[e:, e:] -= L[e:, k:e] @ L[e:, k:e].T
    return torch.tril(L)


def _mos_by_cholesky(torch, S, rng, device="cuda"):
    """C with C^T S C = 1 and the distribution of S^-1/2 Q (Q Haar): C = L^-T Q with S = L L^T, because S^-1/2 = L^-T W for an
    orthogonal W and W Q is Haar again.  Q = the orthogonal factor of a seeded Gaussian matrix with positive-diagonal R, obtained
    by CholeskyQR2 (two rounds of G <- G chol(G^T G)^-T).  Also returns an estimate of lambda_min(S) by inverse iteration."""
    n = S.shape[0]
    St = torch.from_numpy(S).to(device)
    L = _chol_blocked(torch, St)
    x = torch.from_numpy(rng.normal(size=(n, 1))).to(device)
    lam = 0.0
    for _ in range(40):
        x = x / torch.linalg.norm(x)
        y = torch.linalg.solve_triangular(L, x, upper=False)
        y = torch.linalg.solve_triangular(L.T, y, upper=True)
        lam = float(1.0 / torch.linalg.norm(y))
        x = y
    G = torch.from_numpy(rng.normal(size=(n, n))).to(device)
    for _ in range(2):
        Lg = _chol_blocked(torch, G.T @ G)
        G = torch.linalg.solve_triangular(Lg, G.T, upper=False).T.contiguous()
        del Lg
    C = torch.linalg.solve_triangular(L.T, G, upper=True)
    del G, L
    E = C.T @ (St @ C)
    E.diagonal().sub_(1.0)
    err = float(E.abs().max())
    out = C.cpu().numpy()
    del C, E, St
    if device == "cuda":
        torch.cuda.empty_cache()
    return np.ascontiguousarray(out), lam, err


def make_system(cfg: int, *, base_seed: int = BASE_SEED, counts=None, check: bool = True) -> dict:
    """Build the seeded synthetic system for BASELINE.json configs[cfg-1].

    `counts=(nH, nC, nN, nO)` overrides the atom counts of a cluster config (used by
    tests that want a smaller cluster with the same recipe).  Returns a dict whose
    keys mirror `risp_system` in include/risp.h plus `m`, `nroots`, `name`.
    """
    spec = dict(_CFG[cfg])
    if counts is not None:
        spec["counts"] = tuple(counts)
    geom_seed = 0
    while True:
        rng = np.random.default_rng(base_seed + 1000 * cfg + 0 + 7919 * geom_seed)
        if cfg == 1 and counts is None:
            xyz_a, Z = _alkane(rng)
        elif cfg == 2 and counts is None:
            xyz_a, Z = _polyene(rng)
        else:
            xyz_a, Z = _cluster(rng, spec["counts"])
        xyz = xyz_a / BOHR_ANG
        basis = _element_basis(_seed(cfg, 1, base_seed))
        shl_atom, shl_l, shl_nprim, shl_poff, pe, pc = [], [], [], [], [], []
        for ia, z in enumerate(Z):
            for l, e, c in basis[int(z)]:
                shl_atom.append(ia); shl_l.append(l); shl_nprim.append(len(e)); shl_poff.append(len(pe))
                pe.extend(e.tolist()); pc.extend(c.tolist())
        shl_atom = np.array(shl_atom, dtype=np.int32); shl_l = np.array(shl_l, dtype=np.int32)
        shl_nprim = np.array(shl_nprim, dtype=np.int32); shl_poff = np.array(shl_poff, dtype=np.int32)
        pe = np.array(pe); pc = np.array(pc)
        nao = int(np.sum(2 * shl_l + 1))
        S = _overlap(xyz, shl_atom, shl_l, shl_nprim, shl_poff, pe, pc)
        gpu = _torch_cuda() if nao >= 6000 else None    # harness only: dense eigh / QR of the generator on the GPU when there is one
        if gpu is not None and nao > 25000:
            # 3000-atom scale: cuSOLVER's eigen solver and QR stop near n = 30 000 (32-bit work space, the limit PAPER.md:211
            # mentions), so the same distribution of MOs is drawn with Cholesky factors only (see _mos_by_cholesky)
            C, w0, ortho_err = _mos_by_cholesky(gpu, S, _seed(cfg, 2, base_seed))
            w = np.array([w0]); U = None
            if w0 > 1e-6 or not check:
                break
            geom_seed += 1
            continue
        if gpu is not None:
            St = gpu.from_numpy(S).cuda()
            wt, Ut = gpu.linalg.eigh(St)
            w = wt.cpu().numpy()
            U = Ut
        else:
            w, U = np.linalg.eigh(S)
        if w[0] > 1e-6 or not check:
            break
        geom_seed += 1                                    # near-singular overlap: redraw the geometry
        if geom_seed > 20:
            raise RuntimeError("could not draw a well-conditioned geometry")
    # hydrogen-free aux basis: one s + one p primitive per heavy atom, exponent theta/R_A^2 (Eq. 4)
    aux_atom, aux_l, aux_exp, aux_in_K = [], [], [], []
    for ia, z in enumerate(Z):
        if z == 1:
            continue
        g = THETA / _AUX_RADIUS[int(z)] ** 2
        aux_atom += [ia, ia]; aux_l += [0, 1]; aux_exp += [g, g]; aux_in_K += [1, 0]
    # MOs: C = S^-1/2 Q, Q Haar orthogonal
    if U is None:
        pass                                              # built by _mos_by_cholesky above
    elif gpu is not None:
        G = _seed(cfg, 2, base_seed).normal(size=(nao, nao))
        Qt, Rt = gpu.linalg.qr(gpu.from_numpy(G).cuda())
        del G
        Qt = Qt * gpu.sign(gpu.diagonal(Rt))[None, :]
        del Rt
        Ct = (Ut * (wt ** -0.5)[None, :]) @ (Ut.T @ Qt)
        del Qt, Ut
        E = Ct.T @ (St @ Ct)
        E.diagonal().sub_(1.0)
        ortho_err = float(E.abs().max())
        C = Ct.cpu().numpy()
        del Ct, St, E
        gpu.cuda.empty_cache()
    else:
        G = _seed(cfg, 2, base_seed).normal(size=(nao, nao))
        Q, R = np.linalg.qr(G)
        Q = Q * np.sign(np.diag(R))[None, :]
        C = (U * (w ** -0.5)[None, :]) @ U.T @ Q
        ortho_err = float(np.max(np.abs(C.T @ S @ C - np.eye(nao))))
    nelec = int(np.sum(Z))
    nocc = nelec // 2
    nvir = nao - nocc
    rng_e = _seed(cfg, 3, base_seed)
    nheavy = int(np.sum(Z > 1))
    if spec["fv"] is None:
        eo = np.sort(rng_e.uniform(-30.0, -5.0, size=nocc))
        ev = np.sort(rng_e.uniform(0.5, 30.0, size=nvir))
        alpha, beta, omega, cutoff = 0.25, 0.0, 0.0, 0.0
    else:
        core = rng_e.uniform(-560.0, -270.0, size=nheavy)
        val = rng_e.uniform(-30.0, -5.0, size=nocc - nheavy)
        eo = np.sort(np.concatenate([core, val]))
        nin = int(round(spec["fv"] * nvir))
        ev = np.sort(np.concatenate([rng_e.uniform(0.5, 30.0, size=nin), rng_e.uniform(45.0, 150.0, size=nvir - nin)]))
        alpha, beta, omega, cutoff = 0.16, 0.84, 0.2, 40.0
    eps = np.concatenate([eo, ev]) / HARTREE_EV
    return dict(
        name=CONFIG_NAMES[cfg] if counts is None else f"cfg{cfg}-custom-{len(Z)}atoms", cfg=cfg,
        natm=len(Z), xyz_bohr=np.ascontiguousarray(xyz), Z=Z.astype(np.int32),
        nshl=len(shl_l), shl_atom=shl_atom, shl_l=shl_l, shl_nprim=shl_nprim, shl_poff=shl_poff,
        prim_exp=pe, prim_coef=pc,
        naux=len(aux_l), aux_atom=np.array(aux_atom, dtype=np.int32), aux_l=np.array(aux_l, dtype=np.int32),
        aux_exp=np.array(aux_exp), aux_in_K=np.array(aux_in_K, dtype=np.uint8),
        nao=nao, nocc=nocc, nvir=nvir, C=np.ascontiguousarray(C), eps=eps,
        alpha=alpha, beta=beta, omega=omega, cutoff_ev=cutoff,
        m=spec["m"], nroots=spec["nroots"],
        overlap_min_eig=float(w[0]), ortho_err=ortho_err,
    )


def trial_vectors(sys: dict, m: int | None = None, *, base_seed: int = BASE_SEED, out: np.ndarray | None = None) -> np.ndarray:
    """m seeded Gaussian trial vectors [m][nocc][nvir], orthonormalised (DESIGN.md recipe)."""
    m = sys["m"] if m is None else m
    dim = sys["nocc"] * sys["nvir"]
    if dim * m > 1e9:
        # 3000-atom scale: m seeded Gaussian vectors, normalised only (in 1e8 dimensions they are orthogonal to ~1e-4; the
        # sigma-build is linear, so orthonormality is not needed for a throughput run)
        rng = _seed(sys["cfg"], 4, base_seed)
        X = np.empty((m, sys["nocc"], sys["nvir"])) if out is None else out      # `out`: e.g. a pinned buffer (no second 30 GB copy)
        for k in range(m):
            v = rng.standard_normal(dim)
            X[k] = (v / np.linalg.norm(v)).reshape(sys["nocc"], sys["nvir"])
        return X
    G = _seed(sys["cfg"], 4, base_seed).normal(size=(dim, m))
    Q, R = np.linalg.qr(G)
    Q = Q * np.sign(np.diag(R))[None, :]
    return np.ascontiguousarray(Q.T).reshape(m, sys["nocc"], sys["nvir"])
