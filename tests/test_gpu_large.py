"""Compositional parity at the large configurations (BASELINE.json configs[2..4]).

The full oracle (every integral, explicit MO tensors) is infeasible from ~1000 atoms on, so the stages of the CUDA path are
checked one by one against quantities the oracle CAN compute at full size:

  (i)   sampled three-centre integrals of all six pair classes, both operators        -> oracle McMurchie-Davidson integrals
  (ii)  both metrics                                                                   -> oracle two-centre integrals
  (iii) R_mQ of pass 1 (Eq. 14) for sampled Q over ALL AO pairs (checks the screening)  -> oracle (mu nu|Q) . (C_occ X C_vir^T)
  (iv)  R~ (Eq. 15) through (P|Q) R~ = R;  U (Eq. 16) on sampled shell pairs           -> oracle (mu nu|all P) . R~
  (v)   J_mia (Eq. 17) on sampled (i, a) from the device U
  (vi)  T_ab^P full slices for sampled P (device- and host-resident)                    -> C_v'^T (mu nu|J^|P) C_v'
  (vii) T_ij^P through the metric: sum_P (Q|P) u^T T_ij^P v = u^T (ij|J^|Q) v for sampled Q
  (viii) sigma: symmetry <x, A y> = <y, A x>, and independence of the memory plan (dense vs sub-batched / panelled / small
        aux chunks), which together with (vi)-(vii) and the element-wise K parity of the small configs covers Eq. 22-23.

The 300- and 1000-atom configurations always run (about 2.5 minutes together on a B200 box); the 3000-atom one needs ~25
minutes (11 of them risp_setup) and more than the 1200 s the driver gives `pytest -m gpu`, so it runs only with RISP_LARGE=5
and its log is kept under profiles/.  The element-by-element comparison against the FULL oracle at 300 atoms is
tests/test_gpu_cfg3.py.
"""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu
HARTREE_EV = 27.211386245988
_CFGS = sorted({3, 4} | {int(c) for c in os.environ.get("RISP_LARGE", "").split(",") if c.strip()})


def _rel(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / max(np.linalg.norm(b), 1e-300))


def _sub_oracle(s, shells, auxs):
    """Oracle over a few AO shells and aux shells of system s (integrals only)."""
    from oracle.risp_oracle import Oracle
    shells = list(shells); auxs = list(auxs)
    pe, pc, poff, nprim = [], [], [], []
    for sh in shells:
        k, o = int(s["shl_nprim"][sh]), int(s["shl_poff"][sh])
        poff.append(len(pe)); nprim.append(k)
        pe += list(s["prim_exp"][o:o + k]); pc += list(s["prim_coef"][o:o + k])
    nao = int(sum(2 * int(s["shl_l"][sh]) + 1 for sh in shells))
    sub = dict(s)
    sub.update(nshl=len(shells), shl_atom=np.asarray(s["shl_atom"])[shells], shl_l=np.asarray(s["shl_l"])[shells],
               shl_nprim=np.array(nprim, dtype=np.int32), shl_poff=np.array(poff, dtype=np.int32), prim_exp=np.array(pe), prim_coef=np.array(pc),
               naux=len(auxs), aux_atom=np.asarray(s["aux_atom"])[auxs], aux_l=np.asarray(s["aux_l"])[auxs], aux_exp=np.asarray(s["aux_exp"])[auxs],
               aux_in_K=np.asarray(s["aux_in_K"])[auxs], nao=nao, nocc=1, nvir=nao - 1 if nao > 1 else 1,
               C=np.eye(nao, max(nao, 2))[:, :max(nao, 2)], eps=np.arange(max(nao, 2), dtype=float))
    return Oracle(sub)


@pytest.mark.parametrize("cfg", _CFGS)
def test_large_configuration_compositional_parity(cfg):
    import time
    import torch
    from oracle.risp_oracle import Oracle
    from paper_2603_29257_b200 import setup
    from workloads import make_system, trial_vectors
    t0 = time.time()
    s = make_system(cfg)
    o = Oracle(s)
    nao, nocc, nvir = s["nao"], s["nocc"], s["nvir"]
    m = 2
    print(f"\n[cfg{cfg}] system {s['name']} nao={nao} generated in {time.time() - t0:.1f} s", flush=True)
    t0 = time.time()
    c = setup(s, flags=1, max_batch=m)
    d = c.dims()
    print(f"[cfg{cfg}] risp_setup {time.time() - t0:.1f} s; dims {d}", flush=True)
    rng = np.random.default_rng(1234 + cfg)
    soff = np.concatenate([[0], np.cumsum(2 * np.asarray(s["shl_l"]) + 1)])
    aoff = np.concatenate([[0], np.cumsum(2 * np.asarray(s["aux_l"]) + 1)])
    try:
        # ---- (i) sampled integrals, every pair class, both operators; near pairs (same / neighbouring atoms) and random ones
        by_l = {l: np.nonzero(np.asarray(s["shl_l"]) == l)[0] for l in (0, 1, 2)}
        worst = 0.0
        for la in (0, 1, 2):
            for lb in (0, 1, 2):
                for t in range(6):
                    si = int(rng.choice(by_l[la]))
                    if t < 3:       # a partner on a nearby atom
                        at = s["shl_atom"][si]
                        dist = np.linalg.norm(s["xyz_bohr"] - s["xyz_bohr"][at], axis=1)
                        near = np.argsort(dist)[:6]
                        cand = [x for x in by_l[lb] if s["shl_atom"][x] in near]
                        sj = int(rng.choice(cand))
                    else:
                        sj = int(rng.choice(by_l[lb]))
                    ak = [int(x) for x in rng.choice(len(s["aux_l"]), size=3, replace=False)]
                    so = _sub_oracle(s, [si, sj], ak)
                    for op, (ca, cb, w) in ((0, (1.0, 0.0, 0.0)), (1, (s["alpha"], s["beta"], s["omega"]))):
                        I3 = so.int3c(np.arange(len(ak)), ca, cb, w)
                        n_i = 2 * la + 1
                        a0 = 0
                        for k, a in enumerate(ak):
                            nk = 2 * int(s["aux_l"][a]) + 1
                            ref = I3[a0:a0 + nk, :n_i, n_i:].transpose(1, 2, 0) if si != sj else I3[a0:a0 + nk, :n_i, :n_i].transpose(1, 2, 0)
                            a0 += nk
                            if si == sj:
                                continue
                            got = c.eri3c_shell(si, sj, a, op)
                            worst = max(worst, float(np.abs(got - ref).max()))
        print(f"[cfg{cfg}] (i) max |d(mu nu|P)| over sampled shell triples = {worst:.2e}", flush=True)
        assert worst <= 1e-12
        # ---- (ii) metrics
        MJ, MK = c.stage("METRIC_J"), c.stage("METRIC_K")
        e1 = float(np.abs(MJ - o.int2c(o.selJ)).max()); e2 = float(np.abs(MK - o.int2c(o.selK, o.alpha, o.beta, o.omega)).max())
        print(f"[cfg{cfg}] (ii) max |d(P|Q)_J| = {e1:.2e}, max |d(P|J^|Q)_K| = {e2:.2e}", flush=True)
        assert e1 <= 1e-12 and e2 <= 1e-12
        # ---- sigma-build on m vectors
        X = trial_vectors(s, m)
        Xd = torch.from_numpy(X).cuda()
        t0 = time.time()
        sig = c.matvec(Xd)
        torch.cuda.synchronize()
        print(f"[cfg{cfg}] risp_matvec(m={m}) {time.time() - t0:.2f} s, plan {c.dims()['j_sub_batch']}/{c.dims()['j_panels']}/{c.dims()['aux_chunk']}", flush=True)
        Co, Cv = o.Co, o.Cv
        # ---- (iii) R for sampled aux shells, oracle integrals over ALL AO pairs (unscreened)
        D = [Co @ X[k] @ Cv.T for k in range(m)]
        R = c.stage("R", m)
        qs = [int(x) for x in rng.choice(len(s["aux_l"]), size=3, replace=False)]
        for q in qs:
            I3 = o.int3c([q])
            ref = np.array([[np.vdot(I3[f], D[k]) for k in range(m)] for f in range(I3.shape[0])])
            e = _rel(R[aoff[q]:aoff[q + 1]], ref)
            print(f"[cfg{cfg}] (iii) R_mQ aux shell {q} (l={s['aux_l'][q]}): rel err {e:.2e}", flush=True)
            assert e <= 1e-10
        # ---- (iv) R~ and U
        Rt = c.stage("RTILDE", m)
        e = _rel(MJ @ Rt, R)
        print(f"[cfg{cfg}] (iv) |(P|Q) R~ - R| / |R| = {e:.2e}", flush=True)
        assert e <= 1e-10
        U = c.stage("U", m, sel=[1])
        kept = c.stage("PAIRS")
        # half of the sample from same-atom / neighbouring-atom pairs (large blocks), half uniformly from the kept list (mostly far
        # pairs, tiny blocks); error measured PER BLOCK against the block's own norm, with the absolute floor the integral
        # tolerance implies: |dU| <= 1e-12 * sum_P |R~_P|
        at_of = np.asarray(s["shl_atom"])
        dist_at = np.linalg.norm(s["xyz_bohr"][at_of[kept[:, 0]]] - s["xyz_bohr"][at_of[kept[:, 1]]], axis=1)
        near = np.nonzero((dist_at < 3.0) & (kept[:, 0] != kept[:, 1]))[0]
        sample = list(rng.choice(near, size=8, replace=False)) + list(rng.choice(len(kept), size=8, replace=False))
        floor = 1e-12 * float(np.abs(Rt[:, 1]).sum())
        worstU, worst_rel = 0.0, 0.0
        for idx in sample:
            si, sj = int(kept[idx][0]), int(kept[idx][1])
            if si == sj:
                continue
            so = _sub_oracle(s, [si, sj], range(len(s["aux_l"])))
            I3 = so.int3c(np.arange(len(s["aux_l"])))
            n_i = 2 * int(s["shl_l"][si]) + 1
            ref = np.einsum('pij,p->ij', I3[:, :n_i, n_i:], Rt[:, 1])
            got = U[soff[si]:soff[si + 1], soff[sj]:soff[sj + 1]]
            err, nrm = float(np.abs(got - ref).max()), float(np.linalg.norm(ref))
            worstU = max(worstU, err / (1e-10 * nrm + floor))
            worst_rel = max(worst_rel, err / max(nrm, 1e-300))
        print(f"[cfg{cfg}] (iv) U on {len(sample)} kept shell pairs (8 near, 8 random): worst err / (1e-10 |block| + {floor:.1e}) = {worstU:.2e}; "
              f"worst err / |block| = {worst_rel:.2e}", flush=True)
        assert worstU <= 1.0
        assert np.abs(U - U.T).max() <= 1e-12 * np.abs(U).max()
        # ---- (v) J on sampled (i, a)
        J = c.stage("J", m)
        ii = rng.choice(nocc, size=8); aa = rng.choice(nvir, size=8)
        ref = np.einsum('mi,mn,na->ia', Co[:, ii], U, Cv[:, aa])
        e = float(np.abs(J[1][np.ix_(ii, aa)] - ref).max() / np.abs(ref).max())
        print(f"[cfg{cfg}] (v) J_ia on sampled (i,a): max rel err {e:.2e}", flush=True)
        assert e <= 1e-10
        del U, D
        # ---- (vi) T_ab slices (first, last device-resident, first host-resident if any, last)
        nK, nKd = d["nauxK"], d["nauxK_device"]
        selP = sorted({0, max(nKd - 1, 0), min(nKd, nK - 1), nK - 1})[:3]
        Kshell_of_fn = []
        for sh in o.selK:
            Kshell_of_fn += [(int(sh), f) for f in range(2 * int(s["aux_l"][sh]) + 1)]
        Cok, Cvk = Co[:, o.occK], Cv[:, o.virK]
        for P in selP:
            sh, f = Kshell_of_fn[P]
            I3 = o.int3c([sh], o.alpha, o.beta, o.omega)[f]
            ref = Cvk.T @ I3 @ Cvk
            got = c.stage("TAB", sel=[P])[0]
            e = _rel(got, ref)
            print(f"[cfg{cfg}] (vi) T_ab^P slice P={P} ({'HBM' if P < nKd else 'host'}): rel err {e:.2e}", flush=True)
            assert e <= 1e-11
        # ---- (vii) T_ij through the metric
        u, v = rng.normal(size=len(o.occK)), rng.normal(size=len(o.occK))
        tP = np.zeros(nK)
        for p0 in range(0, nK, 32):
            sel = list(range(p0, min(nK, p0 + 32)))
            T = c.stage("TIJ", sel=sel)
            tP[p0:p0 + len(sel)] = np.einsum('i,pij,j->p', u, T, v)
        lhs = MK @ tP
        for P in selP:
            sh, f = Kshell_of_fn[P]
            I3 = o.int3c([sh], o.alpha, o.beta, o.omega)[f]
            ref = float((Cok @ u) @ I3 @ (Cok @ v))
            e = abs(lhs[P] - ref) / max(np.abs(lhs).max(), 1e-300)
            print(f"[cfg{cfg}] (vii) sum_P (Q|P) u^T T_ij^P v vs u^T (ij|Q) v, Q={P}: err {e:.2e}", flush=True)
            assert e <= 1e-10
        # ---- (viii) symmetry of A and plan independence
        sg = sig.cpu().numpy()
        a01, a10 = float(np.vdot(X[0], sg[1])), float(np.vdot(X[1], sg[0]))
        print(f"[cfg{cfg}] (viii) <x0, A x1> = {a01:.15e}, <x1, A x0> = {a10:.15e}", flush=True)
        assert abs(a01 - a10) <= 1e-11 * max(abs(a01), np.linalg.norm(sg[0]) * 1e-3)
        c.force_plan(1, max(64, nao // 7), max(1, d["aux_chunk"] // 3))
        sig2 = c.matvec(Xd).cpu().numpy()
        e = _rel(sig2, sg)
        dd = c.dims()
        print(f"[cfg{cfg}] (viii) plan (mj=1, {dd['j_panels']} panels, pc={dd['aux_chunk']}) vs default plan: rel diff {e:.2e}", flush=True)
        assert e <= 1e-12
    finally:
        c.close()
