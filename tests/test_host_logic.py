"""CPU-only checks of the product's host side: the C-ABI library loads and exports every symbol of include/risp.h,
argument validation works without a GPU, the host eigen solver of the Davidson subspace matches LAPACK, and the
N > 1 bench path (per-rank trial-vector shards, max-over-ranks timing) works under gloo with world_size 2."""
import os
import re
import subprocess
import sys

import ctypes as C
import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2603_29257_b200.build import build
    build()
    from paper_2603_29257_b200 import load_library
    return load_library()


def test_library_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "risp.h")).read() + open(os.path.join(ROOT, "include", "risp_debug.h")).read()
    declared = set(re.findall(r"\b(risp_[a-z0-9_]+)\s*\(", hdr))
    assert {"risp_setup", "risp_matvec", "risp_matvec_host", "risp_tda_solve", "risp_destroy", "risp_last_error", "risp_get_dims",
            "risp_get_timings", "risp_eri3c_shell", "risp_get_stage"} <= declared
    assert {"risp_debug_dgemm", "risp_debug_sym_eig_lowest", "risp_debug_force_plan", "risp_debug_yardstick"} <= declared
    for name in declared:
        assert hasattr(lib, name), name
    # and nothing is exported that no header declares
    out = subprocess.run(["nm", "-D", "--defined-only", os.path.join(ROOT, "paper_2603_29257_b200", "librisp.so")], capture_output=True, text=True).stdout
    exported = {ln.split()[-1] for ln in out.splitlines() if " T " in ln and ln.split()[-1].startswith("risp_") and "_Z" not in ln}
    assert exported <= declared, exported - declared


def test_setup_validates_arguments_without_a_gpu(lib, sys1):
    from paper_2603_29257_b200 import RispContext, RispError
    bad = dict(sys1); bad["shl_l"] = np.array(sys1["shl_l"]).copy(); bad["shl_l"][0] = 3
    with pytest.raises(RispError) as e:
        RispContext(bad)
    assert e.value.code == -1 and "l outside" in str(e.value)
    bad = dict(sys1); bad["nao"] = sys1["nao"] + 1
    with pytest.raises(RispError) as e:
        RispContext(bad)
    assert e.value.code == -1
    assert lib.risp_matvec(None, 1, None, None, None) == -1
    assert b"no context" in lib.risp_last_error(None)


def test_no_cpu_fallback_when_library_missing(monkeypatch):
    import paper_2603_29257_b200.binding as b
    monkeypatch.setattr(b, "_LIB", None)
    monkeypatch.setattr(b, "library_path", lambda: "/nonexistent/librisp.so")
    with pytest.raises(b.RispError):
        b.load_library()


@pytest.mark.parametrize("n", [1, 2, 5, 40, 150, 315])
def test_host_lowest_eigenpairs_against_lapack(lib, n):
    """the Davidson loop's projected eigenproblem: lowest nv pairs by inverse iteration, incl. clustered / degenerate spectra"""
    rng = np.random.default_rng(100 + n)
    A = rng.normal(size=(n, n)); A = A + A.T
    if n == 40:
        Q, _ = np.linalg.qr(rng.normal(size=(n, n)))
        A = Q @ np.diag(np.repeat(np.arange(8.0), 5) + 1e-9 * rng.normal(size=n)) @ Q.T
        A = 0.5 * (A + A.T)
    if n == 315:                                  # Davidson-like: dominant diagonal with meV-spaced lowest levels
        A = np.diag(np.sort(rng.uniform(0.15, 2.0, size=n))) + 1e-3 * A
        A[np.arange(15), np.arange(15)] = 0.15 + 3e-5 * np.arange(15)
    nv = min(n, 15)
    w = np.zeros(n); z = np.zeros((n, n))
    assert lib.risp_debug_sym_eig_lowest(n, nv, A.ctypes.data, w.ctypes.data, z.ctypes.data) == 0
    scale = max(1.0, np.abs(A).max()) * n
    assert np.abs(w - np.linalg.eigvalsh(A)).max() < 1e-12 * scale
    Z = z[:, :nv]
    assert np.abs(Z.T @ Z - np.eye(nv)).max() < 1e-10
    assert np.abs(A @ Z - Z * w[None, :nv]).max() < 1e-11 * scale


_WORKER = r"""
import os, sys, numpy as np, torch, torch.distributed as dist
sys.path.insert(0, sys.argv[1])
from workloads import make_system, trial_vectors
dist.init_process_group("gloo")
rank = dist.get_rank()
s = make_system(1)
X = trial_vectors(s, base_seed=260329257 + 17 * rank)          # the per-rank shard bench.py uses
t = torch.tensor([1.0 + rank, float(np.abs(X).sum())], dtype=torch.float64)
g = [torch.zeros_like(t) for _ in range(dist.get_world_size())]
dist.all_gather(g, t)
mx = t.clone(); dist.all_reduce(mx, op=dist.ReduceOp.MAX)
assert float(mx[0]) == dist.get_world_size()                   # max-over-ranks timing
assert abs(float(g[0][1]) - float(g[1][1])) > 1e-6             # ranks really hold different trial vectors
dist.barrier(); dist.destroy_process_group()
print("ok", rank)
"""


def test_trial_vector_sharding_world_size_2_gloo(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(_WORKER)
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
                        "--master-port", "29533", str(w), ROOT], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr
    assert r.stdout.count("ok") == 2


def test_bench_reference_arm_prints_the_contract_line():
    """`bench.py --impl reference` (the CPU oracle as the reference arm) on the tiny config: one JSON line with the contract's keys"""
    import json
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    for k in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert k in line, k
    assert line["impl"] == "reference" and line["value"] > 0 and line["config"]["workload"].startswith("cfg1")
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0


_SHARD_WORKER = r"""
import os, sys, numpy as np, torch, torch.distributed as dist
sys.path.insert(0, sys.argv[1])
from workloads import make_system, trial_vectors
from oracle.risp_oracle import Oracle
from paper_2603_29257_b200.sharded import sharded_matvec, shard_of_pair, shard_of_aux_centre
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
s = make_system(3, counts=(6, 4, 1, 1))
o = Oracle(s); o.build()
X = trial_vectors(s, 3)


class OracleShard:
    # a CPU stand-in for one rank's sharded context, built on the oracle: AO pairs and whitened K aux functions dealt round robin
    def __init__(self):
        self.I3 = o.int3c(o.selJ)
        n = o.nao
        iu = np.array([(a, b) for a in range(n) for b in range(a + 1)])
        mine = np.array([shard_of_pair(k, world) == rank for k in range(len(iu))])
        self.mask = np.zeros((n, n), dtype=bool)
        self.mask[iu[mine, 0], iu[mine, 1]] = True
        self.full = np.zeros((n, n)); self.full[self.mask] = 1.0
        self.w = self.full + np.tril(self.full, -1).T                  # (mu, nu) and (nu, mu) of an owned lower-triangular pair
        self.kfun = [p for p in range(o.BijW.shape[0]) if shard_of_aux_centre(p, world) == rank]

    def matvec_shard_begin(self, Xt):
        Xn = Xt.numpy()
        D = [o.Co @ Xn[k] @ o.Cv.T for k in range(len(Xn))]
        R = np.zeros((self.I3.shape[0], 32))
        for k, Dk in enumerate(D):
            R[:, k] = np.einsum('qmn,mn->q', self.I3, Dk * self.w)
        return torch.from_numpy(R)

    def matvec_shard_end(self, Xt, R):
        Xn = Xt.numpy(); m = len(Xn)
        Rt = np.linalg.solve(o.MJ, R.numpy()[:, :m])
        sig = np.zeros_like(Xn)
        for k in range(m):
            U = np.einsum('pmn,p->mn', self.I3, Rt[:, k]) * self.w
            sig[k] = 2.0 * (o.Co.T @ U @ o.Cv)
        Xw = Xn[:, o.occK][:, :, o.virK]
        Kw = np.zeros_like(Xw)
        for P in self.kfun:
            Kw += o.BijW[P][None] @ (Xw @ o.BabW[P].T)
        sig[np.ix_(np.arange(m), o.occK, o.virK)] -= Kw
        if rank == 0:
            sig += o.delta[None] * Xn
        return torch.from_numpy(sig)


sig = sharded_matvec(OracleShard(), torch.from_numpy(X)).numpy()
ref = o.sigma(X)
err = float(np.linalg.norm(sig - ref) / np.linalg.norm(ref))
assert err < 1e-11, err
dist.barrier(); dist.destroy_process_group()
print("ok", rank, err)
"""


def test_p_sharded_driver_world_size_2_gloo(tmp_path):
    """The two collectives of the P-sharded sigma-build (all-reduce of R between the passes, all-reduce of sigma) under gloo with
    two ranks; each rank's context is an oracle-backed stand-in that owns every second AO pair and every second K aux function."""
    w = tmp_path / "shard_worker.py"
    w.write_text(_SHARD_WORKER)
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
                        "--master-port", "29547", str(w), ROOT], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stdout + r.stderr
    assert r.stdout.count("ok") == 2
