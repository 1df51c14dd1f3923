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
