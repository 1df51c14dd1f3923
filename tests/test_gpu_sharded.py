"""P-sharded sigma-build (row f1; paper_2603_29257_b200/sharded.py, risp_matvec_shard_begin / _end): the shards of one problem are
emulated one after the other on ONE GPU (separate contexts; the sums that the two all-reduces would form are formed here), and
their sum must reproduce the oracle and the unsharded context -- per term, so that J (pairs sharded) and K (aux slices sharded)
are both covered."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


@pytest.mark.parametrize("count", [2, 3])
@pytest.mark.parametrize("which", ["tiny", "rsh"])
def test_sharded_sigma_equals_unsharded(which, count, sys1, oracle1, sys_small_rsh, oracle_small_rsh):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    from paper_2603_29257_b200 import setup
    from workloads import trial_vectors
    s, o = (sys1, oracle1) if which == "tiny" else (sys_small_rsh, oracle_small_rsh)
    m = 5
    X = trial_vectors(s, m)
    Xd = torch.from_numpy(X).cuda()
    sig_ref, dg, J_ref, K_ref = o.sigma(X, parts=True)
    ctxs = [setup(s, shard_rank=r, shard_count=count) for r in range(count)]
    full = setup(s)
    try:
        d0 = full.dims()
        dd = [c.dims() for c in ctxs]
        assert sum(d["n_shell_pairs_kept"] for d in dd) == d0["n_shell_pairs_kept"]
        assert sum(d["nauxK"] for d in dd) == d0["nauxK"]
        Rs = [c.matvec_shard_begin(Xd) for c in ctxs]
        R = torch.stack(Rs).sum(0)                                   # the first all-reduce
        parts = [c.matvec_shard_end(Xd, R) for c in ctxs]
        sig = torch.stack(parts).sum(0).cpu().numpy()                # the second all-reduce
        assert _rel(sig, sig_ref) <= 1e-10
        full.matvec(Xd)
        assert _rel(R[:, :m].cpu().numpy(), full.stage("R", m)) <= 1e-12
        assert float(R[:, m:].abs().max()) == 0.0
        # per term: K is what the shards' K slices sum to (the last matvec of each context left its K' behind)
        K = sum(c.stage("K", m) for c in ctxs)
        assert _rel(K, K_ref) <= 1e-10
        J = (sig - dg + K) / 2.0
        assert _rel(J, J_ref) <= 1e-9
        # rank 0 carries the diagonal, the others none
        e = np.zeros((1, o.nocc, o.nvir)); e[0, 0, o.nvir - 1] = 1.0
        ed = torch.from_numpy(e).cuda()
        Rz = torch.stack([c.matvec_shard_begin(ed) for c in ctxs]).sum(0)
        got = torch.stack([c.matvec_shard_end(ed, Rz) for c in ctxs]).sum(0).cpu().numpy()
        assert _rel(got, o.sigma(e)) <= 1e-10
    finally:
        for c in ctxs + [full]:
            c.close()
