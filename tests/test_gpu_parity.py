"""GPU parity: the CUDA path (through the C ABI, paper_2603_29257_b200.binding) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances are BASELINE.json's: |d(mu nu|P)| <= 1e-12 absolute,
||sigma_gpu - sigma_ref||_F / ||sigma_ref||_F <= 1e-10 (also per term for J and K), roots within 1e-6 eV."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

HARTREE_EV = 27.211386245988


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    return torch


def _rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


# ------------------------------------------------------------------------------------------------ GEMM
@pytest.mark.parametrize("a_kc,b_kc", [(1, 1), (1, 0), (0, 1), (0, 0)])
@pytest.mark.parametrize("shape", [(129, 67, 33), (300, 257, 129), (5, 1000, 3), (128, 128, 16), (1, 1, 1)])
def test_dgemm_against_torch(torch_cuda, a_kc, b_kc, shape):
    torch = torch_cuda
    from paper_2603_29257_b200 import load_library
    lib = load_library()
    M, N, K = shape
    g = torch.Generator(device="cuda").manual_seed(M * 7 + N * 3 + K)
    A = torch.randn((M, K) if a_kc else (K, M), dtype=torch.float64, device="cuda", generator=g)
    B = torch.randn((N, K) if b_kc else (K, N), dtype=torch.float64, device="cuda", generator=g)
    Cm = torch.randn((M, N), dtype=torch.float64, device="cuda", generator=g)
    ref = 0.7 * (A if a_kc else A.T) @ (B.T if b_kc else B) - 0.3 * Cm
    out = Cm.clone()
    rc = lib.risp_debug_dgemm(M, N, K, A.data_ptr(), A.shape[1], a_kc, B.data_ptr(), B.shape[1], b_kc, out.data_ptr(), N, 0.7, -0.3,
                              1, 0, 0, 0, 1, 0, 0, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert rc == 0
    assert float((out - ref).abs().max()) <= 1e-12 * max(1.0, K ** 0.5) * float(ref.abs().max() + 1)


@pytest.mark.parametrize("a_kc,b_kc", [(1, 1), (1, 0), (0, 1), (0, 0)])
@pytest.mark.parametrize("M", [9, 20, 40, 60, 75, 90, 110, 128, 200, 423])
def test_dgemm_tma_tile_heights(torch_cuda, a_kc, b_kc, M):
    """The TMA/mbarrier kernel (even leading dimensions, aligned bases) for every tile height 16..128, ragged M, N, K, a batch,
    alpha/beta, against torch and against the cp.async kernel (variant 0) on the same operands."""
    torch = torch_cuda
    from paper_2603_29257_b200 import load_library
    lib = load_library()
    N, K, nb = 150, 70, 3
    lda = (K if a_kc else M) + 2 + ((K if a_kc else M) & 1)           # even, padded
    ldb = (K if b_kc else N) + 4 + ((K if b_kc else N) & 1)
    ra, rb = (M if a_kc else K), (N if b_kc else K)
    g = torch.Generator(device="cuda").manual_seed(1000 * M + 10 * a_kc + b_kc)
    A = torch.randn((nb, ra, lda), dtype=torch.float64, device="cuda", generator=g)
    B = torch.randn((nb, rb, ldb), dtype=torch.float64, device="cuda", generator=g)
    C0 = torch.randn((nb, M, N), dtype=torch.float64, device="cuda", generator=g)
    Aop = A[:, :, :K] if a_kc else A[:, :, :M].transpose(1, 2)
    Bop = B[:, :, :K].transpose(1, 2) if b_kc else B[:, :, :N]
    ref = 1.3 * Aop @ Bop + 0.5 * C0
    outs = []
    for variant in (1, 0):
        out = C0.clone()
        rc = lib.risp_debug_dgemm(M, N, K, A.data_ptr(), lda, a_kc, B.data_ptr(), ldb, b_kc, out.data_ptr(), N, 1.3, 0.5, nb, ra * lda, rb * ldb, M * N,
                                  variant, 0, 0, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        assert rc == 0
        outs.append(out)
    assert float((outs[0] - ref).abs().max()) <= 1e-12 * float(ref.abs().max() + 1)
    assert float((outs[0] - outs[1]).abs().max()) <= 1e-12 * float(ref.abs().max() + 1)


@pytest.mark.parametrize("no,nv", [(7, 10), (6, 9), (11, 33)])
@pytest.mark.parametrize("variant", [1, 0])
def test_dgemm_row_split_epilogue(torch_cuda, no, nv, variant):
    """Eq. 22 as the matvec launches it: one product per aux function P (batch), rows (mi, j) split by mi into M[mi][P][j][a] with
    padded leading dimensions."""
    torch = torch_cuda
    from paper_2603_29257_b200 import load_library
    lib = load_library()
    m, npc, pc = 5, 4, 6
    no_p, nv_p = no + (no & 1), nv + (nv & 1)
    X = torch.randn((m * no, nv_p), dtype=torch.float64, device="cuda")
    T = torch.randn((npc, nv, nv_p), dtype=torch.float64, device="cuda")
    Mout = torch.full((m, pc, no_p, nv_p), -7.0, dtype=torch.float64, device="cuda")
    rc = lib.risp_debug_dgemm(m * no, nv, nv, X.data_ptr(), nv_p, 1, T.data_ptr(), nv_p, 1, Mout.data_ptr(), nv_p, 1.0, 0.0,
                              npc, 0, nv * nv_p, no_p * nv_p, variant, no, pc * no_p * nv_p, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert rc == 0
    ref = torch.einsum('mjb,pab->mpja', X[:, :nv].reshape(m, no, nv), T[:, :, :nv])
    got = Mout[:, :npc, :no, :nv]
    assert float((got - ref).abs().max()) <= 1e-12 * float(ref.abs().max() + 1)
    untouched = Mout.clone(); untouched[:, :npc, :no, :nv] = -7.0
    assert bool((untouched == -7.0).all())                       # padding rows / columns / unused P slots are never written


@pytest.mark.parametrize("rows,no", [(3100, 775), (2960, 370)])
def test_dgemm_grouped_tile_order(torch_cuda, rows, no):
    """Eq. 22 with X' shared by the batch and larger than a quarter of L2: the TMA kernel walks its tiles in row groups
    (gemm_tma.cu, tile_coords<true>).  Several groups with a short last one, ragged M, N, K, the row-split epilogue; against
    torch and against the cp.async kernel (variant 0), which has no grouped order."""
    torch = torch_cuda
    from paper_2603_29257_b200 import load_library
    lib = load_library()
    l2 = torch.cuda.get_device_properties(0).L2_cache_size
    npc, pc, N = 5, 6, 290
    K = max(1402, (l2 // 4) // (rows * 8) + 2) & ~1
    assert rows * K * 8 > l2 // 4 and rows % no == 0
    m = rows // no
    no_p, ldn = no + (no & 1), N + 2
    g = torch.Generator(device="cuda").manual_seed(rows)
    X = torch.randn((rows, K), dtype=torch.float64, device="cuda", generator=g)
    T = torch.randn((npc, N, K), dtype=torch.float64, device="cuda", generator=g)
    outs = []
    for variant in (1, 0):
        Mout = torch.full((m, pc, no_p, ldn), -7.0, dtype=torch.float64, device="cuda")
        rc = lib.risp_debug_dgemm(rows, N, K, X.data_ptr(), K, 1, T.data_ptr(), K, 1, Mout.data_ptr(), ldn, 1.0, 0.0,
                                  npc, 0, N * K, no_p * ldn, variant, no, pc * no_p * ldn, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        assert rc == 0
        outs.append(Mout)
    ref = torch.einsum('mjb,pab->mpja', X.reshape(m, no, K), T)
    got = outs[0][:, :npc, :no, :N]
    assert float((got - ref).abs().max()) <= 1e-12 * K ** 0.5 * float(ref.abs().max() + 1)
    assert float((outs[0] - outs[1]).abs().max()) <= 1e-12 * K ** 0.5 * float(ref.abs().max() + 1)
    untouched = outs[0].clone(); untouched[:, :npc, :no, :N] = -7.0
    assert bool((untouched == -7.0).all())


def test_dgemm_batched(torch_cuda):
    torch = torch_cuda
    from paper_2603_29257_b200 import load_library
    lib = load_library()
    nb, M, N, K = 5, 70, 90, 50
    A = torch.randn((nb, M, K), dtype=torch.float64, device="cuda")
    B = torch.randn((nb, K, N), dtype=torch.float64, device="cuda")
    out = torch.zeros((nb, M, N), dtype=torch.float64, device="cuda")
    rc = lib.risp_debug_dgemm(M, N, K, A.data_ptr(), K, 1, B.data_ptr(), N, 0, out.data_ptr(), N, 1.0, 0.0, nb, M * K, K * N, M * N,
                              1, 0, 0, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert rc == 0
    assert float((out - A @ B).abs().max()) < 1e-11


# ------------------------------------------------------------------------------------------------ integrals
@pytest.fixture(scope="module")
def ctx1(torch_cuda, sys1):
    from paper_2603_29257_b200 import setup
    c = setup(sys1, flags=1)              # RISP_FLAG_KEEP_STAGES: J_mia stays available to the getter
    yield c
    c.close()


@pytest.fixture(scope="module")
def ctx_rsh(torch_cuda, sys_small_rsh):
    from paper_2603_29257_b200 import setup
    c = setup(sys_small_rsh, flags=1)
    yield c
    c.close()


def _shell_offsets(o):
    return np.concatenate([[0], np.cumsum(2 * o.shl_l + 1)]), np.concatenate([[0], np.cumsum(2 * o.aux_l + 1)])


@pytest.mark.parametrize("which", ["tiny", "rsh"])
def test_eri3c_every_class_both_operators(which, ctx1, oracle1, ctx_rsh, oracle_small_rsh):
    """|d(mu nu|P)| <= 1e-12 for shell triples covering all 6 pair classes x (s, p) aux, Coulomb and K operator."""
    ctx, o = (ctx1, oracle1) if which == "tiny" else (ctx_rsh, oracle_small_rsh)
    soff, aoff = _shell_offsets(o)
    rng = np.random.default_rng(17)
    by_l = {l: np.nonzero(o.shl_l == l)[0] for l in (0, 1, 2)}
    worst = 0.0
    for op, (ca, cb, w) in ((0, (1.0, 0.0, 0.0)), (1, (o.alpha, o.beta, o.omega))):
        I3 = o.int3c(o.selJ, ca, cb, w)
        for la in (0, 1, 2):
            for lb in (0, 1, 2):
                for _ in range(6):
                    si, sj = int(rng.choice(by_l[la])), int(rng.choice(by_l[lb]))
                    for ak in rng.choice(len(o.aux_l), size=4, replace=False):
                        ak = int(ak)
                        got = ctx.eri3c_shell(si, sj, ak, op)
                        ref = I3[aoff[ak]:aoff[ak + 1], soff[si]:soff[si + 1], soff[sj]:soff[sj + 1]].transpose(1, 2, 0)
                        worst = max(worst, float(np.abs(got - ref).max()))
    assert worst <= 1e-12, worst


def test_eri3c_same_shell_and_same_centre(ctx1, oracle1):
    o = oracle1
    soff, aoff = _shell_offsets(o)
    I3 = o.int3c(o.selJ)
    for si in range(0, 12):                      # shells of the first two carbons: includes (shell|shell) and same-atom pairs
        for sj in (si, 0, 5):
            for ak in (0, 1):
                got = ctx1.eri3c_shell(si, sj, ak, 0)
                ref = I3[aoff[ak]:aoff[ak + 1], soff[si]:soff[si + 1], soff[sj]:soff[sj + 1]].transpose(1, 2, 0)
                assert np.abs(got - ref).max() <= 1e-12


def test_metrics(ctx1, oracle1, ctx_rsh, oracle_small_rsh):
    for ctx, o in ((ctx1, oracle1), (ctx_rsh, oracle_small_rsh)):
        assert np.abs(ctx.stage("METRIC_J") - o.MJ).max() <= 1e-12
        assert np.abs(ctx.stage("METRIC_K") - o.MK).max() <= 1e-12


# ------------------------------------------------------------------------------------------------ sigma, per stage
@pytest.mark.parametrize("which", ["tiny", "rsh"])
def test_sigma_and_stages(which, torch_cuda, sys1, ctx1, oracle1, sys_small_rsh, ctx_rsh, oracle_small_rsh):
    torch = torch_cuda
    from workloads import trial_vectors
    s, ctx, o = (sys1, ctx1, oracle1) if which == "tiny" else (sys_small_rsh, ctx_rsh, oracle_small_rsh)
    m = 5
    X = trial_vectors(s, m)
    sig_ref, dg, J_ref, K_ref = o.sigma(X, parts=True)
    Xd = torch.from_numpy(X).cuda()
    sig = ctx.matvec(Xd).cpu().numpy()
    d = ctx.dims()
    assert (d["noccK"], d["nvirK"]) == (len(o.occK), len(o.virK))
    assert d["occK_first"] == (o.occK[0] if len(o.occK) else 0)
    # stages of the AO-direct J path against the oracle's literal Eq. 11-17
    J_ao = o.coulomb_ao_direct(X)
    R_ref = np.array([st[1] for st in o.ao_stages]).T
    Rt_ref = np.array([st[2] for st in o.ao_stages]).T
    assert _rel(ctx.stage("R", m), R_ref) <= 1e-11
    assert _rel(ctx.stage("RTILDE", m), Rt_ref) <= 1e-10       # cond (P|Q)_J ~ 5e3: ~1e-12 expected
    U = ctx.stage("U", m, sel=[2])
    assert _rel(U, o.ao_stages[2][3]) <= 1e-10
    assert _rel(ctx.stage("J", m), J_ref) <= 1e-10
    assert _rel(ctx.stage("K", m), K_ref) <= 1e-10
    assert _rel(sig, sig_ref) <= 1e-10
    assert _rel(J_ao, J_ref) <= 1e-10


def test_K_tensors(ctx_rsh, oracle_small_rsh):
    o = oracle_small_rsh
    sel = [0, len(o.selK) // 2, len(o.selK) - 1]
    Tab = ctx_rsh.stage("TAB", sel=sel)
    assert _rel(Tab, o.Bab[sel]) <= 1e-12                                   # Eq. 21 (reading G3): T_ab^P = (ab|P)
    Tij_ref = np.einsum('qij,qp->pij', o.Bij, np.linalg.inv(o.MK))[sel]     # Eq. 20
    assert _rel(ctx_rsh.stage("TIJ", sel=sel), Tij_ref) <= 1e-10


def test_sigma_structured_vectors(torch_cuda, ctx_rsh, oracle_small_rsh):
    """unit vectors e_jb inside / outside the window, and a vector supported on the window only."""
    torch = torch_cuda
    o = oracle_small_rsh
    X = np.zeros((4, o.nocc, o.nvir))
    X[0, o.occK[0], o.virK[0]] = 1.0
    X[1, 0, o.nvir - 1] = 1.0                                   # outside the window (core-like occupied, high virtual)
    X[2][np.ix_(o.occK, o.virK)] = np.random.default_rng(3).normal(size=(len(o.occK), len(o.virK)))
    X[3, o.nocc - 1, 0] = 1.0                                   # HOMO -> LUMO
    ref = o.sigma(X)
    got = ctx_rsh.matvec(torch.from_numpy(X).cuda()).cpu().numpy()
    for k in range(4):
        assert _rel(got[k], ref[k]) <= 1e-10


def test_matvec_host_equals_device(torch_cuda, sys1, ctx1):
    torch = torch_cuda
    from workloads import trial_vectors
    X = trial_vectors(sys1, 3)
    a = ctx1.matvec(torch.from_numpy(X).cuda()).cpu().numpy()
    b = ctx1.matvec_host(X)
    assert np.array_equal(a, b)


def test_matvec_rejects_bad_arguments(torch_cuda, ctx1):
    torch = torch_cuda
    from paper_2603_29257_b200 import RispError
    X = torch.zeros((2, ctx1.nocc, ctx1.nvir), dtype=torch.float64, device="cuda")
    with pytest.raises(RispError):
        ctx1.matvec(X, sigma=X)                                  # overlap
    Y = torch.empty_like(X)
    assert ctx1.lib.risp_matvec(ctx1.handle, 0, X.data_ptr(), Y.data_ptr(), None) == -1
    assert ctx1.lib.risp_matvec(ctx1.handle, -3, X.data_ptr(), Y.data_ptr(), None) == -1
    assert ctx1.lib.risp_matvec(ctx1.handle, 2, None, X.data_ptr(), None) == -1


def test_batches_beyond_32_vectors(torch_cuda, sys_small_rsh, ctx_rsh, oracle_small_rsh):
    """m > 32 is worked through in sub-batches of 32 inside the call (device and host entry points): same sigma as the oracle and,
    bit for bit, as separate calls; and a small batch after a large one is not polluted by the lanes the large one used."""
    torch = torch_cuda
    from workloads import trial_vectors
    m = 45
    X = trial_vectors(sys_small_rsh, m)
    ref = oracle_small_rsh.sigma(X)
    Xd = torch.from_numpy(X).cuda()
    sig = ctx_rsh.matvec(Xd).cpu().numpy()
    assert _rel(sig, ref) <= 1e-10
    a = ctx_rsh.matvec(Xd[:32].contiguous()).cpu().numpy(); b = ctx_rsh.matvec(Xd[32:].contiguous()).cpu().numpy()
    assert np.array_equal(sig[:32], a) and np.array_equal(sig[32:], b)
    assert np.array_equal(ctx_rsh.matvec_host(X), sig)
    for _ in range(3):                                        # 32 lanes used, then 2: the idle lanes must stay clean call after call
        ctx_rsh.matvec(Xd[:32].contiguous())
        c = ctx_rsh.matvec(Xd[:2].contiguous()).cpu().numpy()
        assert np.array_equal(c, sig[:2])


def test_no_truncation_and_empty_window(torch_cuda, sys_small_rsh):
    """cutoff <= 0 keeps everything; a cutoff below every |eps| empties the window and K vanishes."""
    torch = torch_cuda
    from paper_2603_29257_b200 import setup
    from oracle.risp_oracle import Oracle
    from workloads import trial_vectors
    X = trial_vectors(sys_small_rsh, 2)
    for cut in (0.0, 0.5 * float(np.min(np.abs(sys_small_rsh["eps"]))) * HARTREE_EV):
        s = dict(sys_small_rsh); s["cutoff_ev"] = cut
        o = Oracle(s)
        c = setup(s)
        got = c.matvec(torch.from_numpy(X).cuda()).cpu().numpy()
        assert _rel(got, o.sigma(X)) <= 1e-10
        c.close()


# ------------------------------------------------------------------------------------------------ edge cases
@pytest.mark.parametrize("m", [1, 32])
def test_batch_extremes(m, torch_cuda, sys_small_rsh, ctx_rsh, oracle_small_rsh):
    """a single trial vector, and the largest batch the ABI takes (32 = one lane per vector in the ERI passes)"""
    torch = torch_cuda
    from workloads import trial_vectors
    X = trial_vectors(sys_small_rsh, m)
    sig_ref, dg, J_ref, K_ref = oracle_small_rsh.sigma(X, parts=True)
    sig = ctx_rsh.matvec(torch.from_numpy(X).cuda()).cpu().numpy()
    assert _rel(ctx_rsh.stage("J", m), J_ref) <= 1e-10
    assert _rel(ctx_rsh.stage("K", m), K_ref) <= 1e-10
    assert _rel(sig, sig_ref) <= 1e-10


@pytest.mark.parametrize("variant", ["s_only_aux", "p_in_K_aux", "no_exchange", "zero_vector"])
def test_auxiliary_set_and_operator_variants(variant, torch_cuda, sys_small_rsh):
    """degenerate / unusual inputs: an s-only auxiliary basis (no p recursion output is used), p functions inside the K auxiliary
    set (the paper's default is s only), alpha = beta = 0 (no K term at all), and X = 0."""
    torch = torch_cuda
    from paper_2603_29257_b200 import setup
    from oracle.risp_oracle import Oracle
    from workloads import trial_vectors
    s = dict(sys_small_rsh)
    if variant == "s_only_aux":
        keep = np.nonzero(np.asarray(s["aux_l"]) == 0)[0]
        for k in ("aux_atom", "aux_l", "aux_exp", "aux_in_K"):
            s[k] = np.ascontiguousarray(np.asarray(s[k])[keep])
        s["naux"] = len(keep)
    if variant == "p_in_K_aux":
        s["aux_in_K"] = np.ones_like(np.asarray(s["aux_in_K"]))
    if variant == "no_exchange":
        s["alpha"], s["beta"] = 0.0, 0.0
    X = trial_vectors(s, 3)
    if variant == "zero_vector":
        X[1] = 0.0
    o = Oracle(s)
    sig_ref, dg, J_ref, K_ref = o.sigma(X, parts=True)
    c = setup(s, flags=1)
    try:
        sig = c.matvec(torch.from_numpy(X).cuda()).cpu().numpy()
        d = c.dims()
        assert d["nauxJ"] == o.nfun(o.selJ) and d["nauxK"] == (o.nfun(o.selK) if len(o.selK) else 0)
        assert _rel(c.stage("J", 3), J_ref) <= 1e-10
        if variant == "no_exchange":
            assert np.abs(c.stage("K", 3)).max() == 0.0 and np.abs(K_ref).max() == 0.0
        else:
            assert _rel(c.stage("K", 3), K_ref) <= 1e-10
        assert _rel(sig, sig_ref) <= 1e-10
        if variant == "zero_vector":
            assert np.abs(sig[1]).max() == 0.0
    finally:
        c.close()


# ------------------------------------------------------------------------------------------------ memory plans
@pytest.mark.parametrize("plan", [dict(mj=2, prow=0, pc=0), dict(mj=0, prow=40, pc=1), dict(mj=3, prow=24, pc=2), dict(mj=1, prow=1, pc=5)])
@pytest.mark.parametrize("which", ["tiny", "rsh"])
def test_sub_batched_and_panelled_plans(which, plan, torch_cuda, sys1, ctx1, oracle1, sys_small_rsh, ctx_rsh, oracle_small_rsh):
    """The large-system layouts on a small system: J transforms in trial-vector sub-batches and AO row panels (D + D^T per
    panel, U = P + P^T), K in small aux chunks.  Every plan must reproduce the oracle, term by term."""
    torch = torch_cuda
    from workloads import trial_vectors
    s, ctx, o = (sys1, ctx1, oracle1) if which == "tiny" else (sys_small_rsh, ctx_rsh, oracle_small_rsh)
    m = 5
    X = trial_vectors(s, m)
    sig_ref, dg, J_ref, K_ref = o.sigma(X, parts=True)
    try:
        ctx.force_plan(**plan)
        sig = ctx.matvec(torch.from_numpy(X).cuda()).cpu().numpy()
        d = ctx.dims()
        if plan["mj"]:
            assert d["j_sub_batch"] == plan["mj"]
        if plan["prow"]:
            assert d["j_panels"] > 1
        if plan["pc"]:
            assert d["aux_chunk"] == min(plan["pc"], d["nauxK"])
        assert _rel(ctx.stage("J", m), J_ref) <= 1e-10
        assert _rel(ctx.stage("K", m), K_ref) <= 1e-10
        assert _rel(sig, sig_ref) <= 1e-10
    finally:
        ctx.force_plan(0, 0, 0)


@pytest.mark.parametrize("pc", [0, 1, 2])
def test_host_spilled_K_tensors(pc, torch_cuda, sys_small_rsh, oracle_small_rsh):
    """Half of the K-tensor slices in pinned host memory, streamed through the side stream: same sigma, same
    slices, and the Davidson roots are unchanged."""
    torch = torch_cuda
    from paper_2603_29257_b200 import setup
    from workloads import trial_vectors
    o = oracle_small_rsh
    c = setup(sys_small_rsh, flags=1 | 2)             # KEEP_STAGES | SPILL_HALF
    try:
        c.force_plan(0, 0, pc)
        m = 4
        X = trial_vectors(sys_small_rsh, m)
        sig_ref, dg, J_ref, K_ref = o.sigma(X, parts=True)
        Xd = torch.from_numpy(X).cuda()
        for _ in range(3):                              # repeated calls reuse the two staging buffers
            sig = c.matvec(Xd).cpu().numpy()
        d = c.dims()
        assert 0 < d["nauxK_device"] < d["nauxK"] and d["bytes_T_host"] > 0
        assert _rel(c.stage("K", m), K_ref) <= 1e-10
        assert _rel(sig, sig_ref) <= 1e-10
        sel = [0, d["nauxK_device"] - 1, d["nauxK_device"], d["nauxK"] - 1]
        assert _rel(c.stage("TAB", sel=sel), o.Bab[sel]) <= 1e-12
        Tij_ref = np.einsum('qij,qp->pij', o.Bij, np.linalg.inv(o.MK))[sel]
        assert _rel(c.stage("TIJ", sel=sel), Tij_ref) <= 1e-10
        if pc == 0:
            w_ref = np.linalg.eigvalsh(o.full_A())[:3]
            omega, _, info = c.tda_solve(3, tol=1e-8)
            assert info["converged"] == 1 and np.abs(omega - w_ref).max() * HARTREE_EV <= 1e-6
    finally:
        c.close()


def test_small_hbm_budget_spills_and_panels(torch_cuda, sys_small_rsh, oracle_small_rsh):
    """An explicit tiny HBM budget makes the planner itself choose host spill, sub-batches and panels."""
    torch = torch_cuda
    from paper_2603_29257_b200 import setup
    from workloads import trial_vectors
    o = oracle_small_rsh
    m = 6
    X = trial_vectors(sys_small_rsh, m)
    ref = o.sigma(X)
    big = setup(sys_small_rsh, max_batch=m)
    big.matvec(torch.from_numpy(X).cuda())
    need = big.dims()["bytes_device_total"]
    big.close()
    from paper_2603_29257_b200 import RispError
    spilled = 0
    for frac in np.arange(1.0, 0.0, -0.01):                          # shrink the budget until slices go to the host, then further
        try:
            c = setup(sys_small_rsh, hbm_budget_bytes=int(frac * need), max_batch=m)
        except RispError as e:
            assert e.code == -2                                       # RISP_ENOMEM: below the minimal work space, reported, not crashed
            break
        if spilled >= 3:
            c.close()
            continue
        try:
            sig = c.matvec(torch.from_numpy(X).cuda()).cpu().numpy()
            d = c.dims()
            assert _rel(sig, ref) <= 1e-10, (frac, d)
            spilled += d["nauxK_device"] < d["nauxK"]
        finally:
            c.close()
    assert spilled > 0


# ------------------------------------------------------------------------------------------------ screening
def test_screened_pairs_are_negligible(ctx1, oracle1, torch_cuda, sys_small_rsh, oracle_small_rsh, ctx_rsh):
    for ctx, o in ((ctx1, oracle1), (ctx_rsh, oracle_small_rsh)):
        kept = {(int(a), int(b)) for a, b in ctx.stage("PAIRS")}
        kept |= {(b, a) for a, b in kept}
        soff, _ = _shell_offsets(o)
        I3 = o.int3c(o.selJ)
        for sa in range(o.nshl):
            for sb in range(sa + 1):
                if (sa, sb) not in kept:
                    assert np.abs(I3[:, soff[sa]:soff[sa + 1], soff[sb]:soff[sb + 1]]).max() < 1e-13


# ------------------------------------------------------------------------------------------------ Davidson
@pytest.mark.parametrize("which", ["tiny", "rsh"])
def test_tda_roots(which, ctx1, oracle1, ctx_rsh, oracle_small_rsh):
    ctx, o = (ctx1, oracle1) if which == "tiny" else (ctx_rsh, oracle_small_rsh)
    n = 5
    w_ref = np.linalg.eigvalsh(o.full_A())[:n]
    omega, X, info = ctx.tda_solve(n, tol=1e-8, n_guess=n if which == "tiny" else 0, want_vectors=True)
    assert info["converged"] == 1
    assert np.abs(omega - w_ref).max() * HARTREE_EV <= 1e-6
    Xh = X.cpu().numpy()
    res = o.sigma(Xh) - omega[:, None, None] * Xh
    assert np.linalg.norm(res.reshape(n, -1), axis=1).max() < 1e-7


@pytest.mark.parametrize("flags", [0, 1, 2])
def test_tda_restart_path(flags, ctx1, oracle1):
    """restart path with the subspace fully cached in HBM (0), fully streamed from pinned host memory (1), and mixed (2)"""
    w_ref = np.linalg.eigvalsh(oracle1.full_A())[:3]
    omega, _, info = ctx1.tda_solve(3, tol=1e-8, max_sub=30, max_iter=300, flags=flags)
    assert info["restarts"] > 0 and info["converged"] == 1
    assert np.abs(omega - w_ref).max() * HARTREE_EV <= 1e-6
    if flags == 1:
        assert info["cached_vectors"] == 0 and info["bytes_h2d"] > 0
    if flags == 2:
        assert info["cached_vectors"] == 5 and info["bytes_h2d"] > 0
    if flags == 0:
        assert info["bytes_h2d"] == 0


# ------------------------------------------------------------------------------------------------ 100-atom config
@pytest.fixture(scope="module")
def cfg2(torch_cuda):
    from workloads import make_system
    from oracle.risp_oracle import Oracle
    from paper_2603_29257_b200 import setup
    s = make_system(2)
    o = Oracle(s)
    o.build()
    c = setup(s, flags=1)
    yield s, o, c
    c.close()


def test_cfg2_sigma_parity(torch_cuda, cfg2):
    """BASELINE.json configs[1] at full size and bench batch (m = 30): several tiles and ragged tails everywhere."""
    torch = torch_cuda
    from workloads import trial_vectors
    s, o, c = cfg2
    X = trial_vectors(s)
    sig_ref, dg, J_ref, K_ref = o.sigma(X, parts=True)
    sig = c.matvec(torch.from_numpy(X).cuda()).cpu().numpy()
    m = X.shape[0]
    assert _rel(c.stage("J", m), J_ref) <= 1e-10
    assert _rel(c.stage("K", m), K_ref) <= 1e-10
    assert _rel(sig, sig_ref) <= 1e-10


def test_cfg2_roots(cfg2):
    s, o, c = cfg2
    th_ref, _, info_ref = o.davidson(15, tol=1e-8)
    assert info_ref["converged"]
    omega, _, info = c.tda_solve(15, tol=1e-8)
    assert info["converged"] == 1
    assert np.abs(omega - th_ref).max() * HARTREE_EV <= 1e-6
    # "no lower root was missed": 20 roots from a different, perturbed start must reproduce the lowest 15
    omega2, _, info2 = c.tda_solve(20, tol=1e-8, flags=4, n_guess=50)
    assert info2["converged"] == 1
    assert np.abs(omega2[:15] - omega).max() * HARTREE_EV <= 1e-6
    assert omega2[15] >= omega[14]


def test_cfg2_every_dropped_shell_pair_is_negligible(cfg2):
    """Reading G14: the pair screen is a magnitude estimate, so it is checked a posteriori on ALL ~61 000 shell pairs the 100-atom
    system drops: the largest |(mu nu|P)| over every aux function, from the unscreened oracle integrals, must stay below 1e-13."""
    s, o, c = cfg2
    d = c.dims()
    kept = np.zeros((o.nshl, o.nshl), dtype=bool)
    pr = c.stage("PAIRS")
    kept[pr[:, 0], pr[:, 1]] = True; kept[pr[:, 1], pr[:, 0]] = True
    assert d["n_shell_pairs"] - d["n_shell_pairs_kept"] > 50000
    soff = np.concatenate([[0], np.cumsum(2 * o.shl_l + 1)])
    ao_kept = np.repeat(np.repeat(kept, 2 * o.shl_l + 1, axis=0), 2 * o.shl_l + 1, axis=1)
    worst = 0.0
    for s0 in range(0, o.naux_shl, 16):
        I3 = o.int3c(o.selJ[s0:s0 + 16])
        worst = max(worst, float(np.abs(I3[:, ~ao_kept]).max()))
    assert worst < 1e-13, worst


# ------------------------------------------------------------------------------------------------ solver options
def test_solver_blocks_chunks_and_fp32_host_store(ctx_rsh, oracle_small_rsh):
    """The lean solver footprint on a small system: roots worked through in chunks of max_block (the 3000-atom layout), subspace
    fully streamed / mixed, single-precision host store -- same roots as the dense eigenvalues."""
    o = oracle_small_rsh
    n = 6
    w_ref = np.linalg.eigvalsh(o.full_A())[:n]
    for kw in (dict(max_block=2), dict(max_block=4, flags=1), dict(max_block=5, flags=2, max_sub=25, max_iter=300),
               dict(max_block=1, flags=1, max_sub=18, max_iter=400)):
        omega, X, info = ctx_rsh.tda_solve(n, tol=1e-8, want_vectors=True, **kw)
        assert info["converged"] == 1 and info["block"] == kw["max_block"], (kw, info)
        assert np.abs(omega - w_ref).max() * HARTREE_EV <= 1e-6, kw
        Xh = X.cpu().numpy()
        res = o.sigma(Xh) - omega[:, None, None] * Xh
        assert np.linalg.norm(res.reshape(n, -1), axis=1).max() < 1e-7
        if kw.get("max_sub"):
            assert info["restarts"] > 0
    # FP32 host store: V exact (rounded before the sigma-build), W rounded on its way to the host; residual floor ~1e-7
    omega, X, info = ctx_rsh.tda_solve(n, tol=2e-6, want_vectors=True, flags=1 | 8, max_block=3, max_sub=30, max_iter=300)
    assert info["converged"] == 1 and info["cached_vectors"] == 0 and info["restarts"] > 0
    assert np.abs(omega - w_ref).max() * HARTREE_EV <= 1e-5
    o64, _, i64 = ctx_rsh.tda_solve(n, tol=2e-6, flags=1, max_block=3, max_sub=30, max_iter=300)
    assert info["bytes_h2d"] < 0.75 * i64["bytes_h2d"] * max(1.0, info["iterations"] / i64["iterations"])


def test_solver_many_roots_and_large_guess(ctx1, oracle1):
    """nroots = 64 (RISP_MAX_ROOTS) and n_guess = 128: blocks larger than one sigma-build batch are chunked."""
    w = np.linalg.eigvalsh(oracle1.full_A())
    omega, _, info = ctx1.tda_solve(64, tol=1e-7, max_iter=200)
    assert info["converged"] == 1 and np.abs(omega - w[:64]).max() * HARTREE_EV <= 1e-6
    omega, _, info = ctx1.tda_solve(10, tol=1e-7, n_guess=128, max_sub=400)
    assert info["converged"] == 1 and np.abs(omega - w[:10]).max() * HARTREE_EV <= 1e-6


def test_solver_out_of_memory_is_reported_and_leak_free(torch_cuda, ctx_rsh):
    torch = torch_cuda
    from paper_2603_29257_b200 import RispError
    ctx_rsh.tda_solve(3, tol=1e-6)                            # work space of the context exists from here on
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    with pytest.raises(RispError) as e:
        ctx_rsh.tda_solve(3, tol=1e-6, device_budget_bytes=4096)
    assert e.value.code == -2
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    omega, _, info = ctx_rsh.tda_solve(3, tol=1e-6)           # and the context still works
    assert info["converged"] == 1
    assert torch.cuda.mem_get_info()[0] == free0


def test_aux_shell_order_s_first_then_p(torch_cuda, sys_small_rsh, oracle_small_rsh):
    """Aux shells not grouped by atom (all s shells, then all p shells) with p functions in the K set and the K tensors built in
    small runs: every slice must land in its own place (later runs used to overwrite earlier slices with zeros)."""
    torch = torch_cuda
    from paper_2603_29257_b200 import setup
    from oracle.risp_oracle import Oracle
    from workloads import trial_vectors
    s = dict(sys_small_rsh)
    order = np.argsort(np.asarray(s["aux_l"]), kind="stable")
    for k in ("aux_atom", "aux_l", "aux_exp"):
        s[k] = np.ascontiguousarray(np.asarray(s[k])[order])
    s["aux_in_K"] = np.ones(len(order), dtype=np.uint8)
    X = trial_vectors(s, 3)
    o = Oracle(s)
    sig_ref, dg, J_ref, K_ref = o.sigma(X, parts=True)
    c = setup(s, flags=1 | 4)
    try:
        sig = c.matvec(torch.from_numpy(X).cuda()).cpu().numpy()
        assert _rel(c.stage("J", 3), J_ref) <= 1e-10
        assert _rel(c.stage("K", 3), K_ref) <= 1e-10
        assert _rel(sig, sig_ref) <= 1e-10
        sel = list(range(0, c.dims()["nauxK"], 3))
        assert _rel(c.stage("TAB", sel=sel), o.Bab[sel]) <= 1e-12
    finally:
        c.close()
