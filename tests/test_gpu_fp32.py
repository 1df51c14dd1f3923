"""GPU parity of the single-precision mode: the tcgen05 GEMM of gemm_tc.cu on its own against FP64
products, and risp_matvec / risp_tda_solve with RISP_PRECISION_FP32_K against the FP64 oracle, inside the forward error bound of
a binary32 contraction (oracle/risp_fp32.py), with the error of the oracle's plain binary32 contraction printed beside it.  Tolerances
(DESIGN.md "FP32 mode"): every element of the K term within the bound gamma_n sum|T_ij||X||T_ab|; ||K32 - K64|| / ||K64|| <= 1e-6;
J and the diagonal unchanged; roots within 1e-4 eV of the FP64 oracle."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

HARTREE_EV = 27.211386245988
U32 = 2.0 ** -24


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    return torch


def _tcgemm(torch, A, B, C0=None, via_planes=0, seg_kb=0, shape=0):
    from paper_2603_29257_b200.binding import load_library
    lib = load_library()
    nb, M, K = A.shape
    N = B.shape[1]
    Cc = torch.zeros(nb, N, M, dtype=torch.float64, device="cuda") if C0 is None else C0.clone()
    rc = lib.risp_debug_tcgemm(M, N, K, nb, A.data_ptr(), B.data_ptr(), Cc.data_ptr(), 0 if C0 is None else 1, via_planes, seg_kb, shape, None)
    assert rc == 0
    torch.cuda.synchronize()
    return Cc


@pytest.mark.parametrize("tile_shape", [0, 1, 2])
@pytest.mark.parametrize("via_planes", [0, 1])
@pytest.mark.parametrize("shape", [(128, 256, 32, 1), (128, 16, 64, 1), (1, 1, 1, 1), (100, 200, 40, 2), (129, 257, 33, 1), (300, 423, 1496, 2),
                                   (1496, 423, 3392, 3), (640, 700, 999, 2)])
def test_tcgemm_against_fp64(torch_cuda, shape, via_planes, tile_shape):
    """Several row / column tiles, ragged tails in M, N and K (K not a multiple of the 32-element stage nor of 8), batches, both
    epilogues.  Elementwise bound of an FP32-accumulated inner product of K terms whose operands carry 24 bits:
    |err| <= (K + 6) u sum_k |a_k||b_k|  (+ 3 u |c| when the result is re-split into three bf16 planes)."""
    torch = torch_cuda
    M, N, K, nb = shape
    g = torch.Generator(device="cuda").manual_seed(M * 7 + N * 3 + K)
    A = torch.randn(nb, M, K, dtype=torch.float64, device="cuda", generator=g) * torch.exp(torch.randn(nb, M, 1, dtype=torch.float64, device="cuda", generator=g))
    B = torch.randn(nb, N, K, dtype=torch.float64, device="cuda", generator=g)
    got = _tcgemm(torch, A, B, via_planes=via_planes, shape=tile_shape)
    ref = torch.einsum("zrk,zck->zcr", A, B)
    bound = (K + 6) * U32 * torch.einsum("zrk,zck->zcr", A.abs(), B.abs()) + 3 * U32 * ref.abs()
    assert bool(torch.all((got - ref).abs() <= bound))
    assert float((got - ref).norm() / ref.norm()) <= 5e-7
    assert float((got - ref).norm() / ref.norm()) > 1e-12 or K == 1      # it is not an FP64 product in disguise


def test_tcgemm_accumulates_in_fp64(torch_cuda):
    torch = torch_cuda
    g = torch.Generator(device="cuda").manual_seed(5)
    A = torch.randn(2, 200, 300, dtype=torch.float64, device="cuda", generator=g)
    B = torch.randn(2, 150, 300, dtype=torch.float64, device="cuda", generator=g)
    C0 = 1e6 * torch.randn(2, 150, 200, dtype=torch.float64, device="cuda", generator=g)
    got = _tcgemm(torch, A, B, C0=C0)
    ref = torch.einsum("zrk,zck->zcr", A, B)
    # the large addend must not cost the product its digits: the sum over chunks is FP64
    assert float(((got - C0) - ref).norm() / ref.norm()) <= 5e-7


def _check_mode(torch, s, o, c, m):
    from workloads import trial_vectors
    from oracle.risp_fp32 import exchange_fp32, exchange_error_bound
    X = trial_vectors(s)[:m]
    Xd = torch.from_numpy(X).cuda()
    sig_ref, dg, J_ref, K_ref = o.sigma(X, parts=True)
    sig64 = c.matvec(Xd).cpu().numpy()
    c.set_precision(1)
    try:
        sig32 = c.matvec(Xd).cpu().numpy()
        K32 = c.stage("K", m)
        J32 = c.stage("J", m)
    finally:
        c.set_precision(0)
    bound = exchange_error_bound(o, X)
    assert np.all(np.abs(K32 - K_ref) <= bound + 1e-300)
    relK = np.linalg.norm(K32 - K_ref) / np.linalg.norm(K_ref)
    rel_plain = np.linalg.norm(exchange_fp32(o, X) - K_ref) / np.linalg.norm(K_ref)
    assert relK <= 1e-6
    assert relK > 1e-12                            # the mode is on
    assert np.linalg.norm(J32 - J_ref) / np.linalg.norm(J_ref) <= 1e-10
    mask = np.ones_like(X, dtype=bool); mask[np.ix_(np.arange(m), o.occK, o.virK)] = False
    assert np.array_equal(sig32[mask], sig64[mask])  # outside the window nothing changes
    assert np.linalg.norm(sig32 - sig_ref) / np.linalg.norm(sig_ref) <= 1e-6
    return relK, rel_plain


def test_fp32_mode_small(torch_cuda, sys_small_rsh, oracle_small_rsh):
    from paper_2603_29257_b200 import setup
    c = setup(sys_small_rsh, flags=1)
    try:
        _check_mode(torch_cuda, sys_small_rsh, oracle_small_rsh, c, 5)
        # chunk sizes that leave a ragged last chunk and a single-function chunk
        for pc in (1, 2):
            c.force_plan(0, 0, pc)
            _check_mode(torch_cuda, sys_small_rsh, oracle_small_rsh, c, 3)
    finally:
        c.close()


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


def test_fp32_mode_cfg2_sigma(torch_cuda, cfg2):
    s, o, c = cfg2
    relK, rel_plain = _check_mode(torch_cuda, s, o, c, 30)
    print(f"cfg2 single-precision K: rel error {relK:.3e} (plain binary32 contraction {rel_plain:.3e})")


def test_fp32_mode_cfg2_roots(cfg2):
    s, o, c = cfg2
    th_ref, _, info_ref = o.davidson(15, tol=1e-8)
    c.set_precision(1)
    try:
        omega, _, info = c.tda_solve(15, tol=1e-5)
    finally:
        c.set_precision(0)
    assert info["converged"] == 1
    d = np.abs(omega - th_ref).max() * HARTREE_EV
    print(f"cfg2 single-precision roots: max deviation {d:.3e} eV")
    assert d <= 1e-4


# ------------------------------------------------------------------------------------------------ RISP_PRECISION_FP32_JK
# Tolerance of the J term in this mode (J transforms): each of the four transform GEMMs carries the
# normwise error of a binary32 product, eps = 1e-6 (the bound used for the K term above); the two of the forward transform
# reach R~ = (P|Q)_J^-1 R, whose relative error is at most cond((P|Q)_J) times that of R, the two of the back-transform add theirs:
#     ||dJ|| / ||J|| <= (2 cond + 2) eps
_EPS32 = 1e-6


def _check_mode_jk(torch, s, o, c, m):
    from workloads import trial_vectors
    from oracle.risp_fp32 import exchange_error_bound
    X = trial_vectors(s)[:m]
    Xd = torch.from_numpy(X).cuda()
    sig_ref, dg, J_ref, K_ref = o.sigma(X, parts=True)
    c.set_precision(1)
    try:
        sig_k = c.matvec(Xd).cpu().numpy()
        K_k = c.stage("K", m)
        c.set_precision(2)
        sig32 = c.matvec(Xd).cpu().numpy()
        K32 = c.stage("K", m)
        J32 = c.stage("J", m)
    finally:
        c.set_precision(0)
    assert np.linalg.norm(K32 - K_k) <= 1e-12 * np.linalg.norm(K_k)    # the K term is that of RISP_PRECISION_FP32_K (up to the aux chunking)
    assert np.all(np.abs(K32 - K_ref) <= exchange_error_bound(o, X) + 1e-300)
    cond = np.linalg.cond(o.MJ)
    relJ = np.linalg.norm(J32 - J_ref) / np.linalg.norm(J_ref)
    assert relJ > 1e-12                                   # the mode is on (no silent FP64 fallback at these sizes)
    assert relJ <= (2 * cond + 2) * _EPS32
    rel_sig = np.linalg.norm(sig32 - sig_ref) / np.linalg.norm(sig_ref)
    assert rel_sig <= (2 * cond + 3) * _EPS32
    # sigma is assembled from the same terms as in the K-only mode: diagonal and K identical, J as checked
    assert np.linalg.norm((sig32 - sig_k) - 2 * (J32 - J_ref)) <= 1e-9 * np.linalg.norm(sig_ref)
    return relJ, rel_sig, cond


def test_fp32_jk_mode_small(torch_cuda, sys_small_rsh, oracle_small_rsh):
    from paper_2603_29257_b200 import setup
    c = setup(sys_small_rsh, flags=1)
    try:
        relJ, rel_sig, cond = _check_mode_jk(torch_cuda, sys_small_rsh, oracle_small_rsh, c, 5)
        print(f"12-atom system, single-precision J transforms: J rel error {relJ:.3e}, sigma {rel_sig:.3e}, cond(P|Q)_J {cond:.2e}")
        # sub-batches of two vectors (2, 2, 1): the planes of one sub-batch at a time
        c.force_plan(2, 0, 0)
        relJ2, _, _ = _check_mode_jk(torch_cuda, sys_small_rsh, oracle_small_rsh, c, 5)
        assert c.dims()["j_sub_batch"] == 2 and relJ2 <= 4 * relJ
        c.force_plan(0, 0, 0)
        # row panels: the transforms stay FP64 (documented fallback), the K term stays single precision
        from workloads import trial_vectors
        X = trial_vectors(sys_small_rsh)[:3]
        _, _, J_ref, _ = oracle_small_rsh.sigma(X, parts=True)
        c.force_plan(0, 16, 0)
        c.set_precision(2)
        c.matvec(torch_cuda.from_numpy(X).cuda())
        assert np.linalg.norm(c.stage("J", 3) - J_ref) / np.linalg.norm(J_ref) <= 1e-10
    finally:
        c.set_precision(0)
        c.close()


def test_fp32_jk_mode_cfg2_sigma(torch_cuda, cfg2):
    s, o, c = cfg2
    relJ, rel_sig, cond = _check_mode_jk(torch_cuda, s, o, c, 30)
    print(f"cfg2 single-precision J transforms: J rel error {relJ:.3e}, sigma {rel_sig:.3e}, cond(P|Q)_J {cond:.2e}")


def test_fp32_jk_mode_cfg2_roots(cfg2):
    s, o, c = cfg2
    th_ref, _, info_ref = o.davidson(15, tol=1e-8)
    c.set_precision(2)
    try:
        omega, _, info = c.tda_solve(15, tol=1e-5)
    finally:
        c.set_precision(0)
    assert info["converged"] == 1
    d = np.abs(omega - th_ref).max() * HARTREE_EV
    print(f"cfg2 single-precision J and K roots: max deviation {d:.3e} eV")
    assert d <= 1e-4


def test_fp32_mode_host_spilled_slices(torch_cuda, sys_small_rsh, oracle_small_rsh):
    from paper_2603_29257_b200 import setup
    c = setup(sys_small_rsh, flags=1 | 2)          # RISP_FLAG_SPILL_HALF: half of the K slices stream from pinned host memory
    try:
        _check_mode(torch_cuda, sys_small_rsh, oracle_small_rsh, c, 4)
    finally:
        c.close()


def test_fp32_mode_rejects_tddft(torch_cuda, sys_small_rsh):
    from paper_2603_29257_b200 import setup
    from paper_2603_29257_b200.binding import RispError
    torch = torch_cuda
    c = setup(sys_small_rsh, flags=8)
    try:
        c.set_precision(1)
        X = torch.zeros(1, sys_small_rsh["nocc"], c.dims()["nvir"], dtype=torch.float64, device="cuda")
        with pytest.raises(RispError):
            c.matvec_tddft(X)
        with pytest.raises(RispError):
            c.set_precision(7)
    finally:
        c.close()


def test_tcgemm_segment_length(torch_cuda):
    """The tensor core truncates when it adds an MMA result to the FP32 accumulator; accumulating the whole K range in tensor memory
    lets that bias grow linearly with K.  The record of why the kernel promotes every 32 k to register sums: the error of the
    default must be several times smaller than that of one long segment, and below cuBLAS SGEMM's on the same product."""
    torch = torch_cuda
    g = torch.Generator(device="cuda").manual_seed(1)
    A = torch.randn(1, 512, 3392, dtype=torch.float64, device="cuda", generator=g)
    B = torch.randn(1, 423, 3392, dtype=torch.float64, device="cuda", generator=g)
    ref = torch.einsum("zrk,zck->zcr", A, B)
    err = {seg: float((_tcgemm(torch, A, B, seg_kb=seg) - ref).norm() / ref.norm()) for seg in (0, 1, 4, 1000)}
    sgemm = float((torch.einsum("zrk,zck->zcr", A.float(), B.float()).double() - ref).norm() / ref.norm())
    print(f"relative error, K = 3392: default {err[0]:.2e}, 32 k {err[1]:.2e}, 128 k {err[4]:.2e}, unsegmented {err[1000]:.2e}; torch FP32 matmul {sgemm:.2e}")
    assert err[0] == err[1]
    assert err[1] < err[4] < err[1000]
    assert err[1000] > 20 * err[1]
    assert err[1] <= 5e-7


def test_fp32_mode_in_the_sharded_sigma_build(torch_cuda, sys_small_rsh, oracle_small_rsh):
    """RISP_PRECISION_FP32_K with the P-sharded sigma-build (risp_matvec_shard_begin / _end on two shards emulated on one GPU): the sum
    of the shards' partial sigma lies as close to the FP64 oracle as the unsharded single-precision product, and the J part, which
    stays FP64, is unchanged."""
    torch = torch_cuda
    from paper_2603_29257_b200 import setup
    from workloads import trial_vectors
    s, o = sys_small_rsh, oracle_small_rsh
    m = 4
    X = trial_vectors(s, m)
    Xd = torch.from_numpy(X).cuda()
    sig_ref, dg, J_ref, K_ref = o.sigma(X, parts=True)
    ctxs = [setup(s, shard_rank=r, shard_count=2) for r in range(2)]
    try:
        for c in ctxs:
            c.set_precision(1)
        R = torch.stack([c.matvec_shard_begin(Xd) for c in ctxs]).sum(0)
        sig = torch.stack([c.matvec_shard_end(Xd, R) for c in ctxs]).sum(0).cpu().numpy()
        K = sum(c.stage("K", m) for c in ctxs)
        relK = np.linalg.norm(K - K_ref) / np.linalg.norm(K_ref)
        assert 1e-12 < relK <= 1e-6
        J = (sig - dg + K) / 2.0
        assert np.linalg.norm(J - J_ref) / np.linalg.norm(J_ref) <= 1e-9
        assert np.linalg.norm(sig - sig_ref) / np.linalg.norm(sig_ref) <= 1e-6
    finally:
        for c in ctxs:
            c.close()
