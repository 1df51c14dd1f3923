"""`risp_tcgemm_static` -- the entry point that allocates nothing (operand planes in a static device array, include/risp.h) --
against the existing allocating path `risp_debug_tcgemm` and against the FP64 product, on two calls in a row.  The second call is
smaller and ragged, so whatever the first call left in the shared scratch lies inside and beyond its planes.  Tolerance: the one
tests/test_gpu_fp32.py uses for this GEMM (relative 5e-7 against FP64); against the allocating path the result must agree to the
same tolerance (it is the same arithmetic on the same kernels, so the difference is expected to be exactly zero).
Collected last on purpose (the file name sorts after every other test file)."""
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    return torch


def _allocating_path(torch, A, B, C0=None):
    from paper_2603_29257_b200.binding import load_library
    lib = load_library()
    M, K = A.shape
    N = B.shape[0]
    Cc = torch.zeros(N, M, dtype=torch.float64, device="cuda") if C0 is None else C0.clone()
    rc = lib.risp_debug_tcgemm(M, N, K, 1, A.data_ptr(), B.data_ptr(), Cc.data_ptr(), 0 if C0 is None else 1, 0, 0, 0, None)
    assert rc == 0
    torch.cuda.synchronize()
    return Cc


def test_static_scratch_gemm_two_calls_in_a_row(torch_cuda):
    torch = torch_cuda
    from paper_2603_29257_b200.binding import tcgemm_static
    g = torch.Generator(device="cuda").manual_seed(29257)
    calls = [(300, 423, 1496, False), (129, 67, 33, True)]        # (M, N, K, accumulate): several tiles, then a ragged small one
    data = []
    for M, N, K, acc in calls:
        A = torch.randn(M, K, dtype=torch.float64, device="cuda", generator=g)
        B = torch.randn(N, K, dtype=torch.float64, device="cuda", generator=g)
        C0 = torch.randn(N, M, dtype=torch.float64, device="cuda", generator=g) if acc else None
        data.append((A, B, C0, torch.empty(N, M, dtype=torch.float64, device="cuda")))
    # both calls back to back on one stream, nothing in between
    for A, B, C0, out in data:
        if C0 is not None:
            out.copy_(C0)
        tcgemm_static(A, B, C_out=out, accumulate=C0 is not None)
    torch.cuda.synchronize()
    for A, B, C0, out in data:
        prod = A.unsqueeze(0) @ B.t().unsqueeze(0)                                   # [1][M][N] FP64
        ref64 = prod[0].t() + (C0 if C0 is not None else 0)
        ref_alloc = _allocating_path(torch, A, B, C0)
        scale = float((prod[0]).norm())
        assert float((out - ref64).norm()) / scale <= 5e-7
        assert float((out - ref_alloc).norm()) / scale <= 5e-7
        assert float((out - ref64).norm()) > 0.0                                     # the single-precision path ran, not an FP64 product


def test_static_scratch_gemm_allocates_nothing_and_rejects_oversize(torch_cuda):
    torch = torch_cuda
    from paper_2603_29257_b200.binding import tcgemm_static, RispError, STATIC_SCRATCH_BYTES
    g = torch.Generator(device="cuda").manual_seed(7)
    A = torch.randn(256, 512, dtype=torch.float64, device="cuda", generator=g)
    B = torch.randn(200, 512, dtype=torch.float64, device="cuda", generator=g)
    out = torch.empty(200, 256, dtype=torch.float64, device="cuda")
    tcgemm_static(A, B, C_out=out)                 # first use on this device: module load, symbol address, function attributes
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        tcgemm_static(A, B, C_out=out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0                          # cudaMemGetInfo: no device memory taken or returned by the calls
    ref = (A @ B.t()).t()
    assert float((out - ref).norm() / ref.norm()) <= 5e-7
    # the largest problem that fits and the first that does not: 6 (M + N) ceil8(K) bytes against the 16 MiB array
    K = 1024
    rows = STATIC_SCRATCH_BYTES // (6 * K)         # M + N
    M = rows // 2
    A2 = torch.randn(M, K, dtype=torch.float64, device="cuda", generator=g)
    B2 = torch.randn(rows - M, K, dtype=torch.float64, device="cuda", generator=g)
    big = tcgemm_static(A2, B2)
    torch.cuda.synchronize()
    ref2 = (A2 @ B2.t()).t()
    assert float((big - ref2).norm() / ref2.norm()) <= 5e-7
    B3 = torch.randn(rows - M + 1, K, dtype=torch.float64, device="cuda", generator=g)
    with pytest.raises(RispError) as ei:
        tcgemm_static(A2, B3)
    assert "static scratch holds" in str(ei.value)
    with pytest.raises(RispError):
        tcgemm_static(A2[:0], B2)
