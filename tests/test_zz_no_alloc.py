"""crown_gemm_noalloc: the A.W contraction (Eq. 1) with its TF32 operand limbs in the library's static
device scratch, for callers that cannot call cudaMalloc.  Checked against the existing path (crown_split_tf32 x 2 +
crown_gemm on caller buffers) within the parity tolerance 1e-5 + 1e-4 |ref|, on two calls in a row that share the scratch
(the second smaller and ragged, so stale limbs of the first stay behind it), and against a float64 product.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import ctypes

import numpy as np
import pytest

ATOL, RTOL = 1e-5, 1e-4


def _excess(got, ref):
    got = np.asarray(got, np.float64); ref = np.asarray(ref, np.float64)
    return float((np.abs(got - ref) - (ATOL + RTOL * np.abs(ref))).max())


def test_limits_are_rejected_before_any_cuda_call():
    """size and shape checks need no device: they run here on the CPU box too"""
    from paper_2606_09377_b200 import load_library
    lib = load_library()
    cap = lib.crown_gemm_noalloc_max_elems()
    assert cap == 1 << 21
    one = ctypes.c_void_p(256)                                 # never dereferenced: rejected first
    # 2048 x 1024 + 1024 x 1024 elements > 2^21
    assert lib.crown_gemm_noalloc(2048, 1024, 1024, one, one, one, None) == -1
    msg = lib.crown_gemm_noalloc_error().decode()
    assert "too large" in msg and str(cap) in msg and str(3 * 1024 * 1024) in msg
    assert lib.crown_gemm_noalloc(64, 100, 64, one, one, one, None) == -1        # N < 128
    assert "N >= 128" in lib.crown_gemm_noalloc_error().decode()
    assert lib.crown_gemm_noalloc(64, 128, 30, one, one, one, None) == -1        # K % 4
    assert lib.crown_gemm_noalloc(64, 128, 64, None, one, one, None) == -1
    assert "null" in lib.crown_gemm_noalloc_error().decode()
    assert lib.crown_gemm_noalloc(64, 128, 64, one, one, ctypes.c_void_p(260), None) == -1
    assert "aligned" in lib.crown_gemm_noalloc_error().decode()


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_existing_path():
    import torch
    import workloads as W
    from paper_2606_09377_b200 import CrownContext, gemm_noalloc

    wl = W.small_mlp([16, 160, 144, 5], seed=3, B=1, eps=0.05, S=4)
    ctx = CrownContext(wl.net, 1, wl.S)                        # the existing path needs a context (caller-owned buffers)
    rng = np.random.default_rng(2606)
    # first call fills most of the scratch; the second is smaller and ragged (M, N not tile multiples), so limbs of the
    # first call stay in the array behind and between its operands; the third repeats the first shape with new values
    shapes = [(1000, 1024, 1024), (333, 260, 516), (1000, 1024, 1024)]
    free_before = None
    for it, (M, N, K) in enumerate(shapes):
        A = rng.standard_normal((M, K)).astype(np.float32)
        A[rng.random((M, K)) < 0.3] = 0.0                       # A of a backward pass is sparse through inactive ReLUs
        Wm = (rng.standard_normal((K, N)) * np.sqrt(2.0 / K)).astype(np.float32)
        A_d, W_d = torch.from_numpy(A).cuda(), torch.from_numpy(Wm).cuda()
        out = torch.full((M, N), float("nan"), device="cuda")
        if it == 2:
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info()[0]
        got = gemm_noalloc(A_d, W_d, out=out)
        if it == 2:
            torch.cuda.synchronize()
            assert torch.cuda.mem_get_info()[0] == free_before, "the call changed the device's free memory"
        ref = ctx.gemm(A_d, W_d, scheme=0)                      # crown_split_tf32 x 2 + crown_gemm
        torch.cuda.synchronize()
        got, ref = got.cpu().numpy(), ref.cpu().numpy()
        assert np.isfinite(got).all()
        assert _excess(got, ref) <= 0, f"call {it}: off the existing path by {_excess(got, ref):.3e} beyond tolerance"
        assert np.array_equal(got, ref), f"call {it}: same kernels, same order -- expected bitwise equality"
        exact = A.astype(np.float64) @ Wm.astype(np.float64)
        assert _excess(got, exact) <= 0, f"call {it}: off the float64 product by {_excess(got, exact):.3e} beyond tolerance"
    ctx.close()


@pytest.mark.gpu
def test_rejects_oversize_with_device_pointers_and_then_still_works():
    import torch
    from paper_2606_09377_b200 import CrownError, gemm_noalloc

    A = torch.zeros(2048, 1024, device="cuda"); Wm = torch.zeros(1024, 1024, device="cuda")
    with pytest.raises(CrownError, match="too large"):
        gemm_noalloc(A, Wm)
    with pytest.raises(CrownError, match="N >= 128"):
        gemm_noalloc(torch.zeros(8, 64, device="cuda"), torch.zeros(64, 64, device="cuda"))
    g = torch.Generator(device="cuda").manual_seed(5)
    A = torch.randn(128, 64, device="cuda", generator=g); Wm = torch.randn(64, 128, device="cuda", generator=g)
    got = gemm_noalloc(A, Wm).cpu().numpy()
    exact = A.cpu().numpy().astype(np.float64) @ Wm.cpu().numpy().astype(np.float64)
    assert _excess(got, exact) <= 0
