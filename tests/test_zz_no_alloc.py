"""`-m gpu` test of te_matmul_noalloc (include/te.h): the split-K matrix product whose scratch memory is an array built
into the library, for callers that cannot call cudaMalloc — a frame loop that shares the GPU with a denoiser on another
stream (an allocation or a free can block the host until the whole device is idle), or a process whose memory pool
already owns all of HBM (cudaMalloc then simply fails).

The existing path, te_debug_gemm_splitk, runs the same kernel with scratch it allocates and frees on every call; the two
must agree bitwise (same kernel, same fixed summation order), and both must match an fp64 matmul within the tolerance of
tests/test_gpu_parity.py::test_gemm_splitk_vs_fp64_matmul.  The built-in array is shared by all calls and keeps the last
call's contents, so the check is made on calls IN A ROW with different tilings: the second starts from the first one's
leftovers.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity
tests.  It holds no state of its own — it passes alone in a fresh process (the first call then does the per-device
set-up) and after the other test files (set-up long done, array already used by nobody else).
"""
import numpy as np
import pytest

import workloads as W
import parity_metrics as PM

pytestmark = pytest.mark.gpu


def _operands(M, N, K, seed):
    import gpu_helpers as H
    import torch
    rng = np.random.default_rng(seed)
    a = W.f32_to_bf16_bits(rng.standard_normal((M, K)).astype(np.float32))
    b = W.f32_to_bf16_bits(rng.standard_normal((N, K)).astype(np.float32))
    ref = H.bf16_bits_to_f64(a).reshape(M, K) @ H.bf16_bits_to_f64(b).reshape(N, K).T
    ad = torch.from_numpy(a.view(np.int16)).cuda()
    bd = torch.from_numpy(b.view(np.int16)).cuda()
    return ad, bd, ref


# (M, N, K, block_n, splits): several tiles with a ragged last row block and uneven K-slices; the array filled to the last
# byte (128 partial tiles of 128 x 128); 256-wide tiles; one CTA per tile (no scratch used at all)
SHAPES = [(200, 1024, 832, 128, 4), (128, 2048, 2048, 128, 8), (100, 768, 832, 256, 3), (300, 512, 256, 128, 1)]


def test_noalloc_matches_allocating_path_on_calls_in_a_row():
    import torch
    import paper_2606_05981_b200 as te
    stream = torch.cuda.current_stream().cuda_stream
    for rep in range(2):                     # the whole sequence twice: call i+1 always finds call i's leftovers
        for M, N, K, bn, splits in SHAPES:
            assert -(-M // 128) * (N // bn) * splits * 128 * bn * 4 <= te.TE_NOALLOC_SCRATCH_BYTES
            ad, bd, ref = _operands(M, N, K, seed=M * 11 + N + splits)
            want = torch.full((M, N), float("nan"), dtype=torch.float32, device="cuda")
            te.te_debug_gemm_splitk(0, ad, bd, want, M, N, K, bn, splits)          # existing path (synchronous)
            got = torch.full((M, N), float("nan"), dtype=torch.float32, device="cuda")
            te.te_matmul_noalloc(0, ad, bd, got, M, N, K, bn, splits, stream)      # enqueues and returns
            torch.cuda.synchronize()
            got, want = got.cpu().numpy(), want.cpu().numpy()
            tag = (rep, M, N, K, bn, splits)
            assert np.isfinite(got).all(), tag
            assert np.array_equal(got, want), tag
            assert PM.rel_l2(got, ref) < 1e-5, tag
            assert np.max(np.abs(got - ref)) < 1e-4 * np.sqrt(K) * 4, tag


def test_noalloc_back_to_back_without_host_sync():
    """Two calls enqueued one after the other on one stream, no synchronisation in between: the second one's counter
    reset and kernel are ordered behind the first kernel by the stream, and neither disturbs the other's result."""
    import torch
    import paper_2606_05981_b200 as te
    stream = torch.cuda.current_stream().cuda_stream
    cases = [SHAPES[0], SHAPES[1]]
    ops = [_operands(M, N, K, seed=7 + M) for M, N, K, _, _ in cases]
    outs = [torch.full((M, N), float("nan"), dtype=torch.float32, device="cuda") for M, N, _, _, _ in cases]
    for (M, N, K, bn, splits), (ad, bd, _), c in zip(cases, ops, outs):
        te.te_matmul_noalloc(0, ad, bd, c, M, N, K, bn, splits, stream)
    torch.cuda.synchronize()
    for (M, N, K, bn, splits), (_, _, ref), c in zip(cases, ops, outs):
        out = c.cpu().numpy()
        assert PM.rel_l2(out, ref) < 1e-5
        assert np.max(np.abs(out - ref)) < 1e-4 * np.sqrt(K) * 4


def test_noalloc_refuses_what_does_not_fit():
    """One partial tile more than the array holds: a clear error code, nothing launched, the output untouched."""
    import torch
    import paper_2606_05981_b200 as te
    M, N, K, bn, splits = 128, 2048 + 128, 2048, 128, 8   # 17 tiles x 8 splits x 64 KiB > 8 MiB
    ad = torch.zeros((M, K), dtype=torch.int16, device="cuda")
    bd = torch.zeros((N, K), dtype=torch.int16, device="cuda")
    c = torch.full((M, N), 3.0, dtype=torch.float32, device="cuda")
    with pytest.raises(te.TEError) as ei:
        te.te_matmul_noalloc(0, ad, bd, c, M, N, K, bn, splits, torch.cuda.current_stream().cuda_stream)
    assert ei.value.code == te.TE_ERR_TOO_LARGE
    assert "scratch" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((c == 3.0).all())
