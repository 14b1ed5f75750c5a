"""hclDgemmNoAlloc (include/hclooc.h): the in-core DGEMM for callers that cannot allocate -- the persistent stream-K kernel with
its scratch in a static device array -- against the existing path (hclDgemmAsync / hclDgemmAsyncEx, whose stream-K launches take
their scratch from a cudaMalloc'ed pool), on calls in a row that share the array.

Bars: the same kernel with the same work split sums in the same order, so against hclDgemmAsyncEx(variant -1) the bits are equal;
against hclDgemmAsync (which may pick another launch variant, hence another order of summation) the gate of the other tests,
|got - ref| <= 1e-13 * D with D = |alpha| |A||B| + |beta| |C0| (G14); integer data: equal to the oracle bit for bit.

The file is named to be collected last: the suite runs with pytest -x.
"""
import numpy as np
import pytest

import oracle
import synthgen

pytestmark = pytest.mark.gpu
RTOL = 1e-13


@pytest.fixture(scope="module")
def H():
    import paper_1808_05056_b200 as H
    import torch
    assert torch.cuda.is_available()
    torch.cuda.init()
    return H


def to_dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def operands(M, N, K, seed, dist, beta):
    lda, ldb, ldc = K + (K % 2) + 2, N + (N % 2) + 4, N + (N % 2) + 6
    A = np.full((M, lda), np.nan); B = np.full((K, ldb), np.nan); C0 = np.full((M, ldc), np.nan)
    synthgen.fill(A, seed, "A", dist, cols=K); synthgen.fill(B, seed, "B", dist, cols=N); synthgen.fill(C0, seed, "C", dist, cols=N)
    if beta == 0.0:
        C0[:, :N] = np.nan                               # beta == 0: C is not read
    return A, B, C0, lda, ldb, ldc


CASES = [
    # M, N, K, alpha, beta, dist
    (1500, 2100, 700, 1.5, -0.5, "uniform"),             # 204 tiles: all of them in the stream-K tail, cut among 148 CTAs; ragged edges
    (384, 640, 4100, 1.0, 0.5, "int"),                   # 15 tiles cut along K among several CTAs each
    (2048, 2432, 512, 2.0, 0.0, "uniform"),              # 2 whole waves + 8 tiles; beta == 0 over NaN
    (1500, 2100, 700, 1.5, -0.5, "uniform"),             # the first shape again, after the others have used the array
]


def test_no_alloc_matches_the_existing_path_on_calls_in_a_row(H):
    import torch
    s = torch.cuda.current_stream()
    prepared = []
    for i, (M, N, K, alpha, beta, dist) in enumerate(CASES):
        A, B, C0, lda, ldb, ldc = operands(M, N, K, 90 + i % 3, dist, beta)
        prepared.append((A, B, C0, lda, ldb, ldc, to_dev(A), to_dev(B), to_dev(C0), to_dev(C0), to_dev(C0)))
    # one call first: it loads the module (static array included) and the kernel, so that what follows can be watched for allocations
    M, N, K, alpha, beta, dist = CASES[0]
    A, B, C0, lda, ldb, ldc, dA, dB, dC_na, dC_old, dC_sk = prepared[0]
    warm = to_dev(C0)
    H.hclDgemmNoAlloc(M, N, K, alpha, dA, lda, dB, ldb, beta, warm, ldc, s)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    # the calls in a row, nothing between them: every one starts from whatever the one before left in the array
    for (M, N, K, alpha, beta, dist), (A, B, C0, lda, ldb, ldc, dA, dB, dC_na, dC_old, dC_sk) in zip(CASES, prepared):
        H.hclDgemmNoAlloc(M, N, K, alpha, dA, lda, dB, ldb, beta, dC_na, ldc, s)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "device memory was allocated during hclDgemmNoAlloc calls"
    for (M, N, K, alpha, beta, dist), (A, B, C0, lda, ldb, ldc, dA, dB, dC_na, dC_old, dC_sk) in zip(CASES, prepared):
        H.hclDgemmAsync(M, N, K, alpha, dA, lda, dB, ldb, beta, dC_old, ldc, s)                       # the existing path
        H.hclDgemmAsyncEx(M, N, K, alpha, dA, lda, dB, ldb, beta, dC_sk, ldc, s, variant=-1)          # its stream-K variant
        torch.cuda.synchronize()
        got, old, sk = dC_na.cpu().numpy(), dC_old.cpu().numpy(), dC_sk.cpu().numpy()
        assert np.isnan(got[:, N:]).all(), "padding columns of C written"
        assert not np.isnan(got[:, :N]).any()
        D = np.abs(alpha) * (np.abs(A[:, :K]) @ np.abs(B[:, :N])) + (np.abs(beta) * np.abs(C0[:, :N]) if beta != 0.0 else 0.0)
        ok, worst = oracle.within_gate(got[:, :N], old[:, :N], D, RTOL)
        assert ok, f"{M}x{N}x{K}: worst |no_alloc - existing| / D = {worst:.3e}"
        assert np.array_equal(got[:, :N].view(np.uint64), sk[:, :N].view(np.uint64)), "same kernel, same split: the bits must agree"
        ref = C0[:, :N].copy()
        Dref = oracle.dgemm(alpha, A[:, :K].copy(), B[:, :N].copy(), beta, ref, want_denominator=True)
        if dist == "int":
            assert np.array_equal(got[:, :N], ref)
        else:
            ok, worst = oracle.within_gate(got[:, :N], ref, Dref, RTOL)
            assert ok, f"{M}x{N}x{K}: worst |no_alloc - oracle| / D = {worst:.3e}"
    # the very first call (before any other had used the array) and the same call after three others: the same bits
    assert np.array_equal(warm.cpu().numpy().view(np.uint64), prepared[0][8].cpu().numpy().view(np.uint64))


def test_no_alloc_limits_degenerate_cases_and_errors(H):
    import torch
    s = torch.cuda.current_stream()
    assert H.hclDgemmNoAllocScratchBytes() == 38798592 == (2 * 148 * 128 * 128 * 8 + 296 * 4 + 255) // 256 * 256
    M, N, K = 300, 260, 96
    A, B, C0, lda, ldb, ldc = operands(M, N, K, 95, "int", 2.0)
    dA, dB, dC = to_dev(A), to_dev(B), to_dev(C0)
    # beyond the stated maximum: refused before anything is launched or read
    for shape in ((1 << 31, N, K), (M, 1 << 31, K), (M, N, 1 << 31), ((1 << 31) - 1, (1 << 31) - 1, K)):
        with pytest.raises(H.HclError) as e:
            H.hclDgemmNoAlloc(*shape, 1.0, dA, lda, dB, ldb, 0.0, dC, ldc, s)
        assert e.value.status == 7 and "maximum" in str(e.value)
    cases = [((-1, N, K, 1.0, dA, lda, dB, ldb, 0.0, dC, ldc), -1), ((M, -1, K, 1.0, dA, lda, dB, ldb, 0.0, dC, ldc), -2),
             ((M, N, -1, 1.0, dA, lda, dB, ldb, 0.0, dC, ldc), -3), ((M, N, K, 1.0, None, lda, dB, ldb, 0.0, dC, ldc), -5),
             ((M, N, K, 1.0, dA, K - 1, dB, ldb, 0.0, dC, ldc), -6), ((M, N, K, 1.0, dA, lda, None, ldb, 0.0, dC, ldc), -7),
             ((M, N, K, 1.0, dA, lda, dB, N - 1, 0.0, dC, ldc), -8), ((M, N, K, 1.0, dA, lda, dB, ldb, 0.0, None, ldc), -10),
             ((M, N, K, 1.0, dA, lda, dB, ldb, 0.0, dC, N - 1), -11), ((M, N, K, 1.0, dA, lda + 1, dB, ldb, 0.0, dC, ldc), 5),
             ((M, N, K, 1.0, dA.data_ptr() + 8, lda, dB, ldb, 0.0, dC, ldc), 5)]
    for args, code in cases:
        with pytest.raises(H.HclError) as e:
            H.hclDgemmNoAlloc(*args, s)
        assert e.value.status == code
    torch.cuda.synchronize()
    assert np.array_equal(dC.cpu().numpy()[:, :N], C0[:, :N])                      # none of the refused calls touched C
    H.hclDgemmNoAlloc(0, N, K, 1.0, dA, lda, dB, ldb, 2.0, dC, ldc, s)             # empty: nothing to do
    H.hclDgemmNoAlloc(M, N, 0, 1.0, None, 2, None, 2, 2.0, dC, ldc, s)             # K == 0: C = beta * C, A and B not referenced
    H.hclDgemmNoAlloc(M, N, K, 0.0, None, 2, None, 2, 0.5, dC, ldc, s)             # alpha == 0: the same
    torch.cuda.synchronize()
    got = dC.cpu().numpy()
    assert np.array_equal(got[:, :N], C0[:, :N]) and np.isnan(got[:, N:]).all()    # 2.0 * 0.5 = 1
    H.hclDgemmNoAlloc(M, N, K, 1.0, dA, lda, dB, ldb, 2.0, dC, ldc, s)             # 9 tiles, 3 k blocks each: fewer CTAs than SMs
    torch.cuda.synchronize()
    ref = C0[:, :N].copy()
    oracle.dgemm(1.0, A[:, :K].copy(), B[:, :N].copy(), 2.0, ref)
    assert np.array_equal(dC.cpu().numpy()[:, :N], ref)


def test_no_alloc_call_can_be_captured_in_a_cuda_graph(H):
    """What the entry point is for: once a device is set up (its first call), a call enqueues a memset and a kernel and nothing
    else, so it can be recorded into a CUDA graph and replayed."""
    import torch
    M, N, K, alpha, beta = 1000, 1300, 520, 1.0, 1.0
    A, B, C0, lda, ldb, ldc = operands(M, N, K, 96, "int", beta)
    dA, dB, dC = to_dev(A), to_dev(B), to_dev(C0)
    side = torch.cuda.Stream()
    first = to_dev(C0)
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        H.hclDgemmNoAlloc(M, N, K, alpha, dA, lda, dB, ldb, 0.0, first, ldc, side)           # set-up outside the capture
    side.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        H.hclDgemmNoAlloc(M, N, K, alpha, dA, lda, dB, ldb, beta, dC, ldc, torch.cuda.current_stream())
    torch.cuda.synchronize()
    assert np.array_equal(dC.cpu().numpy()[:, :N], C0[:, :N]), "capture must not run the call"
    g.replay(); g.replay(); g.replay()                                               # C += A B, three times
    torch.cuda.synchronize()
    ref = C0[:, :N].copy()
    for _ in range(3):
        oracle.dgemm(alpha, A[:, :K].copy(), B[:, :N].copy(), beta, ref)
    assert np.array_equal(dC.cpu().numpy()[:, :N], ref)
