"""GPU parity for the in-core calls on DEVICE pointers (reading G26: what hclDgemmAsync is to hclooc_dgemm):
hclDtrsmAsync (both sides) and hclDpotrfAsync -- the recursive device phases of hclooc_dtrsm[_side] / hclooc_dpotrf as calls of their
own -- against the CPU oracles, and the two substitution block kernels (one thread per right-hand side for large panels, four
lanes per right-hand side for small ones: trsm_sm100.cu) against each other, bit for bit.

Bars as in test_gpu_dtrsm.py / test_gpu_factor.py: integer data with power-of-two diagonals exact; otherwise the backward gates
(oracle.dtrsm_gate, oracle.dpotrf_gate) and, the operands being well conditioned, 1e-12 of the largest entry forward.
"""
import numpy as np
import pytest

import oracle
import synthgen

pytestmark = pytest.mark.gpu
FWD_RTOL = 1e-12


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


def triangle(n, seed, dist, uplo, unit):
    """A well-conditioned triangular matrix with NaN in the other triangle (never read) and, for a unit diagonal, on the diagonal:
    integer entries -2..2 with a diagonal in {1, 2, 4} (dist == "int"), else uniform entries scaled by 1/n with a diagonal near 1."""
    G = synthgen.fill_numpy(n, n, seed, "A", dist)
    if dist == "int":
        T = np.clip(G, -2, 2) - np.diag(np.diag(np.clip(G, -2, 2))) + np.diag(2.0 ** (np.abs(np.diag(G)) % 3))
    else:
        T = G / n + np.diag(1.0 + 0.5 * np.abs(np.diag(G)))
    T = np.tril(T) if uplo == 0 else np.triu(T)
    stored = T.copy()
    stored[np.triu(np.ones((n, n), bool), 1) if uplo == 0 else np.tril(np.ones((n, n), bool), -1)] = np.nan
    if unit:
        T = T - np.diag(np.diag(T)) + np.eye(n)
        stored[np.arange(n), np.arange(n)] = np.nan
    return T, stored


def pad_cols(x, pad):
    out = np.full((x.shape[0], x.shape[1] + pad), np.nan)
    out[:, :x.shape[1]] = x
    return out


@pytest.mark.parametrize("split", ["0", "1"])
@pytest.mark.parametrize("side,uplo,trans,unit", [(0, 0, 0, 0), (0, 1, 1, 1), (0, 1, 0, 0), (1, 0, 1, 0), (1, 1, 0, 1), (1, 0, 0, 0)])
@pytest.mark.parametrize("M,N,alpha,dist", [
    (384, 200, 1.0, "int"),             # three 128-blocks (left) / a ragged 72-column block (right)
    (300, 640, -2.0, "uniform"),        # ragged blocks on the left, five whole ones on the right
    (1024, 77, 0.5, "int"),
])
def test_dtrsm_async_matches_oracle_with_either_block_kernel(H, monkeypatch, split, side, uplo, trans, unit, M, N, alpha, dist):
    import torch
    monkeypatch.setenv("HCLOOC_TRSM_SPLIT", split)         # 0: one thread per right-hand side always, 1: four lanes always
    n = M if side == 0 else N
    T, stored = triangle(n, 31, dist, uplo, unit)
    opT = T.T if trans else T
    X0 = synthgen.fill_numpy(M, N, 32, "B", dist)
    if dist == "int":
        B0 = (opT.astype(np.int64) @ X0.astype(np.int64) if side == 0 else X0.astype(np.int64) @ opT.astype(np.int64)).astype(np.float64)
    else:
        B0 = X0
    ref = B0.copy()
    clean = np.nan_to_num(stored)
    (oracle.dtrsm if side == 0 else oracle.dtrsm_right)(uplo, trans, unit, alpha, clean, ref)
    lda, ldb = n + (n % 2) + 2, N + (N % 2) + 4
    dA, dB = to_dev(pad_cols(stored, lda - n)), to_dev(pad_cols(B0, ldb - N))
    H.hclDtrsmAsync(side, uplo, trans, unit, M, N, alpha, dA, lda, dB, ldb, torch.cuda.current_stream())
    torch.cuda.synchronize()
    out = dB.cpu().numpy()
    got = out[:, :N]
    assert np.isnan(out[:, N:]).all() and not np.isnan(got).any()
    if dist == "int":
        assert np.array_equal(ref, alpha * X0) and np.array_equal(got, alpha * X0), f"{np.count_nonzero(got != alpha * X0)} elements differ"
    else:
        assert np.abs(got - ref).max() <= FWD_RTOL * np.abs(ref).max()
        if side == 0:
            res, den = oracle.dtrsm_residual(uplo, trans, unit, alpha, clean, B0, got)
            assert (res <= oracle.dtrsm_gate(M) * den).all(), float((res / den).max())


@pytest.mark.parametrize("side,uplo,trans,unit,M,N", [(0, 0, 0, 0, 640, 1000), (0, 1, 1, 0, 300, 517), (1, 0, 1, 0, 1000, 640), (1, 1, 0, 1, 517, 300)])
def test_the_two_substitution_kernels_give_the_same_bits(H, monkeypatch, side, uplo, trans, unit, M, N):
    """Same operations on every element in the same order: one thread per right-hand side and four lanes per right-hand side
    must agree bit for bit, ragged blocks and unaligned panels included."""
    import torch
    n = M if side == 0 else N
    T, stored = triangle(n, 33, "uniform", uplo, unit)
    B0 = synthgen.fill_numpy(M, N, 34, "B", "uniform")
    lda, ldb = n + (n % 2), N + (N % 2) + 2
    outs = []
    for split in ("0", "1"):
        monkeypatch.setenv("HCLOOC_TRSM_SPLIT", split)
        dA, dB = to_dev(pad_cols(stored, lda - n)), to_dev(pad_cols(B0, ldb - N))
        H.hclDtrsmAsync(side, uplo, trans, unit, M, N, 1.5, dA, lda, dB, ldb, torch.cuda.current_stream())
        torch.cuda.synchronize()
        outs.append(dB.cpu().numpy()[:, :N].copy())
    assert np.array_equal(outs[0].view(np.uint64), outs[1].view(np.uint64)), f"{np.count_nonzero(outs[0] != outs[1])} elements differ"


@pytest.mark.parametrize("uplo", [0, 1])
@pytest.mark.parametrize("N,dist", [(128, "int"), (300, "uniform"), (1000, "int"), (2049, "uniform")])
def test_dpotrf_async_matches_oracle(H, uplo, N, dist):
    import torch
    if dist == "int":
        G = synthgen.fill_numpy(N, N, 35, "A", "int")
        L0 = np.tril(np.clip(G, -2, 2), -1) + np.diag(2.0 ** (np.abs(np.diag(G)) % 3))
        S = (L0.astype(np.int64) @ L0.astype(np.int64).T).astype(np.float64)
    else:
        K = max(8, N // 4)
        G = synthgen.fill_numpy(N, K, 35, "A", "uniform")
        S = G @ G.T / K + np.eye(N)
    other = np.triu(np.ones((N, N), bool), 1) if uplo == 0 else np.tril(np.ones((N, N), bool), -1)
    A0 = S.copy()
    A0[other] = np.nan                                                    # the other triangle is never read ...
    ref = A0.copy()
    assert oracle.dpotrf(uplo, ref) == 0
    lda = N + (N % 2) + 2
    dA = to_dev(pad_cols(A0, lda - N))
    d_info = torch.full((1,), -7, dtype=torch.int64, device="cuda")
    H.hclDpotrfAsync(uplo, N, dA, lda, d_info, torch.cuda.current_stream())
    torch.cuda.synchronize()
    assert int(d_info.item()) == 0
    out = dA.cpu().numpy()
    got = out[:, :N]
    assert np.isnan(got[other]).all() and np.isnan(out[:, N:]).all()      # ... nor written
    tri = ~other
    if dist == "int":
        want = L0 if uplo == 0 else L0.T
        assert np.array_equal(got[tri], want[tri]), f"{np.count_nonzero(got[tri] != want[tri])} elements differ"
    else:
        res, den = oracle.dpotrf_residual(uplo, S, np.nan_to_num(got))
        assert (res <= oracle.dpotrf_gate(N) * den).all(), float((res / den).max() / oracle.dpotrf_gate(N))
        assert np.abs(got[tri] - ref[tri]).max() <= FWD_RTOL * np.abs(ref[tri]).max()
    # a matrix that is not positive definite: info = the order of the first bad leading minor
    k = N // 2
    bad = S.copy(); bad[k, k] = -1.0
    dA = to_dev(pad_cols(bad, lda - N))
    H.hclDpotrfAsync(uplo, N, dA, lda, d_info, torch.cuda.current_stream())
    torch.cuda.synchronize()
    assert int(d_info.item()) == k + 1 == oracle.dpotrf(uplo, bad.copy())
