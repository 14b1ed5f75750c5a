"""GPU parity for hclooc_dtrmm and hclooc_dsymm (the level-3 BLAS routines whose operand is a triangle of a stored matrix;
PAPER.md:412) against the CPU oracles of oracle/level3_oracle.c / oracle.dsymm.

Bar: the DGEMM gate (|C_gpu - C_ref| <= 1e-13 * D, D the absolute-value product; G14, G25); integer data bit for bit.
The part of the stored matrix that the routine must not reference (the other triangle, a unit diagonal) is NaN throughout.
"""
import numpy as np
import pytest

import oracle
import synthgen

pytestmark = pytest.mark.gpu
MiB = 1 << 20
RTOL = 1e-13


@pytest.fixture(scope="module")
def H():
    import paper_1808_05056_b200 as H
    import torch
    assert torch.cuda.is_available()
    torch.cuda.init()
    return H


def host(H, rows, cols, seed, name, dist, pad=0):
    X = H.HostMatrix(rows, cols, cols + pad)
    X.array[...] = np.nan
    synthgen.fill(X.array, seed, name, dist, cols=cols)
    return X


def poison_tri(Aview, uplo, unit):
    n = Aview.shape[0]
    other = np.triu(np.ones((n, n), bool), 1) if uplo == 0 else np.tril(np.ones((n, n), bool), -1)
    Aview[other] = np.nan
    if unit:
        Aview[np.arange(n), np.arange(n)] = np.nan


def dense_tri(Aview, uplo, trans, unit):
    T = np.tril(Aview) if uplo == 0 else np.triu(Aview)
    if unit:
        T = T - np.diag(np.diag(T)) + np.eye(T.shape[0])
    return T.T if trans else T


@pytest.mark.parametrize("side", [0, 1])
@pytest.mark.parametrize("uplo", [0, 1])
@pytest.mark.parametrize("trans", [0, 1])
@pytest.mark.parametrize("unit", [0, 1])
@pytest.mark.parametrize("M,N,alpha,dist,pad,budget", [
    (300, 260, 1.0, "uniform", 3, 2 * MiB),         # a few blocks, ragged everywhere
    (517, 389, -2.0, "int", 0, 3 * MiB),            # exact
    (1000, 700, 0.5, "uniform", 2, 6 * MiB),        # several column slabs and row bands
    (64, 1, 1.0, "int", 0, 1 * MiB),
])
def test_dtrmm_matches_oracle(H, side, uplo, trans, unit, M, N, alpha, dist, pad, budget):
    n = M if side == 0 else N
    A = host(H, n, n, 101, "A", dist, pad)
    B = host(H, M, N, 101, "B", dist, pad)
    T = dense_tri(np.nan_to_num(A.view.copy()), uplo, trans, unit)
    poison_tri(A.view, uplo, unit)
    B0 = B.view.copy()
    ref = B0.copy()
    oracle.dtrmm(side, uplo, trans, unit, alpha, A.view, ref)
    st = H.hclooc_dtrmm(None, side, uplo, trans, unit, M, N, alpha, A, A.ld, B, B.ld, budget)
    got = B.view.copy()
    assert st.plan.workspace_bytes <= budget and st.n_kernels >= 1
    assert not np.isnan(got).any() and np.isnan(B.array[:, N:]).all()
    if dist == "int":
        Ti, Bi = T.astype(np.int64), B0.astype(np.int64)
        want = (alpha * (Ti @ Bi if side == 0 else Bi @ Ti)).astype(np.float64)
        assert np.array_equal(ref, want)
        assert np.array_equal(got, want), f"{np.count_nonzero(got != want)} elements differ"
    else:
        D = abs(alpha) * (np.abs(T) @ np.abs(B0) if side == 0 else np.abs(B0) @ np.abs(T))
        ok, worst = oracle.within_gate(got, ref, D, RTOL)
        assert ok, worst


def test_dtrmm_degenerate_and_errors(H):
    M, N = 200, 100
    A = host(H, M, M, 102, "A", "uniform")
    B = host(H, M, N, 102, "B", "uniform")
    B.view[3, 4] = np.nan
    H.hclooc_dtrmm(None, 0, 0, 0, 0, M, N, 0.0, None, M, B, B.ld, 1 * MiB)              # alpha == 0: zeros, A not read
    assert np.array_equal(B.view, np.zeros((M, N)))
    synthgen.fill(B.array, 103, "B", "uniform", cols=N)
    keep = B.view.copy()
    H.hclooc_dtrmm(None, 0, 0, 0, 0, 0, N, 1.0, A, M, B, B.ld, 1 * MiB)
    H.hclooc_dtrmm(None, 1, 0, 0, 0, M, 0, 1.0, A, M, B, B.ld, 1 * MiB)
    assert np.array_equal(B.view, keep)
    bad = [((2, 0, 0, 0, M, N, 1.0, A, M, B, N), -2), ((0, 2, 0, 0, M, N, 1.0, A, M, B, N), -3), ((0, 0, 2, 0, M, N, 1.0, A, M, B, N), -4),
           ((0, 0, 0, 2, M, N, 1.0, A, M, B, N), -5), ((0, 0, 0, 0, -1, N, 1.0, A, M, B, N), -6), ((0, 0, 0, 0, M, -1, 1.0, A, M, B, N), -7),
           ((0, 0, 0, 0, M, N, 1.0, None, M, B, N), -9), ((0, 0, 0, 0, M, N, 1.0, A, M - 1, B, N), -10), ((0, 0, 0, 0, M, N, 1.0, A, M, None, N), -11),
           ((0, 0, 0, 0, M, N, 1.0, A, M, B, N - 1), -12)]
    for args, code in bad:
        with pytest.raises(H.HclError) as e:
            H.hclooc_dtrmm(None, *args, 1 * MiB)
        assert e.value.status == code, (args[:6], e.value.status)
    assert np.array_equal(B.view, keep)


@pytest.mark.parametrize("side", [0, 1])
@pytest.mark.parametrize("uplo", [0, 1])
@pytest.mark.parametrize("M,N,alpha,beta,dist,pad,budget", [
    (300, 260, 1.0, 0.5, "uniform", 3, 2 * MiB),
    (517, 389, 2.0, -1.0, "int", 0, 3 * MiB),
    (900, 1100, -0.75, 0.0, "uniform", 1, 6 * MiB),   # beta == 0: C (NaN) is not read in the first pass
    (96, 112, 1.0, 1.0, "int", 0, 400 * 1024),
])
def test_dsymm_matches_oracle(H, side, uplo, M, N, alpha, beta, dist, pad, budget):
    n = M if side == 0 else N
    A = host(H, n, n, 111, "A", dist, pad)
    B = host(H, M, N, 111, "B", dist, pad)
    C = host(H, M, N, 111, "C", dist, pad)
    poison_tri(A.view, uplo, 0)
    if beta == 0.0:
        C.view[...] = np.nan
    ref = np.nan_to_num(C.view.copy()) if beta == 0.0 else C.view.copy()
    D = oracle.dsymm(side, uplo, alpha, A.view, B.view, beta, ref, want_denominator=True)
    st = H.hclooc_dsymm(None, side, uplo, M, N, alpha, A, A.ld, B, B.ld, beta, C, C.ld, budget)
    got = C.view.copy()
    assert st.plan.workspace_bytes <= budget and st.bytes_d2h == 2 * M * N * 8
    assert not np.isnan(got).any() and np.isnan(C.array[:, N:]).all()
    if dist == "int":
        assert np.array_equal(got, ref), f"{np.count_nonzero(got != ref)} elements differ"
    else:
        ok, worst = oracle.within_gate(got, ref, D, RTOL)
        assert ok, worst


def test_dsymm_large_and_errors(H):
    """4000 x 3000 under 64 MiB: both passes run many blocks per column; both triangles of the same symmetric matrix give results
    within the gate of each other and of the oracle."""
    M, N = 4000, 3000
    A = host(H, M, M, 112, "A", "uniform")
    S = np.tril(A.view) + np.tril(A.view, -1).T
    B = host(H, M, N, 112, "B", "uniform")
    C = host(H, M, N, 112, "C", "uniform")
    C0 = C.view.copy()
    ref = C0.copy()
    D = oracle.dgemm(1.5, S, B.view, -0.5, ref, want_denominator=True)
    for uplo in (0, 1):
        A.view[...] = S
        poison_tri(A.view, uplo, 0)
        C.view[...] = C0
        H.hclooc_dsymm(None, 0, uplo, M, N, 1.5, A, A.ld, B, B.ld, -0.5, C, C.ld, 64 * MiB)
        ok, worst = oracle.within_gate(C.view, ref, D, RTOL)
        assert ok, (uplo, worst)
    keep = C.view.copy()
    bad = [((2, 0, M, N, 1.0, A, M, B, N, 1.0, C, N), -2), ((0, 2, M, N, 1.0, A, M, B, N, 1.0, C, N), -3), ((0, 0, -1, N, 1.0, A, M, B, N, 1.0, C, N), -4),
           ((0, 0, M, -1, 1.0, A, M, B, N, 1.0, C, N), -5), ((0, 0, M, N, 1.0, None, M, B, N, 1.0, C, N), -7), ((0, 0, M, N, 1.0, A, M - 1, B, N, 1.0, C, N), -8),
           ((0, 0, M, N, 1.0, A, M, None, N, 1.0, C, N), -9), ((0, 0, M, N, 1.0, A, M, B, N - 1, 1.0, C, N), -10), ((0, 0, M, N, 1.0, A, M, B, N, 1.0, None, N), -12),
           ((0, 0, M, N, 1.0, A, M, B, N, 1.0, C, N - 1), -13), ((0, 0, M, N, 1.0, A, M, B, N, 1.0, B, N), -12)]
    for args, code in bad:
        with pytest.raises(H.HclError) as e:
            H.hclooc_dsymm(None, *args, 8 * MiB)
        assert e.value.status == code, (args[:4], e.value.status)
    assert np.array_equal(C.view, keep)
