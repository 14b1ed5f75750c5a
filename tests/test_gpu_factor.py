"""GPU parity for the routines built on the out-of-core DGEMM: hclooc_dpotrf (Cholesky) and
hclooc_dtrsm_side (DTRSM with side = Right), against the CPU oracles of oracle/level3_oracle.c.

Bars (G23, G24): integer data whose exact result is integer (power-of-two diagonals: the kernels multiply by a
reciprocal) -> bit for bit; otherwise the elementwise backward bound every order of summation satisfies,
|A - L L^T| <= gamma_(N+2) |L||L^T| (oracle.dpotrf_gate, residual in long double) resp. |alpha B - X op(T)| <= gamma_(N+2) (...),
AND, the operands being well conditioned by construction, agreement with the oracle's own result to 1e-12 of the largest entry.
"""
import numpy as np
import pytest

import oracle
import synthgen

pytestmark = pytest.mark.gpu
MiB = 1 << 20
FWD_RTOL = 1e-12


@pytest.fixture(scope="module")
def H():
    import paper_1808_05056_b200 as H
    import torch
    assert torch.cuda.is_available()
    torch.cuda.init()
    return H


def other_triangle(n, uplo):
    return np.triu(np.ones((n, n), bool), 1) if uplo == 0 else np.tril(np.ones((n, n), bool), -1)


def spd_host(H, N, seed, dist, pad=0):
    """A symmetric positive definite N x N matrix in pinned memory with a KNOWN factor where dist == "int":
    integer L0 (entries -2..2 below the diagonal, diagonal in {1, 2, 4}), A := L0 L0^T exactly.  Float: G G^T / K + I with G the
    seeded uniform N x K generator matrix (well conditioned: eigenvalues in about [1, 1 + 4/3])."""
    A = H.HostMatrix(N, N, N + pad)
    A.array[...] = np.nan
    if dist == "int":
        G = synthgen.fill_numpy(N, N, seed, "A", "int")
        L0 = np.tril(np.clip(G, -2, 2), -1) + np.diag(2.0 ** (np.abs(np.diag(G)) % 3))
        A.view[...] = (L0.astype(np.int64) @ L0.astype(np.int64).T).astype(np.float64)
        return A, L0
    K = max(8, N // 4)
    G = synthgen.fill_numpy(N, K, seed, "A", "uniform")
    A.view[...] = G @ G.T / K + np.eye(N)
    return A, None


# ------------------------------------------------------------------------------------------------ the block kernels' recursion
@pytest.mark.parametrize("uplo", [0, 1])
@pytest.mark.parametrize("N,dist,pad,budget", [
    (1, "uniform", 0, 1 * MiB),
    (77, "int", 1, 1 * MiB),                 # one block, smaller than 128
    (128, "uniform", 0, 1 * MiB),            # exactly one potrf block
    (300, "uniform", 2, 8 * MiB),            # one panel: recursion over 128-blocks with a ragged last one
    (1000, "int", 0, 32 * MiB),              # one panel of 1000: three levels of recursion, exact
    (1000, "uniform", 3, 2 * MiB),           # two resident panels of 64 columns: 16 panels, look-ahead updates from host and device
    (1500, "int", 1, 8 * MiB),               # panels of 128 columns, K up to 1280 in the out-of-core updates, exact
    (2049, "uniform", 0, 16 * MiB),          # odd size: panels of 384, a ragged last one of 129
])
def test_dpotrf_matches_oracle(H, uplo, N, dist, pad, budget):
    A, L0 = spd_host(H, N, 71, dist, pad)
    other = other_triangle(N, uplo)
    A.view[other] = np.nan                                   # the other triangle is never read ...
    A0 = A.view.copy()
    ref = A0.copy()
    assert oracle.dpotrf(uplo, ref) == 0
    info, st = H.hclooc_dpotrf(None, uplo, N, A, A.ld, budget)
    got = A.view.copy()
    assert info == 0 and st.plan.workspace_bytes <= budget
    NB, panel_bytes = H.hclooc_dpotrf_plan(N, budget)
    assert (st.plan.nb if uplo == 0 else st.plan.mb) == NB and st.plan.n_steps == -(-N // NB)
    assert np.isnan(got[other]).all() and np.isnan(A.array[:, N:]).all()      # ... nor written; padding untouched
    tri = ~other
    assert not np.isnan(got[tri]).any()
    if dist == "int":
        want = L0 if uplo == 0 else L0.T
        assert np.array_equal(ref[tri], want[tri])                              # the oracle, against the hidden factor
        assert np.array_equal(got[tri], want[tri]), f"{np.count_nonzero(got[tri] != want[tri])} elements differ"
    else:
        res, den = oracle.dpotrf_residual(uplo, np.nan_to_num(A0), np.nan_to_num(got))
        assert (res <= oracle.dpotrf_gate(N) * den).all(), float((res / den).max() / oracle.dpotrf_gate(N))
        assert np.abs(got[tri] - ref[tri]).max() <= FWD_RTOL * np.abs(ref[tri]).max()


def test_dpotrf_not_positive_definite_degenerate_and_errors(H):
    N = 700
    A, _ = spd_host(H, N, 72, "uniform")
    keep = A.view.copy()
    for k in (0, 5, 300, 699):
        bad = keep.copy(); bad[k, k] = -1.0                                     # the leading minor of order k+1 is not positive definite
        A.view[...] = bad
        ref = bad.copy()
        want = oracle.dpotrf(0, ref)
        info, st = H.hclooc_dpotrf(None, 0, N, A, A.ld, 2 * MiB)
        assert info == want == k + 1
        NB = st.plan.nb
        done = (k // NB) * NB                                                   # the panels before the failing one are complete
        assert np.array_equal(A.view[:, done + NB:], bad[:, done + NB:])        # the panels after the failing one are unchanged
        assert np.array_equal(np.triu(A.view, 1), np.triu(bad, 1))              # the other triangle keeps its bits
        if done:
            low = np.tril(np.ones((k, done), bool))                             # rows the oracle completed, columns we completed
            assert np.abs(A.view[:k, :done][low] - ref[:k, :done][low]).max() <= 1e-12
    info, _ = H.hclooc_dpotrf(None, 1, 0, None, 1, 1 * MiB)                    # N == 0
    assert info == 0
    cases = [((2, N, A, N), -2), ((0, -1, A, N), -3), ((0, N, None, N), -4), ((0, N, A, N - 1), -5)]
    for (uplo, n, a, lda), code in cases:
        with pytest.raises(H.HclError) as e:
            H.hclooc_dpotrf(None, uplo, n, a, lda, 1 * MiB)
        assert e.value.status == code
    with pytest.raises(H.HclError) as e:
        H.hclooc_dpotrf(None, 0, N, A, N, 64 * 1024)                             # not even a 32-column panel fits
    assert e.value.status == 1
    pageable = np.eye(64)
    with pytest.raises(H.HclError) as e:
        H.hclooc_dpotrf(None, 0, 64, pageable, 64, 1 * MiB)
    assert e.value.status == 2


@pytest.mark.parametrize("uplo", [0, 1])
def test_dpotrf_large_panels_of_4096(H, uplo):
    """N = 9000 under 2 GiB: panels of 4096 columns (two full, one ragged), the updates are real out-of-core DGEMMs with the
    triangle mask, the diagonal blocks recurse five levels.  The residual gate on sampled rows and columns, forward agreement with
    scipy (an independent factorization; the oracle itself would take minutes at this size)."""
    import scipy.linalg as sl
    N = 9000
    A, _ = spd_host(H, N, 73, "uniform")
    other = other_triangle(N, uplo)
    S = A.view.copy()
    A.view[other] = np.nan
    info, st = H.hclooc_dpotrf(None, uplo, N, A, A.ld, 2048 * MiB)
    assert info == 0 and (st.plan.nb if uplo == 0 else st.plan.mb) == 4096 and st.plan.n_steps == 3 and st.plan.n_sets == 2
    got = np.nan_to_num(A.view)
    assert np.isnan(A.view[other]).all()
    ref = sl.cholesky(S, lower=(uplo == 0))
    assert np.abs(got - ref).max() <= FWD_RTOL * np.abs(ref).max()
    rng = np.random.default_rng(2)
    rows = np.unique(np.concatenate([[0, 127, 128, 4095, 4096, 8191, 8192, N - 1], rng.integers(0, N, 30)]))
    cols = np.unique(np.concatenate([[0, 4095, 4096, N - 1], rng.integers(0, N, 30)]))
    res, den = oracle.dpotrf_residual(uplo, S, got, rows, cols)
    assert (res <= oracle.dpotrf_gate(N) * den).all(), float((res / den).max() / oracle.dpotrf_gate(N))


# ------------------------------------------------------------------------------------------------ DTRSM, side = Right
def tri_host(H, n, seed, dist, pad=0):
    A = H.HostMatrix(n, n, n + pad)
    A.array[...] = np.nan
    synthgen.fill(A.array, seed, "A", dist, cols=n)
    synthgen.shape_triangular(A.view, dist)
    if dist == "int":                                       # power-of-two diagonal: the kernel multiplies by the reciprocal
        d = np.arange(n)
        A.view[d, d] = np.sign(A.view[d, d]) * 2.0 ** (d % 3)
    return A


def dense_op(Aview, uplo, trans, unit):
    T = np.tril(Aview) if uplo == 0 else np.triu(Aview)
    if unit:
        T = T - np.diag(np.diag(T)) + np.eye(T.shape[0])
    return T.T if trans else T


@pytest.mark.parametrize("uplo", [0, 1])
@pytest.mark.parametrize("trans", [0, 1])
@pytest.mark.parametrize("unit", [0, 1])
@pytest.mark.parametrize("M,N,alpha,dist,pad,budget", [
    (200, 300, 1.0, "uniform", 3, 1 * MiB),        # NB = 160..: two block columns, ragged second
    (517, 1000, 2.0, "int", 0, 2 * MiB),           # several block columns and row bands, exact
    (64, 129, -0.5, "uniform", 1, 64 * MiB),       # one block column: no out-of-core update
    (1, 77, 1.0, "int", 0, 512 * 1024),            # a single row
    (700, 1500, 1.5, "uniform", 2, 6 * MiB),
    (700, 2500, 1.5, "uniform", 2, 64 * MiB),      # two resident block columns of 1024 with the look-ahead, ragged third one
    (517, 2100, 2.0, "int", 1, 48 * MiB),          # the same, exact
])
def test_dtrsm_right_matches_oracle(H, uplo, trans, unit, M, N, alpha, dist, pad, budget):
    A = tri_host(H, N, 81, dist, pad)
    B = H.HostMatrix(M, N, N + pad)
    B.array[...] = np.nan
    synthgen.fill(B.array, 81, "B", dist, cols=N)
    if dist == "int":
        X0 = B.view.copy().astype(np.int64)
        T = dense_op(np.nan_to_num(A.view), uplo, trans, unit)
        B.view[...] = X0.astype(np.float64) @ T             # exact: small integers times powers of two
    other = other_triangle(N, uplo)
    A.view[other] = np.nan
    if unit:
        A.view[np.arange(N), np.arange(N)] = np.nan
    B0 = B.view.copy()
    ref = B0.copy()
    oracle.dtrsm_right(uplo, trans, unit, alpha, A.view, ref)
    st = H.hclooc_dtrsm_side(None, H.HCL_SIDE_RIGHT, uplo, trans, unit, M, N, alpha, A, A.ld, B, B.ld, budget)
    got = B.view.copy()
    assert st.plan.workspace_bytes <= budget and st.n_kernels >= 1
    assert st.plan.n_sets == (2 if budget >= 48 * MiB and N > 1024 else 1)       # look-ahead over two resident block columns / staged
    assert not np.isnan(got).any() and np.isnan(B.array[:, N:]).all()
    if dist == "int":
        assert np.array_equal(ref, alpha * X0)
        assert np.array_equal(got, alpha * X0), f"{np.count_nonzero(got != alpha * X0)} elements differ"
    else:
        # X op(T) = alpha B  <=>  op(T)^T X^T = alpha B^T: the left-side residual of the oracle on written-out transposes
        res, den = oracle.dtrsm_residual(uplo, 1 - trans, unit, alpha, np.nan_to_num(A.view), np.ascontiguousarray(B0.T), np.ascontiguousarray(got.T))
        assert (res <= oracle.dtrsm_gate(N) * den).all(), float((res / den).max() / oracle.dtrsm_gate(N))
        assert np.abs(got - ref).max() <= FWD_RTOL * np.abs(ref).max()


def test_dtrsm_side_left_is_hclooc_dtrsm_and_errors(H):
    M, N = 300, 200
    A = tri_host(H, M, 82, "uniform")
    B = H.HostMatrix(M, N, N)
    synthgen.fill(B.array, 82, "B", "uniform")
    B0 = B.view.copy()
    H.hclooc_dtrsm(None, 0, 0, 0, M, N, 1.5, A, A.ld, B, B.ld, 1 * MiB)
    one = B.view.copy()
    B.view[...] = B0
    H.hclooc_dtrsm_side(None, H.HCL_SIDE_LEFT, 0, 0, 0, M, N, 1.5, A, A.ld, B, B.ld, 1 * MiB)
    assert np.array_equal(B.view.view(np.uint64), one.view(np.uint64))
    AN = tri_host(H, N, 83, "uniform")
    B.view[...] = B0
    Bnan = B0.copy(); Bnan[3, 4] = np.nan
    B.view[...] = Bnan
    H.hclooc_dtrsm_side(None, 1, 0, 0, 0, M, N, 0.0, None, N, B, B.ld, 1 * MiB)      # alpha == 0: zeros, A not read
    assert np.array_equal(B.view, np.zeros((M, N)))
    B.view[...] = B0
    bad = [((2, 0, 0, 0, M, N, 1.0, AN, N, B, N), -2), ((1, 2, 0, 0, M, N, 1.0, AN, N, B, N), -3), ((1, 0, 2, 0, M, N, 1.0, AN, N, B, N), -4),
           ((1, 0, 0, 2, M, N, 1.0, AN, N, B, N), -5), ((1, 0, 0, 0, -1, N, 1.0, AN, N, B, N), -6), ((1, 0, 0, 0, M, -1, 1.0, AN, N, B, N), -7),
           ((1, 0, 0, 0, M, N, 1.0, None, N, B, N), -9), ((1, 0, 0, 0, M, N, 1.0, AN, N - 1, B, N), -10), ((1, 0, 0, 0, M, N, 1.0, AN, N, None, N), -11),
           ((1, 0, 0, 0, M, N, 1.0, AN, N, B, N - 1), -12), ((0, 2, 0, 0, M, N, 1.0, A, M, B, N), -3), ((0, 0, 0, 0, M, N, 1.0, A, M - 1, B, N), -10)]
    for args, code in bad:
        with pytest.raises(H.HclError) as e:
            H.hclooc_dtrsm_side(None, *args, 1 * MiB)
        assert e.value.status == code, (args[:7], e.value.status)
    assert np.array_equal(B.view, B0)


@pytest.mark.parametrize("uplo,trans", [(0, 1), (1, 0)])
def test_dtrsm_right_large_block_columns_of_4096(H, uplo, trans):
    """6000 columns under 1 GiB: block columns of 4096 (one ragged), the update is an out-of-core DGEMM with C in device memory;
    the whole result against the oracle and the residual gate on samples."""
    M, N, alpha = 3000, 6000, 1.25
    A = tri_host(H, N, 84, "uniform")
    B = H.HostMatrix(M, N, N)
    synthgen.fill(B.array, 84, "B", "uniform")
    A.view[other_triangle(N, uplo)] = np.nan
    B0 = B.view.copy()
    st = H.hclooc_dtrsm_side(None, 1, uplo, trans, 0, M, N, alpha, A, A.ld, B, B.ld, 1024 * MiB)
    got = B.view.copy()
    assert st.plan.nb == 4096 and st.plan.w == 2 and st.plan.workspace_bytes <= 1024 * MiB
    ref = B0.copy()
    oracle.dtrsm_right(uplo, trans, 0, alpha, A.view, ref)
    assert np.abs(got - ref).max() <= FWD_RTOL * np.abs(ref).max()
    rng = np.random.default_rng(3)
    rows = np.unique(np.concatenate([[0, 127, 128, 4095, 4096, N - 1], rng.integers(0, N, 30)]))       # rows of X^T = columns of X
    cols = np.unique(np.concatenate([[0, M - 1], rng.integers(0, M, 30)]))
    res, den = oracle.dtrsm_residual(uplo, 1 - trans, 0, alpha, np.nan_to_num(A.view), np.ascontiguousarray(B0.T), np.ascontiguousarray(got.T), rows, cols)
    assert (res <= oracle.dtrsm_gate(N) * den).all()
