"""GPU parity for the out-of-core DTRSM (hclooc_dtrsm, side = Left) against the CPU oracle.

Bar (G23): integer data with a +-1 diagonal -> the solution bit for bit; otherwise the elementwise residual bound of
substitution in any summation order, |alpha*B - op(T) X| <= gamma_(M+2) * (|alpha B| + |op(T)||X|) (oracle.dtrsm_gate, evaluated
by the oracle in long double), AND, the operands being well conditioned by construction (synthgen.shape_triangular), agreement
with the oracle's own solution to 1e-12 of the largest entry.
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


def trsm_inputs(H, uplo, unit, M, N, seed, dist, pad=0):
    """A (triangle `uplo` shaped, the other triangle and a unit diagonal NaN), B, and for integers the solution X0 it hides."""
    A = H.HostMatrix(M, M, M + pad); B = H.HostMatrix(M, N, N + pad)
    A.array[...] = np.nan; B.array[...] = np.nan
    synthgen.fill(A.array, seed, "A", dist, cols=M)
    synthgen.shape_triangular(A.view, dist)
    synthgen.fill(B.array, seed, "B", dist, cols=N)
    return A, B


def poison(A, uplo, unit):
    M = A.view.shape[0]
    other = np.triu(np.ones((M, M), bool), 1) if uplo == 0 else np.tril(np.ones((M, M), bool), -1)
    A.view[other] = np.nan
    if unit:
        A.view[np.arange(M), np.arange(M)] = np.nan


def dense_op(Aview, uplo, trans, unit):
    T = np.tril(Aview) if uplo == 0 else np.triu(Aview)
    if unit:
        T = T - np.diag(np.diag(T)) + np.eye(T.shape[0])
    return T.T if trans else T


@pytest.mark.parametrize("uplo", [0, 1])
@pytest.mark.parametrize("trans", [0, 1])
@pytest.mark.parametrize("unit", [0, 1])
@pytest.mark.parametrize("M,N,alpha,dist,pad,budget", [
    (300, 200, 1.0, "uniform", 3, 1 * MiB),        # NB = 256: two block rows, ragged second, 128-row inner blocks
    (1000, 517, 2.0, "int", 0, 2 * MiB),           # NB = 256..384: several block rows, ragged chunk, exact
    (129, 64, -0.5, "uniform", 1, 64 * MiB),       # one block row: no out-of-core update, alpha applied in the diagonal phase
    (77, 1, 1.0, "int", 0, 512 * 1024),            # a single right-hand side
    (1500, 333, 1.5, "uniform", 2, 3 * MiB),
    (500, 130, 1.0, "int", 1, 192 * 1024),         # NB = 96: six block rows of less than one 128-row inner block, tiny DGEMM budgets
])
def test_dtrsm_matches_oracle(H, uplo, trans, unit, M, N, alpha, dist, pad, budget):
    A, B = trsm_inputs(H, uplo, unit, M, N, 91, dist, pad)
    if dist == "int":
        # B := op(T) X0 in int64, so that the exact solution is the integer matrix X0 / alpha-scaled copies of it
        X0 = B.view.copy().astype(np.int64)
        T = dense_op(np.nan_to_num(A.view), uplo, trans, unit).astype(np.int64)
        B.view[...] = (T @ X0).astype(np.float64)
    poison(A, uplo, unit)
    B0 = B.view.copy()
    ref = B0.copy()
    oracle.dtrsm(uplo, trans, unit, alpha, A.view, ref)
    st = H.hclooc_dtrsm(None, uplo, trans, unit, M, N, alpha, A, A.ld, B, B.ld, budget)
    got = B.view.copy()
    assert st.plan.workspace_bytes <= budget and st.n_kernels >= 1
    assert (st.plan.mb, st.plan.n_sets) == H.hclooc_dtrsm_plan(M, N, budget)[::2]
    assert st.plan.n_sets == (1 if (M, budget) in ((129, 64 * MiB), (77, 512 * 1024), (1500, 3 * MiB)) else 0)   # resident block row?
    assert not np.isnan(got).any()
    assert np.isnan(B.array[:, N:]).all()                              # padding untouched
    if dist == "int":
        assert np.array_equal(ref, alpha * X0)                         # the oracle, against the hidden solution
        assert np.array_equal(got, alpha * X0), f"{np.count_nonzero(got != alpha * X0)} elements differ"
    else:
        Aclean = np.nan_to_num(A.view)
        res, den = oracle.dtrsm_residual(uplo, trans, unit, alpha, Aclean, B0, got)
        assert (res <= oracle.dtrsm_gate(M) * den).all(), float((res / den).max())
        assert np.abs(got - ref).max() <= FWD_RTOL * np.abs(ref).max()


def test_dtrsm_alpha_zero_degenerate_and_errors(H):
    M, N = 200, 100
    A, B = trsm_inputs(H, 0, 0, M, N, 92, "uniform")
    B.view[5, 7] = np.nan
    Anan = H.HostMatrix(M, M, M); Anan.array[...] = np.nan
    H.hclooc_dtrsm(None, 0, 0, 0, M, N, 0.0, Anan, M, B, B.ld, 1 * MiB)      # alpha == 0: zeros, A not read, NaN not carried
    assert np.array_equal(B.view, np.zeros((M, N)))
    synthgen.fill(B.array, 93, "B", "uniform", cols=N)
    keep = B.view.copy()
    H.hclooc_dtrsm(None, 0, 0, 0, 0, N, 1.0, A, M, B, B.ld, 1 * MiB)         # M == 0 / N == 0: nothing
    H.hclooc_dtrsm(None, 0, 0, 0, M, 0, 1.0, A, M, B, B.ld, 1 * MiB)
    assert np.array_equal(B.view, keep)
    bad = [((2, 0, 0, M, N, 1.0, A, M, B, N), -2), ((0, 2, 0, M, N, 1.0, A, M, B, N), -3), ((0, 0, 2, M, N, 1.0, A, M, B, N), -4),
           ((0, 0, 0, -1, N, 1.0, A, M, B, N), -5), ((0, 0, 0, M, -1, 1.0, A, M, B, N), -6), ((0, 0, 0, M, N, 1.0, None, M, B, N), -8),
           ((0, 0, 0, M, N, 1.0, A, M - 1, B, N), -9), ((0, 0, 0, M, N, 1.0, A, M, None, N), -10), ((0, 0, 0, M, N, 1.0, A, M, B, N - 1), -11)]
    for args, code in bad:
        with pytest.raises(H.HclError) as ei:
            H.hclooc_dtrsm(None, *args, 1 * MiB)
        assert ei.value.status == code, (args[:6], ei.value.status)
    with pytest.raises(H.HclError) as ei:                                      # not even a 32-row block fits
        H.hclooc_dtrsm(None, 0, 0, 0, M, N, 1.0, A, M, B, N, 16 * 1024)
    assert ei.value.status == 1
    pageable = np.zeros((M, N))
    with pytest.raises(H.HclError) as ei:
        H.hclooc_dtrsm(None, 0, 0, 0, M, N, 1.0, A, M, pageable, N, 1 * MiB)
    assert ei.value.status == 2
    assert np.array_equal(B.view, keep)                                        # validation errors leave B untouched


@pytest.mark.parametrize("budget,resident", [(256 * MiB, 0), (1024 * MiB, 1)])
@pytest.mark.parametrize("uplo,trans,unit", [(0, 0, 0), (1, 0, 1), (0, 1, 0), (1, 1, 0)])
def test_dtrsm_large_block_rows_of_4096(H, uplo, trans, unit, budget, resident):
    """Under 256 MiB: NB = 4096, two block rows (one ragged), staged through two column chunks on two streams, 32 inner blocks
    per chunk.  Under 1 GiB the whole problem is one resident block row of 6000 rows (no out-of-core update; the recursion of the
    diagonal phase is 6 levels deep).  The whole result against the oracle, the residual gate on sampled rows and columns."""
    M, N, alpha = 6000, 4500, 1.25
    A, B = trsm_inputs(H, uplo, unit, M, N, 94, "uniform")
    poison(A, uplo, unit)
    B0 = B.view.copy()
    st = H.hclooc_dtrsm(None, uplo, trans, unit, M, N, alpha, A, A.ld, B, B.ld, budget)
    got = B.view.copy()
    assert (st.plan.mb, st.plan.h) == ((4096, 2) if resident == 0 else (6000, 1))
    assert st.plan.workspace_bytes <= budget and st.plan.n_sets == resident
    ref = B0.copy()
    if trans:   # the oracle walks a transposed triangle column-wise (slow); (uplo, T) on A is (other uplo, N) on the written-out transpose, bit for bit (pinned)
        oracle.dtrsm(1 - uplo, 0, unit, alpha, np.ascontiguousarray(np.nan_to_num(A.view).T), ref)
    else:
        oracle.dtrsm(uplo, trans, unit, alpha, A.view, ref)
    assert np.abs(got - ref).max() <= FWD_RTOL * np.abs(ref).max()
    rng = np.random.default_rng(0)
    rows = np.unique(np.concatenate([[0, 127, 128, 4095, 4096, M - 1], rng.integers(0, M, 40)]))
    cols = np.unique(np.concatenate([[0, 63, 64, N - 1], rng.integers(0, N, 40)]))
    res, den = oracle.dtrsm_residual(uplo, trans, unit, alpha, np.nan_to_num(A.view), B0, got, rows, cols)
    assert (res <= oracle.dtrsm_gate(M) * den).all()


@pytest.mark.parametrize("dist", ["int", "uniform"])
def test_dtrsm_resident_lookahead_and_staged_modes_agree(H, dist):
    """The same solve with two block rows resident in device memory (the look-ahead form: the next block row's update is split
    into the part streamed from the host and the freshest block row's part taken from device memory) and staged through column
    chunks in a caller-owned workspace too small for resident rows.  Same blocked substitution, but the sums over k are cut
    differently, so: bit for bit on integer data, the backward gate and 1e-12 agreement on float data."""
    import torch
    M, N = 3000, 300
    A, B = trsm_inputs(H, 1, 0, M, N, 95, dist, pad=1)
    if dist == "int":
        X0 = B.view.copy().astype(np.int64)
        B.view[...] = (dense_op(np.nan_to_num(A.view), 1, 0, 0).astype(np.int64) @ X0).astype(np.float64)
    poison(A, 1, 0)
    B0 = B.view.copy()
    st = H.hclooc_dtrsm(None, 1, 0, 0, M, N, 1.0, A, A.ld, B, B.ld, 48 * MiB)
    assert st.plan.n_sets == 2 and st.plan.h == 2 and st.plan.workspace_bytes <= 48 * MiB
    res = B.view.copy()
    ws = torch.empty(6 * MiB, dtype=torch.uint8, device="cuda")
    torch.cuda.synchronize()
    ctx = H.hclooc_ctx_create(0, ws.data_ptr(), ws.numel())
    try:
        B.view[...] = B0
        st = H.hclooc_dtrsm(ctx, 1, 0, 0, M, N, 1.0, A, A.ld, B, B.ld, 0)
        assert st.plan.n_sets == 0 and st.plan.workspace_bytes <= 6 * MiB and st.plan.h >= 2
    finally:
        H.hclooc_ctx_destroy(ctx)
    if dist == "int":
        assert np.array_equal(res, X0) and np.array_equal(B.view, res)
    else:
        for got in (res, B.view):
            r, d = oracle.dtrsm_residual(1, 0, 0, 1.0, np.nan_to_num(A.view), B0, np.ascontiguousarray(got))
            assert (r <= oracle.dtrsm_gate(M) * d).all()
        assert np.abs(B.view - res).max() <= FWD_RTOL * np.abs(res).max()


@pytest.mark.parametrize("uplo,trans", [(0, 0), (1, 0)])
def test_dtrsm_two_resident_block_rows_of_8192(H, uplo, trans):
    """Block rows of 8192 rows, both resident under 2 GiB: the second one is uploaded during the first one's diagonal phase and
    updated by the out-of-core DGEMM in device memory.  Forward agreement with the oracle and the residual gate on samples."""
    M, N, alpha = 10000, 2000, 0.75
    A, B = trsm_inputs(H, uplo, 0, M, N, 96, "uniform")
    poison(A, uplo, 0)
    B0 = B.view.copy()
    st = H.hclooc_dtrsm(None, uplo, trans, 0, M, N, alpha, A, A.ld, B, B.ld, 2048 * MiB)
    got = B.view.copy()
    assert (st.plan.mb, st.plan.h, st.plan.n_sets) == (8192, 2, 2) and st.plan.workspace_bytes <= 2048 * MiB
    ref = B0.copy()
    oracle.dtrsm(uplo, trans, 0, alpha, A.view, ref)
    assert np.abs(got - ref).max() <= FWD_RTOL * np.abs(ref).max()
    rng = np.random.default_rng(1)
    rows = np.unique(np.concatenate([[0, 8191, 8192, M - 1], rng.integers(0, M, 40)]))
    cols = np.unique(np.concatenate([[0, N - 1], rng.integers(0, N, 40)]))
    res, den = oracle.dtrsm_residual(uplo, trans, 0, alpha, np.nan_to_num(A.view), B0, got, rows, cols)
    assert (res <= oracle.dtrsm_gate(M) * den).all()


@pytest.mark.parametrize("uplo,trans,budget", [(0, 0, 1 * MiB), (1, 1, 1 * MiB), (1, 0, 64 * MiB)])
def test_dtrsm_ill_conditioned_only_the_backward_gate_holds(H, uplo, trans, budget):
    """A triangle whose off-diagonal entries are as large as its diagonal (uniform[-0.8, 0.8) against |t_ii| in [1, 2)): the
    solution grows by twelve orders of magnitude down the substitution, so agreement with another summation order's solution is
    not a property of the method -- the elementwise backward bound gamma_(M+2) (G23, Higham thm 8.5) is, and it is the
    only thing asserted here (the oracle's own solution satisfies it too: tests/test_oracle_pins.py)."""
    M, N = 600, 40
    rng = np.random.default_rng(3)
    T = np.diag(rng.uniform(1, 2, M) * rng.choice([-1, 1], M)) + 0.8 * np.tril(rng.uniform(-1, 1, (M, M)), -1)
    A = H.HostMatrix(M, M, M); B = H.HostMatrix(M, N, N)
    stored = T if uplo == 0 else np.ascontiguousarray(T.T)        # the triangle `uplo` names; `trans` then picks op(T)
    A.view[...] = stored
    poison(A, uplo, 0)
    B.view[...] = rng.uniform(-1, 1, (M, N))
    B0 = B.view.copy()
    st = H.hclooc_dtrsm(None, uplo, trans, 0, M, N, 1.0, A, A.ld, B, B.ld, budget)
    got = B.view.copy()
    assert np.isfinite(got).all() and np.abs(got).max() > 1e9, "the case is meant to be ill conditioned"
    assert st.plan.h == (1 if budget > 8 * MiB else st.plan.h) and (budget > 8 * MiB or st.plan.h > 1)
    res, den = oracle.dtrsm_residual(uplo, trans, 0, 1.0, np.nan_to_num(A.view), B0, got)
    assert (res <= oracle.dtrsm_gate(M) * den).all(), float((res / den).max() / oracle.dtrsm_gate(M))
