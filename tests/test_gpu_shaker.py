"""The debug shaker (hclooc_ctx_set_debug): random spin kernels in front of every copy and kernel
and NaN in every device buffer the moment the schedule frees it.  The parity cases whose stream choreography lives OUTSIDE the
schedule simulator of tests/test_planner_schedule.py -- the look-ahead forms of hclooc_dtrsm and hclooc_dpotrf, hclooc_dtrsm_side,
the nsteps mode -- and the pipeline's own corner cases (two B buffers, K panels, the triangle mask, transposed operands) must give
the same exact results under several seeds; and the shaker is shown not to be vacuous: with the upload stream's waits removed
(poison = 2) the very same call goes wrong."""
import numpy as np
import pytest

import oracle
import synthgen

pytestmark = pytest.mark.gpu
MiB = 1 << 20
SEEDS = (1, 20261105, 987654321)


@pytest.fixture(scope="module")
def H():
    import paper_1808_05056_b200 as H
    import torch
    assert torch.cuda.is_available()
    torch.cuda.init()
    yield H
    H.hclooc_ctx_set_debug(None, 0, 0)


def ints(H, rows, cols, seed, name, pad=0):
    X = H.HostMatrix(rows, cols, cols + pad)
    X.array[...] = np.nan
    synthgen.fill(X.array, seed, name, "int", cols=cols)
    return X


@pytest.mark.parametrize("M,N,K,budget,bbuf", [(512, 512, 512, 1 * MiB, 0), (700, 900, 300, 3 * MiB, 2), (256, 16, 200000, 1 * MiB, 0), (96, 112, 20000, 600 * 1024, 0)])
def test_pipeline_is_exact_under_the_shaker_and_wrong_without_its_waits(H, monkeypatch, M, N, K, budget, bbuf):
    if bbuf:
        monkeypatch.setenv("HCLOOC_FORCE_BBUF", str(bbuf))
    A, B, C = ints(H, M, K, 61, "A"), ints(H, K, N, 61, "B"), ints(H, M, N, 61, "C", pad=2)
    C0 = C.view.copy()
    ref = C0.copy()
    oracle.dgemm(1.0, A.view, B.view, -2.0, ref)
    try:
        for seed in SEEDS[:2]:
            C.view[...] = C0
            H.hclooc_ctx_set_debug(None, seed, 1)
            st = H.hclooc_dgemm_ex(None, M, N, K, 1.0, A, A.ld, B, B.ld, -2.0, C, C.ld, budget)
            assert np.array_equal(C.view, ref), f"seed {seed}: {np.count_nonzero(C.view != ref)} elements differ"
            assert np.isnan(C.array[:, N:]).all()
        if bbuf:
            assert st.plan.n_bbuf == 2
        # not vacuous: the same call with the upload stream's waits removed
        wrong = 0
        for seed in SEEDS[:2]:
            C.view[...] = C0
            H.hclooc_ctx_set_debug(None, seed, 2)
            H.hclooc_dgemm_ex(None, M, N, K, 1.0, A, A.ld, B, B.ld, -2.0, C, C.ld, budget)
            wrong += int(not np.array_equal(C.view, ref))
        assert wrong > 0, "removing every wait of the upload stream went unnoticed"
    finally:
        H.hclooc_ctx_set_debug(None, 0, 0)


@pytest.mark.parametrize("uplo,trans", [(0, 0), (1, 1)])
def test_dsyrk_and_transposed_dgemm_under_the_shaker(H, uplo, trans):
    N, K = 900, 500
    A = ints(H, K if trans else N, N if trans else K, 62, "A")
    C = ints(H, N, N, 62, "C")
    other = np.triu(np.ones((N, N), bool), 1) if uplo == 0 else np.tril(np.ones((N, N), bool), -1)
    C.view[other] = np.nan
    C0 = C.view.copy()
    ref = C0.copy()
    oracle.dsyrk(uplo, trans, 1.0, A.view, 3.0, ref)
    try:
        for seed in SEEDS[:2]:
            C.view[...] = C0
            H.hclooc_ctx_set_debug(None, seed, 1)
            H.hclooc_dsyrk(None, uplo, trans, N, K, 1.0, A, A.ld, 3.0, C, C.ld, 2 * MiB)
            assert np.array_equal(C.view[~other], ref[~other]) and np.isnan(C.view[other]).all()
    finally:
        H.hclooc_ctx_set_debug(None, 0, 0)


@pytest.mark.parametrize("uplo,trans", [(0, 0), (1, 0), (0, 1)])
def test_dtrsm_lookahead_staged_and_right_side_under_the_shaker(H, uplo, trans):
    from test_gpu_factor import tri_host, dense_op
    M, N = 3000, 300
    try:
        for budget in (48 * MiB, 1 * MiB):                      # two resident block rows with the look-ahead / staged column chunks
            T = tri_host(H, M, 63, "int")
            X0 = synthgen.fill_numpy(M, N, 63, "B", "int").astype(np.int64)
            B = H.HostMatrix(M, N)
            rhs = (dense_op(T.view, uplo, trans, 0).astype(np.int64) @ X0).astype(np.float64)
            for seed in SEEDS[:2]:
                B.view[...] = rhs
                H.hclooc_ctx_set_debug(None, seed, 1)
                st = H.hclooc_dtrsm(None, uplo, trans, 0, M, N, 1.0, T, T.ld, B, B.ld, budget)
                assert np.array_equal(B.view, X0.astype(np.float64)), (budget, seed)
            assert st.plan.n_sets == (2 if budget > 8 * MiB else 0)
        # side = Right: row bands x block columns (staged, 2 MiB), and two resident block columns of 1024 with the look-ahead (48 MiB)
        for Mr, Nr, budget in ((517, 1000, 2 * MiB), (600, 2600, 48 * MiB)):
            T = tri_host(H, Nr, 64, "int")
            X0 = synthgen.fill_numpy(Mr, Nr, 64, "B", "int").astype(np.int64)
            B = H.HostMatrix(Mr, Nr)
            rhs = (X0 @ dense_op(T.view, uplo, trans, 0).astype(np.int64)).astype(np.float64)
            for seed in SEEDS[:2]:
                B.view[...] = rhs
                H.hclooc_ctx_set_debug(None, seed, 1)
                st = H.hclooc_dtrsm_side(None, 1, uplo, trans, 0, Mr, Nr, 1.0, T, T.ld, B, B.ld, budget)
                assert np.array_equal(B.view, X0.astype(np.float64)), (budget, seed)
            assert st.plan.n_sets == (2 if budget > 8 * MiB else 1) and st.plan.workspace_bytes <= budget
    finally:
        H.hclooc_ctx_set_debug(None, 0, 0)


@pytest.mark.parametrize("uplo", [0, 1])
def test_dpotrf_lookahead_under_the_shaker(H, uplo):
    from test_gpu_factor import spd_host, other_triangle
    N = 1500
    A, L0 = spd_host(H, N, 65, "int")
    other = other_triangle(N, uplo)
    A.view[other] = np.nan
    A0 = A.view.copy()
    want = L0 if uplo == 0 else L0.T
    try:
        for seed in SEEDS:
            A.view[...] = A0
            H.hclooc_ctx_set_debug(None, seed, 1)
            info, st = H.hclooc_dpotrf(None, uplo, N, A, A.ld, 8 * MiB)
            assert info == 0 and st.plan.n_steps > 4
            assert np.array_equal(A.view[~other], want[~other]) and np.isnan(A.view[other]).all(), seed
    finally:
        H.hclooc_ctx_set_debug(None, 0, 0)


def test_nsteps_mode_under_the_shaker(H):
    M, N, K, nsteps = 600, 500, 256, 3
    A, B, C = ints(H, M, nsteps * K, 66, "A"), ints(H, nsteps * K, N, 66, "B"), ints(H, M, N, 66, "C")
    ref = C.view.copy()
    oracle.dgemm(1.0, A.view, B.view, 0.5, ref)
    try:
        H.hclooc_ctx_set_debug(None, SEEDS[0], 1)
        step = 0
        for p in range(nsteps):
            step, _ = H.hclooc_dgemm_nsteps(None, M, N, K, 1.0, A.ptr + 8 * p * K, A.ld, B.ptr + 8 * p * K * B.ld, B.ld, 0.5 if p == 0 else 1.0,
                                            C, C.ld, 8 * MiB, nsteps, step)
        assert np.array_equal(C.view, ref)
    finally:
        H.hclooc_ctx_set_debug(None, 0, 0)
