"""GPU parity for the RESIDENT schedule of hclooc_dgemm (resident.cu; DESIGN.md section 7 "Resident schedule"): host matrices that
fit the device budget get device copies, K is streamed in panels (whole-C kernels behind the uploads), then C is finished row block
by row block under its own downloads.  Same bars as the slice pipeline: integer data bit for bit against the oracle, floats within
1e-13 * D elementwise (the order of summation differs from the pipeline's, so the two schedules agree to rounding only).
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


@pytest.fixture()
def forced(monkeypatch):
    monkeypatch.setenv("HCLOOC_RESIDENT", "1")       # the schedule whenever it fits, whatever the cost model says


def host_inputs(H, M, N, K, seed, dist, pads=(0, 0, 0)):
    A, B, C = H.HostMatrix(M, K, K + pads[0]), H.HostMatrix(K, N, N + pads[1]), H.HostMatrix(M, N, N + pads[2])
    for X, name in ((A, "A"), (B, "B"), (C, "C")):
        X.array[...] = np.nan
        synthgen.fill(X.array, seed, name, dist, cols=X.cols)
    return A, B, C


def check(H, st, C, ref, D, exact, M, N):
    got = C.view
    assert np.isnan(C.array[:, N:]).all(), "padding columns of C written"
    if exact:
        assert np.array_equal(got, ref), f"{np.count_nonzero(got != ref)} elements differ"
    else:
        ok, worst = oracle.within_gate(got, ref, D, RTOL)
        assert ok, f"worst |err|/D = {worst:.3e}"


@pytest.mark.parametrize("M,N,K,alpha,beta,dist,pads,budget", [
    (1500, 1100, 2100, 1.0, 0.5, "int", (1, 3, 5), 256 * MiB),         # ragged everywhere, odd N and K, padded leading dimensions
    (1500, 1100, 2100, -2.0, 1.0, "uniform", (0, 0, 0), 256 * MiB),
    (2048, 2048, 4096, 1.5, 0.0, "uniform", (0, 0, 0), 512 * MiB),     # beta == 0: C0 is NaN and never uploaded
    (640, 3000, 1024, 1.0, -1.0, "int", (2, 0, 2), 200 * MiB),         # few rows: 5 row blocks of 128
    (4096, 1024, 1536, 2.0, 2.0, "int", (0, 0, 0), 160 * MiB),         # the staging ring is shorter than the row blocks: slots are reused
])
def test_resident_schedule_matches_oracle(H, forced, M, N, K, alpha, beta, dist, pads, budget):
    A, B, C = host_inputs(H, M, N, K, 61, dist, pads)
    if beta == 0.0:
        C.view[...] = np.nan
    ref = C.view.copy()
    D = oracle.dgemm(alpha, A.view.copy(), B.view.copy(), beta, ref, want_denominator=True)
    st = H.hclooc_dgemm_ex(None, M, N, K, alpha, A, A.ld, B, B.ld, beta, C, C.ld, budget)
    p = st.plan
    assert p.resident >= 2 and p.w == 1 and p.kpanels >= 2 and p.workspace_bytes <= budget
    assert p.n_steps == (p.resident - 1) + p.h
    assert st.bytes_h2d == 8 * (M * K + K * N + (M * N if beta != 0.0 else 0)) and st.bytes_d2h == 8 * M * N
    assert st.n_copies_h2d == 2 * p.kpanels + (p.h if beta != 0.0 else 0) and st.n_copies_d2h == p.h
    check(H, st, C, ref, D, dist == "int", M, N)
    for X in (A, B, C):
        X.free()


def test_resident_schedule_under_the_shaker_and_its_sabotage(H, forced):
    """Random delays in front of every copy and kernel + NaN in every buffer the schedule declares free: the result must not
    change; with the staging ring's waits ignored on both sides (poison mode 2: slots refilled before their tenant was used, blocks
    used before they arrived) the poison must show."""
    M, N, K, alpha, beta = 4096, 1024, 1536, 1.0, 1.0
    A, B, C = host_inputs(H, M, N, K, 62, "int")
    C0 = C.view.copy()
    ref = C0.copy()
    oracle.dgemm(alpha, A.view.copy(), B.view.copy(), beta, ref)
    ctx = H.hclooc_ctx_create(0)
    try:
        for seed in (1, 2, 3):
            H.hclooc_ctx_set_debug(ctx, seed, 1)
            C.view[...] = C0
            st = H.hclooc_dgemm_ex(ctx, M, N, K, alpha, A, A.ld, B, B.ld, beta, C, C.ld, 160 * MiB)
            assert st.plan.resident >= 2 and st.plan.n_sets < st.plan.h
            assert np.array_equal(C.view, ref), f"seed {seed}: {np.count_nonzero(C.view != ref)} elements differ"
        bad = 0
        for seed in (4, 5, 6, 7):
            H.hclooc_ctx_set_debug(ctx, seed, 2)
            C.view[...] = C0
            H.hclooc_dgemm_ex(ctx, M, N, K, alpha, A, A.ld, B, B.ld, beta, C, C.ld, 160 * MiB)
            bad += int(not np.array_equal(C.view, ref))
        assert bad > 0, "the shaker did not notice a schedule whose staging ring ignores its waits"
    finally:
        H.hclooc_ctx_destroy(ctx)
        for X in (A, B, C):
            X.free()


def test_resident_is_chosen_by_the_cost_model_and_can_be_switched_off(H, monkeypatch):
    """Balanced regime (link time ~ flop time): 6144^3 fits 2 GiB and the model prefers the resident schedule; HCLOOC_RESIDENT=0
    gives the slice pipeline on the same call; a traced call records every copy and kernel of the resident schedule."""
    n = 6144
    A, B, C = host_inputs(H, n, n, n, 63, "int")
    C0 = C.view.copy()
    ctx = H.hclooc_ctx_create(0)
    try:
        st = H.hclooc_dgemm_ex(ctx, n, n, n, 1.0, A, n, B, n, 1.0, C, n, 2048 * MiB)
        assert st.plan.resident >= 2, "the cost model no longer picks the resident schedule in the balanced regime"
        got = C.view.copy()
        monkeypatch.setenv("HCLOOC_RESIDENT", "0")
        C.view[...] = C0
        st0 = H.hclooc_dgemm_ex(ctx, n, n, n, 1.0, A, n, B, n, 1.0, C, n, 2048 * MiB)
        assert st0.plan.resident == 0 and st0.plan.h * st0.plan.w > 1
        assert np.array_equal(C.view, got)                                   # integer data: both schedules are exact
        rng = np.random.default_rng(5)
        rows = np.unique(rng.integers(0, n, 24))
        ref = C0[rows].copy()
        oracle.dgemm(1.0, A.view[rows].copy(), B.view.copy(), 1.0, ref)
        assert np.array_equal(got[rows], ref)
        monkeypatch.delenv("HCLOOC_RESIDENT")
        H.hclooc_ctx_set_trace(ctx, 1)
        C.view[...] = C0
        st = H.hclooc_dgemm_ex(ctx, n, n, n, 1.0, A, n, B, n, 1.0, C, n, 2048 * MiB)
        recs = H.hclooc_ctx_get_trace(ctx)
        assert st.plan.resident >= 2 and np.array_equal(C.view, got)
        assert len(recs) == st.n_copies_h2d + st.n_copies_d2h + st.n_kernels
        flops = sum(float(r["flops"]) for r in recs if r["kind"] == 3 and r["flops"] > 4.0 * n * n)     # the GEMM launches (not the axpys)
        assert flops == 2.0 * n ** 3
    finally:
        H.hclooc_ctx_destroy(ctx)
        for X in (A, B, C):
            X.free()
