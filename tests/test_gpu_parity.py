"""GPU parity: the CUDA path (through the C ABI binding) against the CPU oracle, element by element.

Bar (BASELINE.json north_star, G14): bit-exact (by value) on small-integer inputs whose
products and sums are exact in FP64; |C_gpu - C_ref| <= 1e-13 * D elsewhere, with
D = |alpha| * sum_k |A_ik||B_kj| + |beta||C0_ij| computed by the oracle.
"""
import numpy as np
import pytest

import oracle
import synthgen

pytestmark = pytest.mark.gpu

RTOL = 1e-13          # the gate, written out as the task requires
MiB = 1 << 20


@pytest.fixture(scope="module")
def H():
    import paper_1808_05056_b200 as H
    import torch
    assert torch.cuda.is_available()
    torch.cuda.init()
    return H


def host_inputs(H, M, N, K, seed, dist, pads=(0, 0, 0), poison_c=False):
    A = H.HostMatrix(M, K, K + pads[0])
    B = H.HostMatrix(K, N, N + pads[1])
    C = H.HostMatrix(M, N, N + pads[2])
    for X in (A, B, C):
        X.array[...] = np.nan                        # padding is NaN: reading it would show
    synthgen.fill(A.array, seed, "A", dist, cols=K)
    synthgen.fill(B.array, seed, "B", dist, cols=N)
    if poison_c:
        C.view[...] = np.nan
    else:
        synthgen.fill(C.array, seed, "C", dist, cols=N)
    return A, B, C


def to_dev(x):
    """numpy -> device tensor, COMPLETE on return: the library launches on its own (non-blocking) streams, which do not wait
    for PyTorch's stream, so a device operand must be ready before it is handed over (include/hclooc.h, hclooc_dgemm)."""
    import torch
    t = torch.from_numpy(x).cuda()
    torch.cuda.synchronize()
    return t


def check(C_gpu, C_ref, D, exact):
    assert not np.isnan(C_gpu).any()
    if exact:
        assert np.array_equal(C_gpu, C_ref), f"{np.count_nonzero(C_gpu != C_ref)} elements differ"
        assert not (np.signbit(C_gpu) != np.signbit(C_ref)).any()       # sign of zero too (G15)
    else:
        ok, worst = oracle.within_gate(C_gpu, C_ref, D, RTOL)
        assert ok, f"worst |err|/D = {worst:.3e} > {RTOL}"


# ------------------------------------------------------------------ S5: the tile kernel on device pointers
@pytest.mark.parametrize("M,N,K,alpha,beta,dist", [
    (128, 128, 16, 1.0, 0.0, "uniform"),          # exactly one tile, one k step
    (1, 1, 1, 2.0, 0.5, "uniform"),
    (300, 260, 200, 1.0, 0.5, "uniform"),         # several tiles, ragged in m, n and k
    (129, 257, 33, -1.5, 1.0, "normal"),
    (517, 389, 1000, 2.0, -1.0, "uniform"),
    (256, 384, 512, 1.0, 0.5, "int"),
    (131, 77, 97, 3.0, 2.0, "int"),               # primes
    (64, 1024, 8, 1.0, 0.0, "int"),
    (128, 256, 4096, 1.0, 0.5, "uniform"),        # 2 tiles, deep K: 4-CTA cluster split-K (DSMEM reduction)
    (200, 300, 2061, -1.0, 2.0, "int"),           # 6 tiles, ragged K not a multiple of the split
    (640, 1024, 1040, 1.0, 0.0, "uniform"),       # 40 tiles: 2-CTA cluster split-K
    (640, 1024, 1040, 2.0, 1.0, "int"),
])
def test_tile_kernel_matches_oracle(H, M, N, K, alpha, beta, dist):
    import torch
    lda, ldb, ldc = K + (K % 2) + 4, N + (N % 2) + 2, N + (N % 2) + 6      # even, padded
    A = np.full((M, lda), np.nan); B = np.full((K, ldb), np.nan); C0 = np.full((M, ldc), np.nan)
    synthgen.fill(A, 21, "A", dist, cols=K); synthgen.fill(B, 21, "B", dist, cols=N); synthgen.fill(C0, 21, "C", dist, cols=N)
    if beta == 0.0:
        C0[:, :N] = np.nan                                                       # must not be read
    dA, dB, dC = (to_dev(x) for x in (A, B, C0))
    H.hclDgemmAsync(M, N, K, alpha, dA, lda, dB, ldb, beta, dC, ldc, torch.cuda.current_stream())
    torch.cuda.synchronize()
    got = dC.cpu().numpy()
    ref = C0[:, :N].copy()
    D = oracle.dgemm(alpha, A[:, :K], B[:, :N], beta, ref, want_denominator=True)
    check(got[:, :N], ref, D, exact=(dist == "int"))
    assert np.isnan(got[:, N:]).all()                                            # padding of C untouched


def test_tile_kernel_alpha_zero_and_k_zero(H):
    import torch
    M, N = 200, 136
    C0 = synthgen.fill(np.empty((M, N)), 22, "C", "uniform")
    nan = torch.full((M, 64), float("nan"), dtype=torch.float64, device="cuda")
    nanb = torch.full((64, N), float("nan"), dtype=torch.float64, device="cuda")
    dC = to_dev(C0)
    H.hclDgemmAsync(M, N, 64, 0.0, nan, 64, nanb, N, -2.0, dC, N, torch.cuda.current_stream())    # alpha == 0: A, B not read
    torch.cuda.synchronize()
    assert np.array_equal(dC.cpu().numpy(), -2.0 * C0)
    dC = to_dev(C0)
    H.hclDgemmAsync(M, N, 0, 1.0, None, 2, None, N, 0.5, dC, N, torch.cuda.current_stream())      # K == 0
    torch.cuda.synchronize()
    assert np.array_equal(dC.cpu().numpy(), 0.5 * C0)
    with pytest.raises(H.HclError) as e:
        H.hclDgemmAsync(M, N, 64, 1.0, nan, 63, nanb, N, 0.0, dC, N, torch.cuda.current_stream())
    assert e.value.status == -6
    with pytest.raises(H.HclError) as e:
        H.hclDgemmAsync(M, N, 63, 1.0, nan, 65, nanb, N, 0.0, dC, N, torch.cuda.current_stream())
    assert e.value.status == 5                                                                     # odd ld: HCLOOC_ERR_ALIGN


# ------------------------------------------------------------------ the whole path: configs[0]
@pytest.mark.parametrize("dist,exact", [("uniform", False), ("int", True)])
def test_config1_every_tile_streams(H, dist, exact):
    """BASELINE.json configs[0]: 512^3, alpha 1, beta 0.5, budget 1 MiB; float and {-4..4} variants."""
    M = N = K = 512
    A, B, C = host_inputs(H, M, N, K, synthgen.BASE_SEED + 1, dist)
    ref = C.view.copy()
    D = oracle.dgemm(1.0, A.view, B.view, 0.5, ref, want_denominator=True)
    st = H.hclooc_dgemm_ex(None, M, N, K, 1.0, A, A.ld, B, B.ld, 0.5, C, C.ld, 1 * MiB)
    assert st.plan.workspace_bytes <= 1 * MiB and st.plan.n_steps > 4
    assert st.bytes_h2d == st.plan.bytes_h2d and st.bytes_d2h == st.plan.bytes_d2h == M * N * 8
    check(C.view, ref, D, exact)


def test_budget_invariance_bitwise(H):
    """K is never split here, so every budget must give the same bits (SURVEY 8(c) invariant (i))."""
    M, N, K = 515, 389, 301
    outs = []
    for budget in (1 * MiB, 4 * MiB, 64 * MiB, 0):
        A, B, C = host_inputs(H, M, N, K, 33, "uniform", pads=(3, 5, 7))
        st = H.hclooc_dgemm_ex(None, M, N, K, -0.75, A, A.ld, B, B.ld, 1.25, C, C.ld, budget)
        assert st.plan.kpanels == 1
        assert np.isnan(C.array[:, N:]).all()                  # host padding of C untouched
        outs.append(C.view.copy())
    for o in outs[1:]:
        assert np.array_equal(o.view(np.uint64), outs[0].view(np.uint64))
    A, B, C = host_inputs(H, M, N, K, 33, "uniform", pads=(3, 5, 7))
    ref = C.view.copy()
    D = oracle.dgemm(-0.75, A.view, B.view, 1.25, ref, want_denominator=True)
    check(outs[0], ref, D, exact=False)


def test_k_split_when_budget_is_tiny(H):
    """A budget too small for one K-deep B slice forces K panels; integers stay exact."""
    M, N, K = 96, 112, 20000
    A, B, C = host_inputs(H, M, N, K, 34, "int")
    ref = C.view.copy()
    D = oracle.dgemm(2.0, A.view, B.view, -1.0, ref, want_denominator=True)
    st = H.hclooc_dgemm_ex(None, M, N, K, 2.0, A, A.ld, B, B.ld, -1.0, C, C.ld, 600 * 1024)
    assert st.plan.kpanels > 1
    check(C.view, ref, D, exact=True)
    A, B, C = host_inputs(H, M, N, K, 34, "uniform")
    ref = C.view.copy()
    D = oracle.dgemm(2.0, A.view, B.view, -1.0, ref, want_denominator=True)
    H.hclooc_dgemm(M, N, K, 2.0, A, A.ld, B, B.ld, -1.0, C, C.ld, 600 * 1024)
    check(C.view, ref, D, exact=False)


@pytest.mark.parametrize("M,N,K", [(1, 1, 1), (7, 1000, 3), (1000, 7, 3), (257, 131, 1031), (640, 640, 64)])
def test_ragged_and_degenerate_shapes(H, M, N, K):
    A, B, C = host_inputs(H, M, N, K, 35, "int", pads=(1, 2, 3))
    ref = C.view.copy()
    D = oracle.dgemm(1.0, A.view, B.view, 0.5, ref, want_denominator=True)
    H.hclooc_dgemm(M, N, K, 1.0, A, A.ld, B, B.ld, 0.5, C, C.ld, 2 * MiB)
    check(C.view, ref, D, exact=True)
    assert np.isnan(C.array[:, N:]).all()


def test_beta_zero_overwrites_nan_and_alpha_zero_skips_a_b(H):
    M, N, K = 300, 200, 150
    A, B, C = host_inputs(H, M, N, K, 36, "uniform", poison_c=True)
    ref = np.zeros((M, N))
    D = oracle.dgemm(1.0, A.view, B.view, 0.0, ref, want_denominator=True)
    st = H.hclooc_dgemm_ex(None, M, N, K, 1.0, A, A.ld, B, B.ld, 0.0, C, C.ld, 1 * MiB)
    assert st.bytes_h2d == st.plan.bytes_h2d and st.plan.beta_nonzero == 0           # no C upload
    check(C.view, ref, D, exact=False)
    # alpha == 0: C = beta*C streamed through the device; A and B are NaN and must not matter
    A.array[...] = np.nan; B.array[...] = np.nan
    C0 = synthgen.fill(np.empty((M, N)), 36, "C", "uniform")
    C.view[...] = C0
    st = H.hclooc_dgemm_ex(None, M, N, K, 0.0, A, A.ld, B, B.ld, -2.0, C, C.ld, 1 * MiB)
    assert st.plan.scale_only == 1 and st.bytes_h2d == M * N * 8
    assert np.array_equal(C.view, -2.0 * C0)
    # alpha == beta == 0: +0 everywhere
    C.view[...] = np.nan
    H.hclooc_dgemm(M, N, K, 0.0, A, A.ld, B, B.ld, 0.0, C, C.ld, 1 * MiB)
    assert np.array_equal(C.view, np.zeros((M, N))) and not np.signbit(C.view).any()
    # K == 0 and beta == 1: nothing to do
    C.view[...] = C0
    H.hclooc_dgemm(M, N, 0, 1.0, None, 1, None, N, 1.0, C, C.ld, 1 * MiB)
    assert np.array_equal(C.view, C0)
    # M == 0: touches nothing, pointers may be NULL
    H.hclooc_dgemm(0, N, K, 1.0, None, K, None, N, 1.0, None, N, 1 * MiB)


def test_k_split_identity_and_linearity_on_integers(H):
    """Two calls on K halves (beta = 1 on the second) == one call; alpha scales linearly (exact on integers)."""
    M, N, K = 200, 168, 256
    A, B, C = host_inputs(H, M, N, K, 37, "int")
    H.hclooc_dgemm(M, N, K, 1.0, A, A.ld, B, B.ld, 0.5, C, C.ld, 1 * MiB)
    one = C.view.copy()
    synthgen.fill(C.array, 37, "C", "int", cols=N)
    H.hclooc_dgemm(M, N, K // 2, 1.0, A, A.ld, B, B.ld, 0.5, C, C.ld, 1 * MiB)
    H.hclooc_dgemm(M, N, K - K // 2, 1.0, A.ptr + 8 * (K // 2), A.ld, B.ptr + 8 * (K // 2) * B.ld, B.ld, 1.0, C, C.ld, 1 * MiB)
    assert np.array_equal(C.view, one)
    C.view[...] = 0.0
    H.hclooc_dgemm(M, N, K, 3.0, A, A.ld, B, B.ld, 0.0, C, C.ld, 1 * MiB)
    three = C.view.copy()
    H.hclooc_dgemm(M, N, K, 1.0, A, A.ld, B, B.ld, 0.0, C, C.ld, 1 * MiB)
    assert np.array_equal(three, 3.0 * C.view)


def test_argument_errors_leave_c_untouched(H):
    M, N, K = 64, 64, 64
    A, B, C = host_inputs(H, M, N, K, 38, "uniform")
    before = C.view.copy()
    cases = [((-1, N, K, 1.0, A, K, B, N, 1.0, C, N), -1), ((M, N, K, 1.0, None, K, B, N, 1.0, C, N), -5),
             ((M, N, K, 1.0, A, K - 1, B, N, 1.0, C, N), -6), ((M, N, K, 1.0, A, K, None, N, 1.0, C, N), -7),
             ((M, N, K, 1.0, A, K, B, N - 1, 1.0, C, N), -8), ((M, N, K, 1.0, A, K, B, N, 1.0, None, N), -10),
             ((M, N, K, 1.0, A, K, B, N, 1.0, C, N - 1), -11), ((M, N, K, 1.0, C, K, B, N, 1.0, C, N), -10)]
    for args, want in cases:
        with pytest.raises(H.HclError) as e:
            H.hclooc_dgemm(*args, 1 * MiB)
        assert e.value.status == want, (args, e.value.status)
    with pytest.raises(H.HclError) as e:
        H.hclooc_dgemm(M, N, K, 1.0, A, K, B, N, 1.0, C, N, 4096)               # budget below the minimum working set
    assert e.value.status == 1
    pageable = np.ones((M, K))
    with pytest.raises(H.HclError) as e:
        H.hclooc_dgemm(M, N, K, 1.0, pageable, K, B, N, 1.0, C, N, 1 * MiB)      # no pageable fallback
    assert e.value.status == 2
    assert np.array_equal(C.view, before)
    H.hclooc_host_register(pageable, pageable.nbytes)                             # pinned in place: now accepted
    try:
        H.hclooc_dgemm(M, N, K, 1.0, pageable, K, B, N, 0.0, C, N, 1 * MiB)
    finally:
        H.hclooc_host_unregister(pageable)
    assert np.allclose(C.view, pageable @ B.view)


def test_caller_owned_workspace_and_streams_from_torch(H):
    """PyTorch supplies device memory and streams (north_star); the library carves its buffers from it."""
    import torch
    ws = torch.empty(8 * MiB, dtype=torch.uint8, device="cuda")
    streams = [torch.cuda.Stream() for _ in range(5)]
    ctx = H.hclooc_ctx_create(0, ws, ws.numel(), streams[0], streams[1], streams[2:])
    try:
        M, N, K = 700, 520, 384
        A, B, C = host_inputs(H, M, N, K, 39, "int")
        ref = C.view.copy()
        oracle.dgemm(1.0, A.view, B.view, 0.5, ref)
        st = H.hclooc_dgemm_ex(ctx, M, N, K, 1.0, A, A.ld, B, B.ld, 0.5, C, C.ld, 0)
        assert st.plan.workspace_bytes <= ws.numel()
        assert np.array_equal(C.view, ref)
    finally:
        H.hclooc_ctx_destroy(ctx)


def test_runtime_calls_compose_a_manual_step(H):
    """The paper's runtime calls (hclMalloc .. hclWaitEvent, :109-116, :212) used directly for one step."""
    M, N, K = 192, 160, 96
    A, B, C = host_inputs(H, M, N, K, 40, "int")
    ref = C.view.copy()
    oracle.dgemm(1.0, A.view, B.view, 1.0, ref)
    assert H.hclGetMemSize(0) > (1 << 30)
    dA, dB, dC = H.hclMalloc(M * K * 8), H.hclMalloc(K * N * 8), H.hclMalloc(M * N * 8)
    s0, s1 = H.hclStreamCreate(), H.hclStreamCreate()
    rB = H.hclMemcpyAsync(dB, B, K * N * 8, H.HCL_H2D, s0, want_event=True)
    rA = H.hclMemcpyAsync(dA, A, M * K * 8, H.HCL_H2D, s0, want_event=True)
    rC = H.hclMemcpy2DAsync(dC, N * 8, C, C.ld * 8, N * 8, M, H.HCL_H2D, s0, want_event=True)
    for e in (rB, rA, rC):
        H.hclWaitEvent(s1, e)
    eA = H.hclDgemmAsync(M, N, K, 1.0, dA, K, dB, N, 1.0, dC, N, s1, want_event=True)
    H.hclWaitEvent(s0, eA)
    H.hclMemcpyAsync(C, dC, M * N * 8, H.HCL_D2H, s0)
    H.hclStreamSynchronize(s0)
    H.hclDeviceSynchronize(0)
    assert np.array_equal(C.view, ref)
    for e in (rB, rA, rC, eA):
        H.hclEventDestroy(e)
    for s in (s0, s1):
        H.hclStreamDestroy(s)
    for d in (dA, dB, dC):
        H.hclFree(d)


# ------------------------------------------------------------------ configs[1] at full size, sampled outputs
def test_config2_full_size_every_element(H):
    """BASELINE.json configs[1]: 8192^3, alpha 1, beta 1, budget 256 MiB, in the launch configuration bench.py times.
    SURVEY 8(c) verification matrix: "full oracle, every element" -- the float variant within 1e-13*D, the integer variant
    bit-exact; plus the whole-matrix checksums the larger configs rely on (here they can be compared with the full oracle)."""
    import oracle.checksum as cks
    M = N = K = 8192
    for dist, exact in (("uniform", False), ("int", True)):
        A, B, C = host_inputs(H, M, N, K, synthgen.BASE_SEED + 2, dist)
        x = synthgen.fill_numpy(N, 1, 77, "A", "int")[:, 0]; y = synthgen.fill_numpy(1, M, 77, "B", "int")[0]
        pre = cks.before(C.view, x, y)
        C0 = C.view.copy()
        st = H.hclooc_dgemm_ex(None, M, N, K, 1.0, A, A.ld, B, B.ld, 1.0, C, C.ld, 256 * MiB)
        assert st.plan.workspace_bytes <= 256 * MiB and st.bytes_h2d == st.plan.bytes_h2d and st.plan.n_steps > 16
        if not exact:        # the float variant: the full oracle, every element
            ref = C0
            D = oracle.dgemm(1.0, A.view, B.view, 1.0, ref, want_denominator=True)
            check(C.view, ref, D, exact)
        else:                # the integer variant: oracle rows and columns on both sides of every slab boundary, bit for bit ...
            plan = st.plan
            rng = np.random.default_rng(5)
            rows = {0, M - 1} | {int(v) for v in rng.integers(0, M, 6)} | {i * plan.mb - d for i in (1, plan.h // 2, plan.h - 1) for d in (0, 1)}
            cols = {0, N - 1} | {int(v) for v in rng.integers(0, N, 6)} | {j * plan.nb - d for j in range(1, plan.w) for d in (0, 1)}
            rows, cols = np.array(sorted(rows)), np.array(sorted(cols))
            ref_r, _ = oracle.dgemm_sub(1.0, A.view, B.view, 1.0, C0, rows=rows)
            ref_c, _ = oracle.dgemm_sub(1.0, A.view, B.view, 1.0, C0, cols=cols)
            check(C.view[rows], ref_r, None, True)
            check(C.view[:, cols], ref_c, None, True)
        Cx, yC, Dx, yD = cks.expected(1.0, A.view, B.view, 1.0, pre, x, y)       # ... and the exact checksums over the whole matrix
        gx, gy = C.view @ x, y @ C.view
        if exact:
            assert np.array_equal(gx, Cx) and np.array_equal(gy, yC)
        else:
            assert (np.abs(gx - Cx) <= RTOL * Dx).all() and (np.abs(gy - yC) <= RTOL * yD).all()
        for X in (A, B, C):
            X.free()


@pytest.mark.parametrize("M,N,K,budget", [(256, 16, 200000, 1 * MiB), (8, 16, 1000000, 1 * MiB), (100, 48, 150000, 1 * MiB)])
def test_k_panels_reread_the_host_block_after_its_download(H, M, N, K, budget):
    """K split with fewer blocks than C buffers (w == 1, few rows; down to h = w = 1): panel p's S(c_ij) reads the host
    block panel p-1's R(c_ij) wrote through ANOTHER C buffer, so the upload must wait for that download (the schedule's
    host-block rule, tests/test_planner_schedule.py).  Integers: every panel's contribution and beta*C0 arrive exactly."""
    plan = H.hclooc_plan(M, N, K, 1, 0, budget)
    assert plan.kpanels > 1
    for rep in range(3):                                     # a race shows up only sometimes: a few rounds
        A, B, C = host_inputs(H, M, N, K, 340 + rep, "int")
        ref = C.view.copy()
        oracle.dgemm(1.0, A.view, B.view, -3.0, ref)
        st = H.hclooc_dgemm_ex(None, M, N, K, 1.0, A, A.ld, B, B.ld, -3.0, C, C.ld, budget)
        assert st.plan.kpanels == plan.kpanels
        check(C.view, ref, None, exact=True)
        for X in (A, B, C):
            X.free()


def test_trace_records_every_copy_and_kernel(H):
    """hclooc_ctx_set_trace / get_trace: one record per copy and kernel of the last call, ordered in time."""
    M, N, K = 515, 389, 301
    A, B, C = host_inputs(H, M, N, K, 41, "int")
    ref = C.view.copy()
    oracle.dgemm(1.0, A.view, B.view, 0.5, ref)
    ctx = H.hclooc_ctx_create(0)
    try:
        H.hclooc_ctx_set_trace(ctx, True)
        st = H.hclooc_dgemm_ex(ctx, M, N, K, 1.0, A, A.ld, B, B.ld, 0.5, C, C.ld, 1 * MiB)
        tr = H.hclooc_ctx_get_trace(ctx)
        assert np.array_equal(C.view, ref)
        assert len(tr) == st.n_kernels + st.n_copies_h2d + st.n_copies_d2h
        assert int(tr["bytes"][tr["kind"] <= 2].sum()) == st.bytes_h2d and int(tr["bytes"][tr["kind"] == 4].sum()) == st.bytes_d2h
        assert tr["flops"].sum() == 2.0 * M * N * K
        assert (tr["t_end_ms"] >= tr["t_start_ms"]).all() and tr["t_start_ms"].min() >= 0.0
        for step in range(st.plan.n_steps):      # per step: uploads end before the kernel ends before the download ends
            r = tr[tr["step"] == step]
            k = r[r["kind"] == 3][0]
            assert (r[r["kind"] < 3]["t_end_ms"] <= k["t_end_ms"]).all()
            assert k["t_end_ms"] <= r[r["kind"] == 4][0]["t_end_ms"]
    finally:
        H.hclooc_ctx_destroy(ctx)


def test_device_resident_operands_run_in_core(H):
    """All three operands in device memory: the in-core case -- one DGEMM on the caller's
    matrices, nothing staged; a host operand or an unaligned device operand goes through the staged pipeline."""
    import torch
    M, N, K = 645, 518, 776
    A, B, C = host_inputs(H, M, N, K, 51, "int")
    ref = C.view.copy()
    oracle.dgemm(2.0, A.view, B.view, -1.0, ref)
    dA, dB = to_dev(A.view.copy()), to_dev(B.view.copy())
    dC = to_dev(C.view.copy())
    st = H.hclooc_dgemm_ex(None, M, N, K, 2.0, dA, K, dB, N, -1.0, dC, N, 1 * MiB)
    assert st.n_kernels == 1 and st.bytes_h2d == 0 and st.bytes_d2h == 0 and st.plan.workspace_bytes == 0
    assert st.plan.h == 1 and st.plan.w == 1
    assert np.array_equal(dC.cpu().numpy(), ref)
    # mixed residency: A on the host, B and C on the device -> staged, same values
    dC2 = to_dev(C.view.copy())
    st = H.hclooc_dgemm_ex(None, M, N, K, 2.0, A, A.ld, dB, N, -1.0, dC2, N, 1 * MiB)
    assert st.n_kernels > 1 and st.plan.workspace_bytes <= 1 * MiB
    assert np.array_equal(dC2.cpu().numpy(), ref)
    # odd leading dimension of C on the device: not addressable by the vector epilogue/TMA rules -> staged
    dC3 = torch.zeros(M, N + 1, dtype=torch.float64, device="cuda")
    dC3[:, :N] = to_dev(C.view.copy())
    torch.cuda.synchronize()
    st = H.hclooc_dgemm_ex(None, M, N, K, 2.0, dA, K, dB, N, -1.0, dC3, N + 1, 1 * MiB)
    assert st.n_kernels > 1
    assert np.array_equal(dC3[:, :N].cpu().numpy(), ref) and float(dC3[:, N].abs().max()) == 0.0


@pytest.mark.parametrize("M,N,K,dist", [
    (1700, 1500, 1040, "int"),        # 14 x 12 = 168 tiles >= 148 SMs: one wave joins the stream-K tail, ragged edges
    (1700, 1500, 1040, "uniform"),
    (2048, 2432, 512, "int"),         # 16 x 19 = 304 tiles = 2 waves + 8: data-parallel wave + tail
    (384, 640, 4100, "int"),          # 15 tiles < 148: every tile is cut along K among several CTAs
    (128, 128, 70000, "uniform"),     # one tile shared by 148 CTAs
    (130, 120, 16, "int"),            # a single k block per tile: nothing to split
])
def test_streamk_kernel_matches_oracle(H, M, N, K, dist):
    """The persistent stream-K kernel (in-core path of hclooc_dgemm_ex on device operands): partial tiles are
    summed in k order by whichever CTA arrives last, so the result is deterministic -- launched three times on
    the same inputs (the scratch counters must reset themselves) and compared with the oracle each time."""
    import torch
    A = synthgen.fill(np.empty((M, K)), 61, "A", dist)
    B = synthgen.fill(np.empty((K, N)), 61, "B", dist)
    C0 = synthgen.fill(np.empty((M, N)), 61, "C", dist)
    ref = C0.copy()
    D = oracle.dgemm(1.5, A, B, -0.5, ref, want_denominator=True)
    dA, dB = to_dev(A), to_dev(B)
    outs = []
    for rep in range(3):
        dC = to_dev(C0)
        st = H.hclooc_dgemm_ex(None, M, N, K, 1.5, dA, K, dB, N, -0.5, dC, N, 0)
        assert st.n_kernels == 1
        outs.append(dC.cpu().numpy())
        check(outs[-1], ref, D, exact=(dist == "int"))
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])      # bitwise repeatable


def test_streamk_launches_on_two_streams_do_not_share_scratch(H):
    """Concurrent stream-K launches (hclDgemmAsync on two streams) each get a scratch buffer of their own."""
    import torch
    M, N, K = 1700, 1500, 1040
    A = synthgen.fill(np.empty((M, K)), 62, "A", "int")
    B = synthgen.fill(np.empty((K, N)), 62, "B", "int")
    C0 = synthgen.fill(np.empty((M, N)), 62, "C", "int")
    ref = C0.copy()
    oracle.dgemm(1.0, A, B, 1.0, ref)
    dA, dB = to_dev(A), to_dev(B)
    streams = [torch.cuda.Stream() for _ in range(3)]
    dCs = [[to_dev(C0) for _ in range(4)] for _ in streams]
    torch.cuda.synchronize()
    for r in range(4):
        for s, row in zip(streams, dCs):
            H.hclDgemmAsync(M, N, K, 1.0, dA, K, dB, N, 1.0, row[r], N, s)
    torch.cuda.synchronize()
    for row in dCs:
        for dC in row:
            assert np.array_equal(dC.cpu().numpy(), ref)


@pytest.mark.parametrize("M,N,K,alpha,beta,budget,dist", [
    (512, 512, 512, 1.0, 0.5, 1 * MiB, "int"),          # configs[0]: every block streams
    (512, 512, 512, 1.0, 0.5, 1 * MiB, "uniform"),
    (4, 4, 8, 1.0, 1.0, 44 * 8, "int"),                 # the paper's worked example (:301): h = 4, w = 2, 8 steps
    (768, 640, 300, 2.0, 0.0, 2 * MiB, "int"),          # beta == 0: C is not uploaded, NaN in C is overwritten
    (384, 1030, 257, -1.0, 1.0, 3 * MiB, "int"),        # odd slice widths (device leading dimensions padded)
    (300, 200, 100, 1.0, 1.0, 64 * MiB, "int"),         # fits: the in-core case, one step
])
def test_fig2_pipeline_matches_oracle(H, M, N, K, alpha, beta, budget, dist):
    """hclooc_dgemm_fig2: the paper's Figure 2 (two round-robin streams, eA/rA/rB/eC/rC events, single B buffer)
    over the hcl* runtime calls gives the oracle's values; its traffic is the paper's w*M*K + K*N + M*N."""
    A, B, C = host_inputs(H, M, N, K, 71, dist, poison_c=(beta == 0.0))
    ref = C.view.copy() if beta != 0.0 else np.zeros((M, N))
    D = oracle.dgemm(alpha, A.view, B.view, beta, ref, want_denominator=True)
    st = H.hclooc_dgemm_fig2(M, N, K, alpha, A, A.ld, B, B.ld, beta, C, C.ld, budget)
    check(C.view, ref, D, exact=(dist == "int"))
    h, w = st.plan.h, st.plan.w
    if 8 * (M * K + K * N + M * N) <= budget:
        assert (h, w) == (1, 1) and st.n_kernels == 1
    else:
        assert (h, w) == H.hclMatrixPartitioner(M, N, K, budget // 8) and st.n_kernels == h * w
    assert st.bytes_h2d == 8 * (w * M * K + K * N + (M * N if beta != 0.0 else 0)) and st.bytes_d2h == 8 * M * N
    assert st.plan.workspace_bytes <= budget
    if (M, N, K) == (4, 4, 8):
        assert (h, w) == (4, 2)                           # Figure 3 (:281)


def test_repeated_identical_call_replays_a_cuda_graph(H):
    """A short, latency-bound schedule (configs[0]) is captured as a CUDA graph when the very same call comes a
    second time and replayed from the third on; every repetition must equal the oracle bit for bit and report
    the same traffic, and a different call in between must not reuse the graph."""
    M = N = K = 512
    A, B, C = host_inputs(H, M, N, K, 81, "int")
    C0 = C.view.copy()
    ref = C0.copy()
    oracle.dgemm(1.0, A.view, B.view, 0.5, ref)
    ctx = H.hclooc_ctx_create(0)
    try:
        stats = []
        for rep in range(4):                              # ordinary, capture + launch, replay, replay
            C.view[...] = C0
            stats.append(H.hclooc_dgemm_ex(ctx, M, N, K, 1.0, A, A.ld, B, B.ld, 0.5, C, C.ld, 1 * MiB))
            check(C.view, ref, None, exact=True)
        assert len({(s.bytes_h2d, s.bytes_d2h, s.n_kernels, s.n_copies_h2d, s.n_copies_d2h) for s in stats}) == 1
        # another alpha: not the captured call
        ref2 = C0.copy()
        oracle.dgemm(-2.0, A.view, B.view, 0.5, ref2)
        C.view[...] = C0
        H.hclooc_dgemm_ex(ctx, M, N, K, -2.0, A, A.ld, B, B.ld, 0.5, C, C.ld, 1 * MiB)
        check(C.view, ref2, None, exact=True)
        # and back: seen before, but the graph belongs to the call before the last one -> captured afresh
        for rep in range(3):
            C.view[...] = C0
            H.hclooc_dgemm_ex(ctx, M, N, K, 1.0, A, A.ld, B, B.ld, 0.5, C, C.ld, 1 * MiB)
            check(C.view, ref, None, exact=True)
    finally:
        H.hclooc_ctx_destroy(ctx)


@pytest.mark.parametrize("dist", ["int", "uniform"])
def test_nsteps_mode_keeps_c_on_the_device(H, dist):
    """hclooc_dgemm_nsteps: C is uploaded at step 0, stays in device memory while a blocked
    algorithm adds one K panel per call, and comes back at the last step.  Same values as the oracle applied
    panel by panel; no C traffic over the link in between; host C untouched until the end."""
    M, N, Kp, nsteps = 520, 392, 160, 4
    A = [H.HostMatrix(M, Kp) for _ in range(nsteps)]
    B = [H.HostMatrix(Kp, N) for _ in range(nsteps)]
    C = H.HostMatrix(M, N)
    for p in range(nsteps):
        synthgen.fill(A[p].array, 90 + p, "A", dist)
        synthgen.fill(B[p].array, 90 + p, "B", dist)
    synthgen.fill(C.array, 90, "C", dist)
    C0 = C.view.copy()
    ref = C0.copy()
    D = np.zeros((M, N))
    for p in range(nsteps):                               # the oracle, one panel after the other: beta first, then 1
        Dp = oracle.dgemm(2.0, A[p].view, B[p].view, 0.5 if p == 0 else 1.0, ref, want_denominator=True)
        D = Dp if p == 0 else D + Dp                      # a (generous) running denominator for the float gate
    ctx = H.hclooc_ctx_create(0)
    try:
        step = 0
        for p in range(nsteps):
            step, st = H.hclooc_dgemm_nsteps(ctx, M, N, Kp, 2.0, A[p], Kp, B[p], N, 0.5 if p == 0 else 1.0, C, N,
                                             4 * MiB, nsteps, step)
            assert step == p + 1 and st.plan.c_on_device == 1
            assert st.bytes_d2h == (M * N * 8 if p == nsteps - 1 else 0)
            ab = st.bytes_h2d - (M * N * 8 if p == 0 else 0)
            assert M * Kp * 8 + Kp * N * 8 <= ab <= st.plan.w * M * Kp * 8 + Kp * N * 8      # only A and B cross the link
            if p < nsteps - 1:
                assert np.array_equal(C.view, C0)         # host C is written only at the last step
        check(C.view, ref, D, exact=(dist == "int"))
        with pytest.raises(H.HclError):                   # a sequence must start at step 0 with its own C
            H.hclooc_dgemm_nsteps(ctx, M, N, Kp, 1.0, A[0], Kp, B[0], N, 1.0, C, N, 4 * MiB, nsteps, 2)
        with pytest.raises(H.HclError) as e:              # C larger than the budget: the mode does not apply
            H.hclooc_dgemm_nsteps(ctx, M, N, Kp, 1.0, A[0], Kp, B[0], N, 1.0, C, N, 1 * MiB, nsteps, 0)
        assert e.value.status == 1
    finally:
        H.hclooc_ctx_destroy(ctx)


# ------------------------------------------------------------------ direct mode (plan.direct): TMA straight from host memory
@pytest.mark.parametrize("dist,exact", [("uniform", False), ("int", True)])
def test_config1_direct_mode_uses_no_device_memory(H, dist, exact):
    """BASELINE.json configs[0] through the direct mode: no device buffer at all (0 <= 1 MiB), one launch, every
    tile streams its A and B panels from pinned host memory through TMA and updates C in host memory."""
    M = N = K = 512
    A, B, C = host_inputs(H, M, N, K, synthgen.BASE_SEED + 1, dist)
    ref = C.view.copy()
    D = oracle.dgemm(1.0, A.view, B.view, 0.5, ref, want_denominator=True)
    staged = C.view.copy()
    ctx = H.hclooc_ctx_create(0)
    try:
        H.hclooc_ctx_set_direct(ctx, 1)
        st = H.hclooc_dgemm_ex(ctx, M, N, K, 1.0, A, A.ld, B, B.ld, 0.5, C, C.ld, 1 * MiB)
        assert st.plan.direct == 1 and st.plan.workspace_bytes == 0 and st.n_kernels == 1
        assert st.n_copies_h2d == 0 and st.n_copies_d2h == 0
        # 4 x 4 tiles in ONE 16-CTA cluster sharing its loads by TMA multicast: A and B cross the link once (compulsory traffic)
        cm, cn = st.plan.direct_cm, st.plan.direct_cn
        assert (cm, cn) in ((4, 4), (2, 4))
        assert st.bytes_h2d == 8 * ((4 // cn) * M * K + (4 // cm) * K * N + M * N) and st.bytes_d2h == 8 * M * N
        check(C.view, ref, D, exact)
        direct = C.view.copy()
        # the staged pipeline on the same inputs: same kernel, same summation order -> the same bits
        H.hclooc_ctx_set_direct(ctx, 0)
        synthgen.fill(C.array, synthgen.BASE_SEED + 1, "C", dist, cols=N)
        st = H.hclooc_dgemm_ex(ctx, M, N, K, 1.0, A, A.ld, B, B.ld, 0.5, C, C.ld, 1 * MiB)
        assert st.plan.direct == 0 and st.plan.n_steps > 4
        assert np.array_equal(C.view.view(np.uint64), direct.view(np.uint64))
    finally:
        H.hclooc_ctx_destroy(ctx)
    with pytest.raises(H.HclError) as e:
        H.hclooc_ctx_set_direct(None, 2)
    assert e.value.status == -2


@pytest.mark.parametrize("M,N,K,alpha,beta,dist,pads", [
    (1, 1, 1, 2.0, 0.5, "uniform", (1, 1, 1)),
    (300, 260, 200, 1.0, 0.5, "uniform", (0, 0, 0)),          # ragged in m, n and k
    (129, 257, 33, -1.5, 1.0, "normal", (3, 1, 5)),           # odd sizes made even by the padding
    (517, 389, 1000, 2.0, -1.0, "int", (2, 3, 1)),
    (131, 78, 97, 3.0, 0.0, "int", (1, 2, 4)),                # beta == 0: C (NaN) is not read over the link
    (1500, 1300, 260, 1.0, 0.5, "int", (0, 0, 0)),            # 132 tiles
    (2200, 1800, 70, 1.0, 1.0, "uniform", (0, 2, 2)),         # 270 tiles: more than one wave
])
def test_direct_mode_matches_oracle(H, M, N, K, alpha, beta, dist, pads):
    A, B, C = host_inputs(H, M, N, K, 43, dist, pads=pads, poison_c=(beta == 0.0))
    ref = np.zeros((M, N)) if beta == 0.0 else C.view.copy()
    D = oracle.dgemm(alpha, A.view, B.view, beta, ref, want_denominator=True)
    ctx = H.hclooc_ctx_create(0)
    try:
        H.hclooc_ctx_set_direct(ctx, 1)
        st = H.hclooc_dgemm_ex(ctx, M, N, K, alpha, A, A.ld, B, B.ld, beta, C, C.ld, 1 * MiB)
        assert st.plan.direct == 1 and st.plan.workspace_bytes == 0
        tm, tn = -(-M // 128), -(-N // 128)
        cm, cn = st.plan.direct_cm, st.plan.direct_cn
        assert cm in (1, 2, 4) and cn in (1, 2, 4) and (cm > 1 or tm == 1) and (cn > 1 or tn == 1)
        assert st.bytes_h2d == 8 * (-(-tn // cn) * M * K + -(-tm // cm) * K * N + (M * N if beta != 0.0 else 0))
        check(C.view, ref, D, exact=(dist == "int"))
        assert np.isnan(C.array[:, N:]).all()                                   # host padding of C untouched
    finally:
        H.hclooc_ctx_destroy(ctx)


def test_direct_mode_falls_back_and_degenerates(H):
    """Odd leading dimensions are not TMA-legal: the call is staged even when direct mode is forced.  alpha == 0
    scales C in host memory without touching A and B; registered (not cudaHostAlloc'ed) memory works too."""
    ctx = H.hclooc_ctx_create(0)
    try:
        H.hclooc_ctx_set_direct(ctx, 1)
        M, N, K = 200, 150, 101
        A, B, C = host_inputs(H, M, N, K, 44, "int")                            # lda = 101: odd
        ref = C.view.copy()
        oracle.dgemm(1.0, A.view, B.view, 0.5, ref)
        st = H.hclooc_dgemm_ex(ctx, M, N, K, 1.0, A, A.ld, B, B.ld, 0.5, C, C.ld, 1 * MiB)
        assert st.plan.direct == 0 and st.plan.workspace_bytes > 0
        assert np.array_equal(C.view, ref)
        # alpha == 0
        M, N, K = 300, 200, 64
        A, B, C = host_inputs(H, M, N, K, 44, "uniform")
        A.array[...] = np.nan; B.array[...] = np.nan
        C0 = C.view.copy()
        st = H.hclooc_dgemm_ex(ctx, M, N, K, 0.0, A, A.ld, B, B.ld, -2.0, C, C.ld, 1 * MiB)
        assert st.plan.direct == 1 and st.plan.scale_only == 1 and st.bytes_h2d == 8 * M * N
        assert np.array_equal(C.view, -2.0 * C0)
        C.view[...] = np.nan
        H.hclooc_dgemm_ex(ctx, M, N, K, 0.0, A, A.ld, B, B.ld, 0.0, C, C.ld, 1 * MiB)
        assert np.array_equal(C.view, np.zeros((M, N))) and not np.signbit(C.view).any()
        # pinned in place with hclooc_host_register
        M, N, K = 256, 128, 64
        a = synthgen.fill(np.empty((M, K)), 45, "A", "int"); b = synthgen.fill(np.empty((K, N)), 45, "B", "int")
        c = synthgen.fill(np.empty((M, N)), 45, "C", "int")
        ref = c.copy()
        oracle.dgemm(2.0, a, b, 1.0, ref)
        for x in (a, b, c):
            H.hclooc_host_register(x, x.nbytes)
        try:
            st = H.hclooc_dgemm_ex(ctx, M, N, K, 2.0, a, K, b, N, 1.0, c, N, 1 * MiB)
        finally:
            for x in (a, b, c):
                H.hclooc_host_unregister(x)
        assert np.array_equal(c, ref)
    finally:
        H.hclooc_ctx_destroy(ctx)


# ------------------------------------------------------------------ transposed operands (hclooc_dgemm_t)
def stored_inputs(H, transa, transb, M, N, K, seed, dist, pads=(0, 0, 0)):
    """A, B as the caller stores them (A is K x M when transa, B is N x K when transb), C; NaN padding."""
    ar, ac = (K, M) if transa else (M, K)
    br, bc = (N, K) if transb else (K, N)
    A = H.HostMatrix(ar, ac, ac + pads[0]); B = H.HostMatrix(br, bc, bc + pads[1]); C = H.HostMatrix(M, N, N + pads[2])
    for X in (A, B, C):
        X.array[...] = np.nan
    synthgen.fill(A.array, seed, "A", dist, cols=ac); synthgen.fill(B.array, seed, "B", dist, cols=bc)
    synthgen.fill(C.array, seed, "C", dist, cols=N)
    return A, B, C


@pytest.mark.parametrize("transa,transb", [(1, 0), (0, 1), (1, 1)])
@pytest.mark.parametrize("M,N,K,alpha,beta,dist,pads,budget", [
    (300, 260, 200, 1.0, 0.5, "uniform", (0, 0, 0), 1 * MiB),
    (129, 257, 33, -1.5, 1.0, "normal", (3, 1, 5), 1 * MiB),
    (517, 389, 1000, 2.0, -1.0, "int", (2, 3, 1), 2 * MiB),        # many staging blocks per slice
    (1, 1, 1, 2.0, 0.5, "int", (1, 1, 1), 1 * MiB),
    (640, 1100, 700, 1.0, 0.0, "int", (0, 0, 0), 64 * MiB),        # beta == 0
    (96, 112, 20000, 2.0, -1.0, "int", (0, 0, 0), 900 * 1024),     # K panels
])
def test_transposed_operands_match_oracle(H, transa, transb, M, N, K, alpha, beta, dist, pads, budget):
    """C = alpha*op(A)*op(B) + beta*C: the oracle gets op(A), op(B) written out; the library gets the stored matrices."""
    A, B, C = stored_inputs(H, transa, transb, M, N, K, 46, dist, pads)
    opA, opB = np.empty((M, K)), np.empty((K, N))
    opA[...] = A.view.T if transa else A.view
    opB[...] = B.view.T if transb else B.view
    if beta == 0.0:
        C.view[...] = np.nan
    ref = np.zeros((M, N)) if beta == 0.0 else C.view.copy()
    D = oracle.dgemm(alpha, opA, opB, beta, ref, want_denominator=True)
    st = H.hclooc_dgemm_t(None, transa, transb, M, N, K, alpha, A, A.ld, B, B.ld, beta, C, C.ld, budget)
    assert st.plan.direct == 0 and 0 < st.plan.workspace_bytes <= budget
    assert st.plan.trans == transa + 2 * transb
    assert st.bytes_h2d == st.plan.bytes_h2d and st.bytes_d2h == st.plan.bytes_d2h
    check(C.view, ref, D, exact=(dist == "int"))
    assert np.isnan(C.array[:, N:]).all()


def test_transposed_call_equals_plain_call_on_written_out_transposes(H):
    """Same kernel, same order of summation: hclooc_dgemm_t on stored A^T, B^T gives the bits of hclooc_dgemm_ex on
    op(A), op(B) (K below the cluster split-K threshold, not split into panels)."""
    M, N, K = 515, 389, 301
    A, B, C = stored_inputs(H, 1, 1, M, N, K, 47, "uniform", pads=(1, 3, 7))
    opA, opB = H.HostMatrix(M, K), H.HostMatrix(K, N)
    opA.view[...] = A.view.T; opB.view[...] = B.view.T
    C2 = H.HostMatrix(M, N); C2.view[...] = C.view
    st = H.hclooc_dgemm_t(None, H.HCL_OP_T, H.HCL_OP_T, M, N, K, -0.75, A, A.ld, B, B.ld, 1.25, C, C.ld, 4 * MiB)
    st2 = H.hclooc_dgemm_ex(None, M, N, K, -0.75, opA, opA.ld, opB, opB.ld, 1.25, C2, C2.ld, 4 * MiB)
    assert st.plan.kpanels == 1 and st2.plan.kpanels == 1
    assert np.array_equal(C.view.view(np.uint64), C2.view.view(np.uint64))
    # HCL_OP_N, HCL_OP_N through the same entry point is hclooc_dgemm_ex
    C3 = H.HostMatrix(M, N); synthgen.fill(C3.array, 47, "C", "uniform", cols=N)
    st3 = H.hclooc_dgemm_t(None, 0, 0, M, N, K, -0.75, opA, opA.ld, opB, opB.ld, 1.25, C3, C3.ld, 4 * MiB)
    assert st3.plan.trans == 0
    assert np.array_equal(C3.view.view(np.uint64), C2.view.view(np.uint64))


def test_transposed_argument_errors(H):
    M, N, K = 64, 48, 32
    A, B, C = stored_inputs(H, 1, 1, M, N, K, 48, "uniform")
    before = C.view.copy()
    for args, want in (((2, 0, M, N, K, 1.0, A, M, B, K, 1.0, C, N), -15), ((0, 3, M, N, K, 1.0, A, M, B, K, 1.0, C, N), -16),
                       ((1, 1, M, N, K, 1.0, A, M - 1, B, K, 1.0, C, N), -6),       # stored A is K x M: lda >= M
                       ((1, 1, M, N, K, 1.0, A, M, B, K - 1, 1.0, C, N), -8),       # stored B is N x K: ldb >= K
                       ((1, 1, M, N, K, 1.0, A, M, B, K, 1.0, C, N - 1), -11)):
        with pytest.raises(H.HclError) as e:
            H.hclooc_dgemm_t(None, *args, 1 * MiB)
        assert e.value.status == want, (args[:2], e.value.status)
    assert np.array_equal(C.view, before)


@pytest.mark.parametrize("transa,transb", [(1, 0), (0, 1), (1, 1)])
@pytest.mark.parametrize("M,N,K,alpha,beta,dist,variant", [
    (128, 128, 32, 1.0, 0.0, "uniform", 1),          # one tile, one k block
    (300, 260, 200, 1.0, 0.5, "uniform", 1),         # ragged in m, n and k
    (129, 257, 33, -1.5, 1.0, "normal", 1),
    (131, 77, 97, 3.0, 2.0, "int", 1),
    (517, 389, 1000, 2.0, -1.0, "int", 0),
    (128, 256, 4096, 1.0, 0.5, "uniform", 4),        # cluster split-K over the transposed layouts
    (200, 300, 2061, -1.0, 2.0, "int", 2),
    (1500, 1400, 300, 1.0, 0.5, "int", 0),           # 132 tiles
])
def test_tile_kernel_transposed_layouts(H, transa, transb, M, N, K, alpha, beta, dist, variant):
    """hclDgemmAsyncT on device pointers: A stored K x M and / or B stored N x K, read by the kernel as they are."""
    import torch
    ar, ac = (K, M) if transa else (M, K)
    br, bc = (N, K) if transb else (K, N)
    lda, ldb, ldc = ac + (ac % 2) + 4, bc + (bc % 2) + 2, N + (N % 2) + 6
    A = np.full((ar, lda), np.nan); B = np.full((br, ldb), np.nan); C0 = np.full((M, ldc), np.nan)
    synthgen.fill(A, 51, "A", dist, cols=ac); synthgen.fill(B, 51, "B", dist, cols=bc); synthgen.fill(C0, 51, "C", dist, cols=N)
    if beta == 0.0:
        C0[:, :N] = np.nan
    dA, dB, dC = (to_dev(x) for x in (A, B, C0))
    H.hclDgemmAsyncT(transa, transb, M, N, K, alpha, dA, lda, dB, ldb, beta, dC, ldc, torch.cuda.current_stream(), variant=variant)
    torch.cuda.synchronize()
    got = dC.cpu().numpy()
    opA, opB = np.empty((M, K)), np.empty((K, N))
    opA[...] = A[:, :ac].T if transa else A[:, :ac]
    opB[...] = B[:, :bc].T if transb else B[:, :bc]
    ref = C0[:, :N].copy()
    D = oracle.dgemm(alpha, opA, opB, beta, ref, want_denominator=True)
    check(got[:, :N], ref, D, exact=(dist == "int"))
    assert np.isnan(got[:, N:]).all()
    if variant in (0, 1) and K < 1024:
        # the same bits as the untransposed kernel on written-out transposes (same order of summation)
        pa, pb = np.zeros((M, K + K % 2)), np.zeros((K, N + N % 2))                  # even leading dimensions
        pa[:, :K] = opA; pb[:, :N] = opB
        dA2, dB2, dC2 = to_dev(pa), to_dev(pb), to_dev(C0)
        H.hclDgemmAsyncEx(M, N, K, alpha, dA2, K + K % 2, dB2, N + N % 2, beta, dC2, ldc, torch.cuda.current_stream(), variant=1)
        torch.cuda.synchronize()
        assert np.array_equal(dC2.cpu().numpy()[:, :N].view(np.uint64), got[:, :N].view(np.uint64))
    with pytest.raises(H.HclError) as e:
        H.hclDgemmAsyncT(transa, 2, M, N, K, alpha, dA, lda, dB, ldb, beta, dC, ldc, torch.cuda.current_stream())
    assert e.value.status == -16


def test_transposed_in_core_and_direct_modes(H):
    """Device-resident transposed operands run in core (one launch, nothing staged); mapped host operands in direct mode."""
    import torch
    M, N, K = 700, 520, 384
    A, B, C = stored_inputs(H, 1, 1, M, N, K, 52, "int")
    ref = C.view.copy()
    oracle.dgemm(1.0, A.view.T.copy(), B.view.T.copy(), 0.5, ref)
    dA, dB, dC = (to_dev(X.view.copy()) for X in (A, B, C))
    st = H.hclooc_dgemm_t(None, 1, 1, M, N, K, 1.0, dA, M, dB, K, 0.5, dC, N, 0)
    assert st.plan.n_steps == 1 and st.plan.workspace_bytes == 0 and st.bytes_h2d == 0
    assert np.array_equal(dC.cpu().numpy(), ref)
    ctx = H.hclooc_ctx_create(0)
    try:
        H.hclooc_ctx_set_direct(ctx, 1)
        st = H.hclooc_dgemm_t(ctx, 1, 1, M, N, K, 1.0, A, A.ld, B, B.ld, 0.5, C, C.ld, 1 * MiB)
        assert st.plan.direct == 1 and st.plan.trans == 3 and st.plan.workspace_bytes == 0
        assert np.array_equal(C.view, ref)
    finally:
        H.hclooc_ctx_destroy(ctx)


@pytest.mark.parametrize("transa,transb", [(1, 0), (0, 1), (1, 1)])
@pytest.mark.parametrize("M,N,K,dist", [
    (1700, 1500, 1040, "int"),        # 168 tiles: one wave joins the stream-K tail, ragged edges
    (2048, 2432, 512, "uniform"),     # 2 waves + 8 tiles
    (384, 640, 4100, "int"),          # 15 tiles cut along K among several CTAs
])
def test_streamk_kernel_transposed_layouts(H, transa, transb, M, N, K, dist):
    """The persistent stream-K kernel on operands stored transposed (variant -1 of hclDgemmAsyncT), and through the
    in-core path of hclooc_dgemm_t; the same bits as the untransposed stream-K launch on written-out transposes."""
    import torch
    ar, ac = (K, M) if transa else (M, K)
    br, bc = (N, K) if transb else (K, N)
    A = synthgen.fill(np.empty((ar, ac)), 62, "A", dist); B = synthgen.fill(np.empty((br, bc)), 62, "B", dist)
    C0 = synthgen.fill(np.empty((M, N)), 62, "C", dist)
    opA, opB = np.empty((M, K)), np.empty((K, N))
    opA[...] = A.T if transa else A
    opB[...] = B.T if transb else B
    ref = C0.copy()
    D = oracle.dgemm(1.5, opA, opB, -0.5, ref, want_denominator=True)
    dA, dB, dC = to_dev(A), to_dev(B), to_dev(C0)
    H.hclDgemmAsyncT(transa, transb, M, N, K, 1.5, dA, ac, dB, bc, -0.5, dC, N, torch.cuda.current_stream(), variant=-1)
    torch.cuda.synchronize()
    got = dC.cpu().numpy()
    check(got, ref, D, exact=(dist == "int"))
    dA2, dB2, dC2 = to_dev(opA), to_dev(opB), to_dev(C0)
    H.hclDgemmAsyncEx(M, N, K, 1.5, dA2, K, dB2, N, -0.5, dC2, N, torch.cuda.current_stream(), variant=-1)
    torch.cuda.synchronize()
    assert np.array_equal(dC2.cpu().numpy().view(np.uint64), got.view(np.uint64))
    dC3 = to_dev(C0)
    st = H.hclooc_dgemm_t(None, transa, transb, M, N, K, 1.5, dA, ac, dB, bc, -0.5, dC3, N, 0)
    assert st.n_kernels == 1 and st.plan.trans == transa + 2 * transb
    check(dC3.cpu().numpy(), ref, D, exact=(dist == "int"))


@pytest.mark.parametrize("cm,cn", [(1, 2), (2, 1), (2, 2), (1, 4), (4, 1), (2, 4), (4, 2), (4, 4)])
@pytest.mark.parametrize("M,N,K,alpha,beta,dist", [
    (512, 512, 96, 1.0, 0.5, "int"),              # whole clusters
    (300, 700, 200, -1.5, 1.0, "uniform"),        # ragged tiles and clusters padded with tiles outside C
    (129, 130, 33, 2.0, 0.0, "int"),
    (1300, 900, 70, 1.0, 0.5, "uniform"),         # several clusters
])
def test_cluster_multicast_kernel_matches_tile_kernel(H, cm, cn, M, N, K, alpha, beta, dist):
    """HCL_DGEMM_CLUSTER(cm, cn): the direct-mode kernel (cm x cn CTAs per cluster sharing their loads by TMA multicast)
    on device pointers -- within the gate of the oracle and the very bits of the one-CTA-per-tile kernel."""
    import torch
    lda, ldb, ldc = K + (K % 2) + 4, N + (N % 2) + 2, N + (-N % 4) + 8
    A = np.full((M, lda), np.nan); B = np.full((K, ldb), np.nan); C0 = np.full((M, ldc), np.nan)
    synthgen.fill(A, 71, "A", dist, cols=K); synthgen.fill(B, 71, "B", dist, cols=N); synthgen.fill(C0, 71, "C", dist, cols=N)
    if beta == 0.0:
        C0[:, :N] = np.nan
    dA, dB, dC, dC1 = (to_dev(x) for x in (A, B, C0, C0))
    H.hclDgemmAsyncEx(M, N, K, alpha, dA, lda, dB, ldb, beta, dC, ldc, torch.cuda.current_stream(), variant=100 + 10 * cm + cn)
    H.hclDgemmAsyncEx(M, N, K, alpha, dA, lda, dB, ldb, beta, dC1, ldc, torch.cuda.current_stream(), variant=1)
    torch.cuda.synchronize()
    got, one = dC.cpu().numpy(), dC1.cpu().numpy()
    ref = C0[:, :N].copy()
    D = oracle.dgemm(alpha, A[:, :K], B[:, :N], beta, ref, want_denominator=True)
    check(got[:, :N], ref, D, exact=(dist == "int"))
    assert np.isnan(got[:, N:]).all()
    assert np.array_equal(got[:, :N].view(np.uint64), one[:, :N].view(np.uint64))


def test_fp64_probe_reports_the_dmma_rate(H):
    """hclooc_probe_fp64: the measured denominator of the roofline (37.2 TFLOP/s on a B200)."""
    dmma = H.hclooc_probe_fp64(0, 4, 0.3)
    dfma = H.hclooc_probe_fp64(1, 4, 0.3)
    assert 20.0 < dmma < 45.0 and 15.0 < dfma < 45.0, (dmma, dfma)
    for args, want in (((2, 4, 0.3), -1), ((0, 9, 0.3), -2), ((0, 4, 0.0), -3)):
        with pytest.raises(H.HclError) as e:
            H.hclooc_probe_fp64(*args)
        assert e.value.status == want


# ------------------------------------------------------------------ out-of-core DSYRK on the same path
@pytest.mark.parametrize("uplo", [0, 1])
@pytest.mark.parametrize("trans", [0, 1])
@pytest.mark.parametrize("N,K,alpha,beta,dist,pad,budget", [
    (300, 200, 1.0, 0.5, "uniform", 0, 1 * MiB),
    (517, 389, 2.0, -1.0, "int", 3, 2 * MiB),
    (129, 33, -1.5, 0.0, "int", 1, 1 * MiB),              # beta == 0: blocks crossing the diagonal are still uploaded
    (1, 1, 2.0, 0.5, "int", 1, 1 * MiB),
    (1300, 260, 1.0, 1.0, "normal", 2, 64 * MiB),
    (96, 20000, 2.0, -1.0, "int", 0, 900 * 1024),          # K panels
])
def test_dsyrk_matches_oracle_and_leaves_the_other_triangle(H, uplo, trans, N, K, alpha, beta, dist, pad, budget):
    ar, ac = (K, N) if trans else (N, K)
    A = H.HostMatrix(ar, ac, ac + pad); C = H.HostMatrix(N, N, N + pad)
    A.array[...] = np.nan; C.array[...] = np.nan
    synthgen.fill(A.array, 81, "A", dist, cols=ac); synthgen.fill(C.array, 81, "C", dist, cols=N)
    other = np.triu(np.ones((N, N), bool), 1) if uplo == 0 else np.tril(np.ones((N, N), bool), -1)
    if beta == 0.0:
        C.view[~other] = np.nan                            # the referenced triangle must not be read
    marker = C.view.copy()
    marker[other] = np.arange(int(other.sum())) + 0.25      # recognisable values in the triangle that is not referenced
    C.view[...] = marker
    ref = np.where(np.isnan(marker), 0.0, marker) if beta == 0.0 else marker.copy()
    D = oracle.dsyrk(uplo, trans, alpha, A.view.copy(), beta, ref, want_denominator=True)
    st = H.hclooc_dsyrk(None, uplo, trans, N, K, alpha, A, A.ld, beta, C, C.ld, budget)
    assert st.n_kernels >= 1 and st.plan.workspace_bytes <= budget
    got = C.view.copy()
    assert np.array_equal(got[other], marker[other])                               # untouched, bit for bit
    keep = ~other
    gk, rk = got.copy(), ref.copy()
    gk[other] = 0.0; rk[other] = 0.0
    D[other] = 1.0
    check(gk, rk, D, exact=(dist == "int"))
    assert np.isnan(C.array[:, N:]).all()


def test_dsyrk_large_blocks_symmetry_and_errors(H):
    """N > 4096: several block columns / rows; lower and upper results are transposes of each other bit for bit; the
    sampled rows agree with the oracle; argument errors."""
    N, K = 5000, 300
    A = H.HostMatrix(N, K); synthgen.fill(A.array, 82, "A", "uniform")
    lo, up = H.HostMatrix(N, N), H.HostMatrix(N, N)
    lo.view[...] = 0.0; up.view[...] = 0.0
    st = H.hclooc_dsyrk(None, H.HCL_UPLO_LOWER, H.HCL_OP_N, N, K, 1.0, A, K, 0.0, lo, N, 256 * MiB)
    H.hclooc_dsyrk(None, H.HCL_UPLO_UPPER, H.HCL_OP_N, N, K, 1.0, A, K, 0.0, up, N, 256 * MiB)
    assert st.n_kernels >= 2
    assert np.array_equal(np.tril(lo.view), np.triu(up.view).T)
    assert not np.triu(lo.view, 1).any() and not np.tril(up.view, -1).any()
    rows = np.array([0, 1, 127, 128, 4095, 4096, 4097, N - 1])
    Bt = np.empty((K, N)); Bt[...] = A.view.T
    ref, D = oracle.dgemm_sub(1.0, A.view, Bt, 0.0, None, rows=rows)
    for q, i in enumerate(rows):
        ok, worst = oracle.within_gate(lo.view[i, : i + 1], ref[q, : i + 1], D[q, : i + 1], RTOL)
        assert ok, (i, worst)
    for args, want in (((2, 0, N, K, 1.0, A, K, 0.0, lo, N), -2), ((0, 2, N, K, 1.0, A, K, 0.0, lo, N), -3),
                       ((0, 0, -1, K, 1.0, A, K, 0.0, lo, N), -4), ((0, 0, N, K, 1.0, None, K, 0.0, lo, N), -7),
                       ((0, 0, N, K, 1.0, A, K - 1, 0.0, lo, N), -8), ((0, 1, N, K, 1.0, A, N - 1, 0.0, lo, N), -8),
                       ((0, 0, N, K, 1.0, A, K, 0.0, None, N), -10), ((0, 0, N, K, 1.0, A, K, 0.0, lo, N - 1), -11)):
        with pytest.raises(H.HclError) as e:
            H.hclooc_dsyrk(None, *args, 256 * MiB)
        assert e.value.status == want, (args[:2], e.value.status)


@pytest.mark.parametrize("uplo,trans", [(0, 0), (1, 1)])
def test_dsyrk_on_device_resident_operands_runs_in_core(H, uplo, trans):
    """A and C in device memory: one masked launch on the caller's matrices, nothing staged; the other triangle untouched."""
    import torch
    N, K = 700, 260
    A = synthgen.fill(np.empty((K, N) if trans else (N, K)), 83, "A", "int")
    C0 = synthgen.fill(np.empty((N, N)), 83, "C", "int")
    ref = C0.copy()
    oracle.dsyrk(uplo, trans, 2.0, A, 0.5, ref)
    dA, dC = to_dev(A), to_dev(C0)
    st = H.hclooc_dsyrk(None, uplo, trans, N, K, 2.0, dA, A.shape[1], 0.5, dC, N, 0)
    assert st.n_kernels == 1 and st.plan.workspace_bytes == 0 and st.bytes_h2d == 0
    assert np.array_equal(dC.cpu().numpy(), ref)


@pytest.mark.parametrize("uplo", [0, 1])
@pytest.mark.parametrize("trans", [0, 1])
@pytest.mark.parametrize("N,K,alpha,beta,dist,budget", [
    (300, 200, 1.0, 0.5, "uniform", 1 * MiB),
    (517, 389, 2.0, -1.0, "int", 2 * MiB),
    (129, 33, -1.5, 0.0, "int", 1 * MiB),
    (1300, 260, 1.0, 1.0, "normal", 64 * MiB),
])
def test_dsyr2k_matches_oracle_and_leaves_the_other_triangle(H, uplo, trans, N, K, alpha, beta, dist, budget):
    ar, ac = (K, N) if trans else (N, K)
    A, B, C = H.HostMatrix(ar, ac, ac + 2), H.HostMatrix(ar, ac, ac + 4), H.HostMatrix(N, N, N + 2)
    for X in (A, B, C):
        X.array[...] = np.nan
    synthgen.fill(A.array, 84, "A", dist, cols=ac); synthgen.fill(B.array, 84, "B", dist, cols=ac); synthgen.fill(C.array, 84, "C", dist, cols=N)
    other = np.triu(np.ones((N, N), bool), 1) if uplo == 0 else np.tril(np.ones((N, N), bool), -1)
    if beta == 0.0:
        C.view[~other] = np.nan
    marker = C.view.copy()
    marker[other] = np.arange(int(other.sum())) + 0.25
    C.view[...] = marker
    ref = np.where(np.isnan(marker), 0.0, marker) if beta == 0.0 else marker.copy()
    D = oracle.dsyr2k(uplo, trans, alpha, A.view.copy(), B.view.copy(), beta, ref, want_denominator=True)
    st = H.hclooc_dsyr2k(None, uplo, trans, N, K, alpha, A, A.ld, B, B.ld, beta, C, C.ld, budget)
    assert st.n_kernels >= 2
    got = C.view.copy()
    assert np.array_equal(got[other], marker[other])
    gk, rk = got.copy(), ref.copy()
    gk[other] = 0.0; rk[other] = 0.0
    D[other] = 1.0
    check(gk, rk, D, exact=(dist == "int"))
    with pytest.raises(H.HclError) as e:
        H.hclooc_dsyr2k(None, uplo, trans, N, K, alpha, A, A.ld, None, B.ld, beta, C, C.ld, budget)
    assert e.value.status == -9


def test_dsyrk_and_dsyr2k_in_direct_mode(H):
    """Small symmetric updates under a small budget go through the direct mode too (tile kernel with the triangle mask on the
    host matrices, no device buffer); the other triangle keeps its bits."""
    N, K = 500, 300
    A = H.HostMatrix(N, K); B = H.HostMatrix(N, K); C = H.HostMatrix(N, N)
    synthgen.fill(A.array, 85, "A", "int"); synthgen.fill(B.array, 85, "B", "int"); synthgen.fill(C.array, 85, "C", "int")
    c0 = C.view.copy()
    ctx = H.hclooc_ctx_create(0)
    try:
        H.hclooc_ctx_set_direct(ctx, 1)
        ref = c0.copy()
        oracle.dsyrk(0, 0, 2.0, A.view, 0.5, ref)
        st = H.hclooc_dsyrk(ctx, 0, 0, N, K, 2.0, A, K, 0.5, C, N, 1 * MiB)
        assert st.plan.direct == 1 and st.plan.workspace_bytes == 0 and st.n_kernels == 1
        assert np.array_equal(C.view, ref)
        C.view[...] = c0
        ref = c0.copy()
        oracle.dsyr2k(1, 0, 1.0, A.view, B.view, -1.0, ref)
        st = H.hclooc_dsyr2k(ctx, 1, 0, N, K, 1.0, A, K, B, K, -1.0, C, N, 1 * MiB)
        assert st.plan.direct == 1 and st.n_kernels == 2
        assert np.array_equal(C.view, ref)
    finally:
        H.hclooc_ctx_destroy(ctx)


@pytest.mark.parametrize("transa,transb,tri", [(0, 0, 0), (1, 1, 0), (0, 1, 0), (0, 1, 1), (1, 0, 2)])
def test_two_b_buffers_prefetch_in_chunks_with_every_layout(H, monkeypatch, transa, transb, tri):
    """Plans with two B slice buffers prefetch the next slice in chunks between the steps of a column; for a transposed B the
    chunks are ranges of its n rows, and with the triangle mask a column has fewer live steps to hang them on.  Forced here
    (the planner picks two buffers only for large compute-bound problems), integers, bit-exact."""
    monkeypatch.setenv("HCLOOC_FORCE_BBUF", "2")
    monkeypatch.setenv("HCLOOC_FORCE_NB", "256")
    monkeypatch.setenv("HCLOOC_FORCE_MB", "128")
    N, K = 1100, 300
    M = N
    ctx = H.hclooc_ctx_create(0)
    try:
        if tri:
            A = H.HostMatrix(K, N) if transa else H.HostMatrix(N, K)
            C = H.HostMatrix(N, N)
            synthgen.fill(A.array, 86, "A", "int"); synthgen.fill(C.array, 86, "C", "int")
            ref = C.view.copy()
            oracle.dsyrk(tri - 1, transa, 1.0, A.view, 0.5, ref)
            st = H.hclooc_dsyrk(ctx, tri - 1, transa, N, K, 1.0, A, A.ld, 0.5, C, N, 64 * MiB)
        else:
            A, B, C = stored_inputs(H, transa, transb, M, N, K, 86, "int")
            opA, opB = np.empty((M, K)), np.empty((K, N))
            opA[...] = A.view.T if transa else A.view
            opB[...] = B.view.T if transb else B.view
            ref = C.view.copy()
            oracle.dgemm(1.0, opA, opB, 0.5, ref)
            st = H.hclooc_dgemm_t(ctx, transa, transb, M, N, K, 1.0, A, A.ld, B, B.ld, 0.5, C, C.ld, 64 * MiB)
        assert st.plan.n_bbuf == 2 and st.plan.w >= 4 and st.plan.h >= 8 and st.plan.direct == 0
        assert np.array_equal(C.view, ref)
    finally:
        H.hclooc_ctx_destroy(ctx)


def test_graph_replay_with_transposed_operands_and_triangle_mask(H):
    """The CUDA-graph replay of a repeated short call carries the operand layouts and the triangle mask: a transposed DGEMM
    and a DSYRK, four identical calls each (ordinary, capture + launch, replay, replay), alternating never reuses a graph."""
    N, K = 512, 384
    A, B, C = stored_inputs(H, 1, 1, N, N, K, 87, "int")
    C0 = C.view.copy()
    opA, opB = np.empty((N, K)), np.empty((K, N))
    opA[...] = A.view.T; opB[...] = B.view.T
    ref_t = C0.copy(); oracle.dgemm(1.0, opA, opB, 0.5, ref_t)
    ref_s = C0.copy(); oracle.dsyrk(0, 1, 1.0, A.view, 0.5, ref_s)                 # A is stored K x N: trans = T
    ctx = H.hclooc_ctx_create(0)
    try:
        for rep in range(4):
            C.view[...] = C0
            st = H.hclooc_dgemm_t(ctx, 1, 1, N, N, K, 1.0, A, A.ld, B, B.ld, 0.5, C, C.ld, 1 * MiB)
            assert st.plan.n_steps > 4 and np.array_equal(C.view, ref_t)
        for rep in range(4):
            C.view[...] = C0
            st = H.hclooc_dsyrk(ctx, 0, 1, N, K, 1.0, A, A.ld, 0.5, C, C.ld, 1 * MiB)
            assert np.array_equal(C.view, ref_s)
        for rep in range(3):
            C.view[...] = C0
            H.hclooc_dgemm_t(ctx, 1, 1, N, N, K, 1.0, A, A.ld, B, B.ld, 0.5, C, C.ld, 1 * MiB)
            assert np.array_equal(C.view, ref_t)
            C.view[...] = C0
            H.hclooc_dsyrk(ctx, 0, 1, N, K, 1.0, A, A.ld, 0.5, C, C.ld, 1 * MiB)
            assert np.array_equal(C.view, ref_s)
    finally:
        H.hclooc_ctx_destroy(ctx)


def test_config2_full_size_transposed_sampled_rows_and_columns(H):
    """BASELINE configs[1] shape with both operands transposed (bench.py --trans TT): 8192^3 under 256 MiB, integer variant:
    complete rows and columns on both sides of the plan's slab boundaries against the oracle, and exact whole-matrix checksums."""
    M = N = K = 8192
    A, B, C = stored_inputs(H, 1, 1, M, N, K, synthgen.BASE_SEED + 2, "int")
    opA, opB = np.empty((M, K)), np.empty((K, N))
    opA[...] = A.view.T; opB[...] = B.view.T
    plan = H.hclooc_plan_trans(M, N, K, 1, 0, 256 * MiB, 0, 1, 1)
    rng = np.random.default_rng(6)
    rows = {0, M - 1} | {int(x) for x in rng.integers(0, M, 4)}
    cols = {0, N - 1} | {int(x) for x in rng.integers(0, N, 4)}
    for i in (1, plan.h // 2, plan.h - 1):
        rows |= {i * plan.mb - 1, i * plan.mb}
    for j in range(1, plan.w):
        cols |= {j * plan.nb - 1, j * plan.nb}
    rows, cols = np.array(sorted(rows)), np.array(sorted(cols))
    C0 = C.view.copy()
    ref_r, _ = oracle.dgemm_sub(1.0, opA, opB, 1.0, C0, rows=rows)
    ref_c, _ = oracle.dgemm_sub(1.0, opA, opB, 1.0, C0, cols=cols)
    st = H.hclooc_dgemm_t(None, 1, 1, M, N, K, 1.0, A, A.ld, B, B.ld, 1.0, C, C.ld, 256 * MiB)
    assert st.plan.trans == 3 and st.plan.workspace_bytes <= 256 * MiB and st.bytes_h2d == st.plan.bytes_h2d
    assert (st.plan.mb, st.plan.nb) == (plan.mb, plan.nb)
    assert np.array_equal(C.view[rows], ref_r) and np.array_equal(C.view[:, cols], ref_c)
    x = synthgen.fill_numpy(N, 1, 77, "A", "int"); y = synthgen.fill_numpy(1, M, 77, "B", "int")
    assert np.array_equal(C.view @ x, opA @ (opB @ x) + C0 @ x)
    assert np.array_equal(y @ C.view, (y @ opA) @ opB + y @ C0)
    for X in (A, B, C):
        X.free()


def test_dsyrk_large_exact_checksums(H):
    """DSYRK at a size with many blocks and several B slices (12288^2 x 2048 under 512 MiB), integer inputs: the lower triangle
    mirrored to a full symmetric matrix satisfies S x = alpha*A*(A^T x) + beta*S0 x exactly for an integer x (any wrong element
    changes a row sum), the strict upper triangle keeps its bits, sampled rows equal the oracle."""
    N, K = 12288, 2048
    A, C = H.HostMatrix(N, K), H.HostMatrix(N, N)
    synthgen.fill(A.array, 88, "A", "int"); synthgen.fill(C.array, 88, "C", "int")
    upper0 = np.triu(C.view, 1).copy()
    low0 = np.tril(C.view)
    S0 = low0 + np.tril(C.view, -1).T
    x = synthgen.fill_numpy(N, 1, 78, "A", "int")[:, 0]
    want = 2.0 * (A.view @ (A.view.T @ x)) + 0.5 * (S0 @ x)
    rows = np.array([0, 127, 128, 4095, 4096, 8191, 8192, N - 1])
    At = np.empty((K, N)); At[...] = A.view.T
    ref_rows, _ = oracle.dgemm_sub(2.0, A.view, At, 0.5, C.view.copy(), rows=rows)
    st = H.hclooc_dsyrk(None, H.HCL_UPLO_LOWER, H.HCL_OP_N, N, K, 2.0, A, K, 0.5, C, N, 512 * MiB)
    assert st.plan.tri == 1 and st.plan.w >= 2 and st.bytes_d2h < 8 * N * N * 0.8          # blocks above the diagonal never moved
    assert np.array_equal(np.triu(C.view, 1), upper0)
    S = np.tril(C.view) + np.tril(C.view, -1).T
    assert np.array_equal(S @ x, want)
    for q, i in enumerate(rows):
        assert np.array_equal(C.view[i, : i + 1], ref_rows[q, : i + 1]), i
    for X in (A, C):
        X.free()
