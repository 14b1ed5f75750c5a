"""GPU parity for the LU factorization with partial pivoting built on the out-of-core DGEMM:
hclooc_dgetrf (host-resident matrix under a device budget) and hclDgetrf (device matrix), against oracle.dgetrf.

Bars (G27).  Matrices built from known factors whose elimination is exact in FP64 (tests/_lu_inputs.py: L in
{0, +-1/2}, U integer, unique pivots) -> ipiv, L and U bit for bit, in any blocking.  Otherwise: the interchanges are valid
(j <= ipiv[j] < M), |l_ij| <= 1, and the backward bound every order of the operations satisfies, |P A - L U| <= gamma_n |L||U|
(oracle.dgetrf_gate, residual in long double with the CANDIDATE's own interchanges); and where the oracle is affordable, the
same pivot sequence as the oracle (both take the first maximum of FP64 values; the seeded uniform inputs have no near-ties) and
factors within 1e-9 of the largest entry of U.
"""
import numpy as np
import pytest

import oracle
import synthgen
from _lu_inputs import exact_lu_case

pytestmark = pytest.mark.gpu
MiB = 1 << 20


@pytest.fixture(scope="module")
def H():
    import paper_1808_05056_b200 as H
    import torch
    assert torch.cuda.is_available()
    torch.cuda.init()
    return H


def host_matrix(H, values, pad):
    M, N = values.shape
    A = H.HostMatrix(M, N, N + pad)
    A.array[...] = np.nan
    A.view[...] = values
    return A


def check_float(M, N, A0, got, ipiv, info, full_oracle):
    n = min(M, N)
    assert info == 0
    assert ((ipiv >= np.arange(n)) & (ipiv < M)).all()
    assert not np.isnan(got).any()
    assert (np.abs(np.tril(got[:, :n], -1)) <= 1.0).all()                        # partial pivoting
    gate = oracle.dgetrf_gate(n)
    if M * N <= 1200 * 1200:
        res, den = oracle.dgetrf_residual(A0, got, ipiv)
    else:
        rng = np.random.default_rng(5)
        rows = np.unique(np.concatenate([[0, 1, n - 1, M - 1], rng.integers(0, M, 40)]))
        cols = np.unique(np.concatenate([[0, 1, n - 1, N - 1], rng.integers(0, N, 40)]))
        res, den = oracle.dgetrf_residual(A0, got, ipiv, rows, cols)
    worst = float(np.max(res / np.maximum(den, 1e-300)))
    assert (res <= gate * den).all(), f"backward residual {worst:.3e} of |L||U| exceeds gamma_n = {gate:.3e}"
    if full_oracle:
        ref = A0.copy()
        ipiv_ref, info_ref = oracle.dgetrf(ref)
        assert info_ref == 0
        assert np.array_equal(ipiv, ipiv_ref), f"first differing interchange at step {int(np.argmax(ipiv != ipiv_ref))}"
        scale = np.abs(np.triu(ref[:n])).max()
        assert np.abs(got - ref).max() <= 1e-9 * scale


CASES = [
    (1, 1, "uniform", 0, 1 * MiB),
    (5, 3, "uniform", 1, 1 * MiB),
    (3, 5, "exact", 0, 1 * MiB),
    (31, 31, "exact", 1, 1 * MiB),              # one call of the panel kernel, fewer than 32 columns
    (77, 77, "exact", 1, 1 * MiB),              # recursion over 32-column panels with a ragged last one
    (200, 64, "uniform", 0, 1 * MiB),           # tall: two CTAs in the panel kernel
    (128, 128, "uniform", 0, 2 * MiB),
    (300, 300, "uniform", 2, 8 * MiB),
    (1000, 1000, "exact", 0, 32 * MiB),         # one resident panel: the device recursion alone, exact
    (1000, 1000, "uniform", 3, 3 * MiB),        # several panels: interchanges, DTRSM and out-of-core updates per block column
    (1500, 1100, "exact", 1, 8 * MiB),          # tall
    (1100, 1500, "exact", 0, 8 * MiB),          # wide: the last block columns hold no pivots
    (1100, 1500, "uniform", 0, 8 * MiB),
    (2049, 2049, "uniform", 0, 24 * MiB),       # odd size, ragged last panel
    (2500, 2500, "exact", 0, 32 * MiB),
]


@pytest.mark.parametrize("M,N,dist,pad,budget", CASES)
def test_dgetrf_matches_oracle(H, M, N, dist, pad, budget):
    if dist == "exact":
        vals, F_want, ipiv_want = exact_lu_case(M, N, 1000 * M + N)
    else:
        vals = synthgen.fill_numpy(M, N, 17, "A", "uniform")
    A = host_matrix(H, vals, pad)
    A0 = A.view.copy()
    ipiv, info, st = H.hclooc_dgetrf(None, M, N, A, A.ld, budget)
    got = A.view.copy()
    assert st.plan.workspace_bytes <= budget
    NB, reserved = H.hclooc_dgetrf_plan(M, N, budget)
    assert st.plan.nb == NB and st.plan.n_steps == -(-N // NB)
    assert np.isnan(A.array[:, N:]).all()                                        # padding untouched
    if dist == "exact":
        assert info == 0
        assert np.array_equal(ipiv, ipiv_want), f"first differing interchange at step {int(np.argmax(ipiv != ipiv_want))}"
        bad = got != F_want
        assert not bad.any(), f"{np.count_nonzero(bad)} elements differ, first at {tuple(np.argwhere(bad)[0])}"
        ref = A0.copy()                                                          # and the oracle says the same of this matrix
        ipiv_ref, info_ref = oracle.dgetrf(ref)
        assert info_ref == 0 and np.array_equal(ipiv_ref, ipiv_want) and np.array_equal(ref, F_want)
    else:
        check_float(M, N, A0, got, ipiv, info, full_oracle=True)


@pytest.mark.parametrize("M,N,dist", [(700, 700, "exact"), (3000, 1800, "exact"), (1800, 3000, "uniform"), (3000, 3000, "uniform")])
def test_hclDgetrf_on_device_memory(H, M, N, dist):
    import torch
    if dist == "exact":
        vals, F_want, ipiv_want = exact_lu_case(M, N, 3 * M + N)
    else:
        vals = synthgen.fill_numpy(M, N, 23, "A", "uniform")
    ld = N + (N & 1) + 2
    dA = torch.full((M, ld), float("nan"), dtype=torch.float64, device="cuda")
    dA[:, :N] = torch.from_numpy(vals).cuda()
    s = torch.cuda.Stream()
    ipiv, info = H.hclDgetrf(M, N, dA, ld, s)
    torch.cuda.synchronize()
    got = dA[:, :N].cpu().numpy()
    assert torch.isnan(dA[:, N:]).all()
    if dist == "exact":
        assert info == 0 and np.array_equal(ipiv, ipiv_want) and np.array_equal(got, F_want)
    else:
        check_float(M, N, vals, got, ipiv, info, full_oracle=M * N <= 2100 * 2100)


def test_dgetrf_zero_pivot_is_reported_and_the_factorization_completes(H):
    M = N = 600
    vals = synthgen.fill_numpy(M, N, 29, "A", "uniform")
    vals[:, 345] = 0.0                                                            # a zero column stays exactly zero: 0 - l * 0
    A = host_matrix(H, vals, 0)
    A0 = A.view.copy()
    ref = A0.copy()
    ipiv_ref, info_ref = oracle.dgetrf(ref)
    ipiv, info, st = H.hclooc_dgetrf(None, M, N, A, A.ld, 2 * MiB)
    assert info_ref == 346 and info == 346                                        # u_345,345 = 0 exactly: a zero column stays zero
    got = A.view.copy()
    assert got[345, 345] == 0.0 and (got[346:, 345] == 0.0).all()
    res, den = oracle.dgetrf_residual(A0, got, ipiv)
    assert (res <= oracle.dgetrf_gate(N) * den).all()
    Z = H.HostMatrix(40, 40)
    Z.view[...] = 0.0
    ipiv, info, st = H.hclooc_dgetrf(None, 40, 40, Z, Z.ld, 1 * MiB)
    assert info == 1 and np.array_equal(ipiv, np.arange(40)) and not Z.view.any()


def test_dgetrf_argument_errors_and_empty_shapes(H):
    A = H.HostMatrix(8, 8)
    A.view[...] = np.eye(8)
    for (M, N, lda, code) in ((-1, 8, 8, -2), (8, -1, 8, -3), (8, 8, 7, -5)):
        with pytest.raises(H.HclError) as e:
            H.hclooc_dgetrf(None, M, N, A, lda, 1 * MiB)
        assert e.value.status == code
    ipiv, info, st = H.hclooc_dgetrf(None, 0, 8, A, 8, 1 * MiB)
    assert info == 0 and ipiv.size == 0
    ipiv, info, st = H.hclooc_dgetrf(None, 8, 8, A, 8, 1 * MiB)
    assert info == 0 and np.array_equal(ipiv, np.arange(8)) and np.array_equal(A.view, np.eye(8))
    with pytest.raises(H.HclError) as e:
        H.hclooc_dgetrf(None, 100000, 64, A, 64, 1 * MiB)                        # two 32-column panels of 100000 rows: 51 MB
    assert e.value.status == 1                                                   # HCLOOC_ERR_BUDGET


@pytest.mark.parametrize("dist", ["exact", "uniform"])
def test_dgetrf_large(H, dist):
    """8192^2 under 256 MiB: panels of 1024 columns (8 of them), every out-of-core update a pipeline call with K = 1024."""
    M = N = 8192
    if dist == "exact":
        vals, F_want, ipiv_want = exact_lu_case(M, N, 99)
    else:
        vals = synthgen.fill_numpy(M, N, 31, "A", "uniform")
    A = host_matrix(H, vals, 0)
    A0 = A.view.copy()
    ipiv, info, st = H.hclooc_dgetrf(None, M, N, A, A.ld, 256 * MiB)
    got = A.view.copy()
    assert st.plan.workspace_bytes <= 256 * MiB and st.plan.n_steps > 2
    if dist == "exact":
        assert info == 0 and np.array_equal(ipiv, ipiv_want)
        assert np.array_equal(got, F_want), f"{np.count_nonzero(got != F_want)} elements differ"
    else:
        check_float(M, N, A0, got, ipiv, info, full_oracle=False)


@pytest.mark.parametrize("M,N,dist", [(40000, 200, "exact"), (40000, 200, "uniform"), (70000, 96, "exact"), (70000, 96, "uniform"),
                                      (120000, 64, "exact"), (120000, 40, "uniform")])
def test_dgetrf_tall_panels_take_narrower_leaves(H, M, N, dist):
    """The panel kernel keeps a CTA's slab of rows in shared memory: 128-column leaves up to ~32000 rows, 64 up to ~63000, 32 up to
    ~112000, 16 beyond (getrf_panel_shape).  Every width against the oracle on one resident panel."""
    if dist == "exact":
        vals, F_want, ipiv_want = exact_lu_case(M, N, M + N)
    else:
        vals = synthgen.fill_numpy(M, N, 37, "A", "uniform")
    A = host_matrix(H, vals, 0)
    A0 = A.view.copy()
    ipiv, info, st = H.hclooc_dgetrf(None, M, N, A, A.ld, 512 * MiB)
    got = A.view.copy()
    assert st.plan.n_steps == 1 and info == 0
    ref = A0.copy()
    ipiv_ref, info_ref = oracle.dgetrf(ref)
    assert info_ref == 0 and np.array_equal(ipiv, ipiv_ref), f"first differing interchange at step {int(np.argmax(ipiv != ipiv_ref))}"
    if dist == "exact":
        assert np.array_equal(ipiv, ipiv_want) and np.array_equal(got, F_want) and np.array_equal(ref, F_want)
    else:
        rng = np.random.default_rng(9)
        rows = np.unique(np.concatenate([[0, 1, N - 1, N, M - 1], rng.integers(0, M, 200)]))
        res, den = oracle.dgetrf_residual(A0, got, ipiv, rows, None)
        assert (res <= oracle.dgetrf_gate(N) * den).all()
        assert (np.abs(np.tril(got[:, :N], -1)) <= 1.0).all()
        assert np.abs(got - ref).max() <= 1e-9 * np.abs(np.triu(ref[:N])).max()


@pytest.mark.parametrize("panels", [2, 3])
def test_dgetrf_two_and_three_resident_panels(H, panels, monkeypatch):
    """HCLOOC_GETRF_PANELS caps the resident panels: with two, the next panel's upload follows the freshest update range by range
    into the buffer that update is still reading; with three it goes a whole iteration ahead.  Same bits either way."""
    monkeypatch.setenv("HCLOOC_GETRF_PANELS", str(panels))
    M, N = 2300, 2100
    vals, F_want, ipiv_want = exact_lu_case(M, N, 4242)
    ctx = H.hclooc_ctx_create()
    try:
        for seed in (0, 5):
            A = host_matrix(H, vals, 2)
            H.hclooc_ctx_set_debug(ctx, seed, 1 if seed else 0)
            ipiv, info, st = H.hclooc_dgetrf(ctx, M, N, A, A.ld, 24 * MiB)
            assert st.plan.n_sets == panels and st.plan.n_steps >= 4
            assert info == 0 and np.array_equal(ipiv, ipiv_want) and np.array_equal(A.view, F_want)
    finally:
        H.hclooc_ctx_set_debug(ctx, 0, 0)
        H.hclooc_ctx_destroy(ctx)


def test_dgetrf_under_the_debug_shaker(H):
    """Random delays in front of every copy and kernel, NaN in buffers the schedule declares free: an exact case must stay exact."""
    M, N = 1300, 1200
    vals, F_want, ipiv_want = exact_lu_case(M, N, 77)
    ctx = H.hclooc_ctx_create()
    try:
        for seed in (1, 2, 3):
            A = host_matrix(H, vals, 0)
            H.hclooc_ctx_set_debug(ctx, seed, 1)
            ipiv, info, st = H.hclooc_dgetrf(ctx, M, N, A, A.ld, 6 * MiB)
            assert info == 0 and np.array_equal(ipiv, ipiv_want) and np.array_equal(A.view, F_want)
    finally:
        H.hclooc_ctx_set_debug(ctx, 0, 0)
        H.hclooc_ctx_destroy(ctx)
