"""Pins for the CPU oracle (oracle/dgemm_oracle.c) against things other than itself.

What fixes the answer here is the definition C = alpha*A*B + beta*C and
mathematics: brute force in pure Python, exact int64 arithmetic, closed forms, exactly rounded sums
(math.fsum), a library matmul within the gate, and the paper's printed partition example
(tests/golden/paper_partition_example.txt).  A dropped k term, a swapped index,
a transposed operand, a fused multiply-add or a wrong epilogue sign fails at least one of them.
"""
import itertools
import math
import os

import numpy as np
import pytest

import oracle
import synthgen

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def padded(rng, rows, cols, pad, fill="uniform"):
    """rows x cols view into a wider NaN-padded buffer (leading dimension cols + pad)."""
    buf = np.full((max(rows, 1), cols + pad), np.nan)
    v = buf[:rows, :cols]
    if fill == "uniform":
        v[...] = rng.uniform(-1, 1, (rows, cols))
    elif fill == "int":
        v[...] = rng.integers(-4, 5, (rows, cols)).astype(np.float64)
    return buf, v


def naive_ijk(alpha, A, B, beta, C0):
    """The definition in pure Python floats (IEEE double, no fma): i-j-k, in-order k."""
    M, N = C0.shape
    K = A.shape[1]
    out = np.empty((M, N))
    for i in range(M):
        for j in range(N):
            acc = 0.0
            if alpha != 0.0:
                for k in range(K):
                    acc = acc + float(A[i, k]) * float(B[k, j])
            if beta == 0.0:
                out[i, j] = alpha * acc
            else:
                out[i, j] = alpha * acc + beta * float(C0[i, j])
    return out


def bits(x):
    return np.ascontiguousarray(x).view(np.uint64)


# ---------------------------------------------------------------- brute force, bit-identical
def test_brute_force_all_tiny_shapes_bit_identical():
    rng = np.random.default_rng(1)
    for M, N, K in itertools.product(range(0, 6), range(0, 6), [0, 1, 2, 3, 5, 9]):
        pad = int(rng.integers(0, 4))
        _, A = padded(rng, M, K, pad)
        _, B = padded(rng, K, N, pad + 1)
        cbuf, C = padded(rng, M, N, pad + 2)
        alpha, beta = float(rng.uniform(-2, 2)), float(rng.choice([0.0, 1.0, -0.75, 0.5]))
        want = naive_ijk(alpha, A, B, beta, C.copy())
        oracle.dgemm(alpha, A, B, beta, C)
        assert np.array_equal(bits(C), bits(want)), (M, N, K)
        if M:
            assert np.isnan(cbuf[:M, N:]).all()          # padding of C untouched


def test_brute_force_spans_blocks_and_ragged_tail():
    # sizes beyond the oracle's 32-row / 128-k blocking with ragged tails, still bit-identical
    rng = np.random.default_rng(2)
    M, N, K = 37, 11, 263
    _, A = padded(rng, M, K, 3)
    _, B = padded(rng, K, N, 5)
    _, C = padded(rng, M, N, 2)
    want = naive_ijk(-1.25, A, B, 0.5, C.copy())
    oracle.dgemm(-1.25, A, B, 0.5, C)
    assert np.array_equal(bits(C), bits(want))


def test_no_fused_multiply_add():
    # (1+e)*(1-e) = 1 - e^2 rounds to 1.0 as a separate product, so acc = 1.0 - 1.0 = 0 exactly;
    # an fma would keep -e^2.  Catches -ffp-contract / FMA code generation in the oracle.
    e = 2.0 ** -30
    A = np.array([[1.0 + e, 1.0]])
    B = np.array([[1.0 - e], [-1.0]])
    C = np.zeros((1, 1))
    oracle.dgemm(1.0, A, B, 0.0, C)
    assert C[0, 0] == 0.0


# ---------------------------------------------------------------- exact integer arithmetic
@pytest.mark.parametrize("M,N,K,alpha,beta", [(33, 47, 129, 1.0, 0.5), (64, 64, 512, 2.0, -1.0),
                                              (5, 130, 1000, -3.0, 1.0), (70, 3, 77, 1.0, 0.0)])
def test_integer_inputs_equal_int64_reference(M, N, K, alpha, beta):
    rng = np.random.default_rng(M * 1000 + N)
    _, A = padded(rng, M, K, 1, "int")
    _, B = padded(rng, K, N, 2, "int")
    _, C = padded(rng, M, N, 3, "int")
    Ai, Bi, Ci = A.astype(np.int64), B.astype(np.int64), C.astype(np.int64)
    # everything in exact integers scaled by 2 (beta may be a half-integer)
    want2 = int(round(alpha * 2)) * (Ai @ Bi) + int(round(beta * 2)) * Ci
    assert np.abs(want2).max() < 2 ** 52
    oracle.dgemm(alpha, A, B, beta, C)
    assert np.array_equal(C * 2.0, want2.astype(np.float64))


def test_generator_integer_variant_exact():
    M = N = K = 96
    A = synthgen.fill(np.empty((M, K)), 7, "A", "int")
    B = synthgen.fill(np.empty((K, N)), 7, "B", "int")
    C = synthgen.fill(np.empty((M, N)), 7, "C", "int")
    assert A.min() >= -4 and A.max() <= 4 and not np.signbit(A[A == 0]).any()
    want2 = 2 * (A.astype(np.int64) @ B.astype(np.int64)) + C.astype(np.int64)
    oracle.dgemm(1.0, A, B, 0.5, C)
    assert np.array_equal(C * 2.0, want2.astype(np.float64))


# ---------------------------------------------------------------- closed forms
def test_identity_A_gives_alpha_B_plus_beta_C():
    rng = np.random.default_rng(3)
    K = N = 41
    B = rng.uniform(-1, 1, (K, N))
    C0 = rng.uniform(-1, 1, (K, N))
    C = C0.copy()
    oracle.dgemm(1.5, np.eye(K), B, -0.25, C)
    assert np.array_equal(C, 1.5 * B + (-0.25) * C0)     # adding exact zeros changes nothing


def test_permutation_matrices_permute_rows_and_columns():
    rng = np.random.default_rng(4)
    n = 29
    p = rng.permutation(n)
    P = np.zeros((n, n)); P[np.arange(n), p] = 1.0        # (P @ X)[i] = X[p[i]]
    X = rng.uniform(-1, 1, (n, 17))
    C = np.zeros((n, 17))
    oracle.dgemm(1.0, P, X, 0.0, C)
    assert np.array_equal(C, X[p])
    Y = rng.uniform(-1, 1, (13, n))
    C = np.zeros((13, n))
    oracle.dgemm(1.0, Y, P, 0.0, C)                       # (Y @ P)[:, p[i]] = Y[:, i]
    want = np.zeros((13, n)); want[:, p] = Y
    assert np.array_equal(C, want)


def test_rank_one_outer_product_exact_rounding_sequence():
    rng = np.random.default_rng(5)
    u = rng.uniform(-1, 1, (23, 1)); v = rng.uniform(-1, 1, (1, 31))
    C0 = rng.uniform(-1, 1, (23, 31)); C = C0.copy()
    oracle.dgemm(0.75, u, v, 1.25, C)
    want = 0.75 * (0.0 + u * v) + 1.25 * C0               # same three roundings per element
    assert np.array_equal(bits(C), bits(want))


def test_all_ones_and_index_products():
    M, N, K = 19, 21, 300
    C = np.full((M, N), 2.0)
    oracle.dgemm(3.0, np.ones((M, K)), np.ones((K, N)), 0.5, C)
    assert np.array_equal(C, np.full((M, N), 3.0 * K + 1.0))
    A = np.repeat(np.arange(1.0, M + 1)[:, None], K, axis=1)
    B = np.repeat(np.arange(1.0, N + 1)[None, :], K, axis=0)
    C = np.zeros((M, N))
    oracle.dgemm(1.0, A, B, 0.0, C)
    assert np.array_equal(C, np.outer(np.arange(1.0, M + 1), np.arange(1.0, N + 1)) * K)


def test_non_symmetric_shape_catches_transposed_operands():
    # A_ik = 10*i + k, B_kj = k - 3*j : sum_k has a closed form that is not symmetric in (i, j)
    M, N, K = 7, 5, 9
    i = np.arange(M)[:, None]; k = np.arange(K)[None, :]
    A = (10.0 * i + k)
    B = (np.arange(K)[:, None] - 3.0 * np.arange(N)[None, :])
    C = np.zeros((M, N))
    oracle.dgemm(1.0, A, B, 0.0, C)
    kk = np.arange(K)
    want = np.array([[float(sum((10 * ii + q) * (q - 3 * jj) for q in kk)) for jj in range(N)] for ii in range(M)])
    assert np.array_equal(C, want)


def test_alpha_zero_does_not_read_A_B_and_beta_zero_does_not_read_C():
    rng = np.random.default_rng(6)
    M, N, K = 9, 8, 7
    nanA, nanB = np.full((M, K), np.nan), np.full((K, N), np.nan)
    C0 = rng.uniform(-1, 1, (M, N)); C = C0.copy()
    oracle.dgemm(0.0, nanA, nanB, -2.0, C)
    assert np.array_equal(C, -2.0 * C0)
    A = rng.uniform(-1, 1, (M, K)); B = rng.uniform(-1, 1, (K, N))
    C = np.full((M, N), np.nan)
    oracle.dgemm(1.0, A, B, 0.0, C)
    assert np.isfinite(C).all() and np.array_equal(bits(C), bits(naive_ijk(1.0, A, B, 0.0, np.zeros((M, N)))))
    C = np.full((M, N), np.nan)
    oracle.dgemm(0.0, nanA, nanB, 0.0, C)
    assert np.array_equal(bits(C), bits(np.zeros((M, N))))        # +0 everywhere, sign included
    C = C0.copy()
    oracle.dgemm(1.0, np.empty((M, 0)), np.empty((0, N)), 0.5, C)  # K == 0
    assert np.array_equal(C, 0.5 * C0)


# ---------------------------------------------------------------- error bound vs exactly rounded sums
@pytest.mark.parametrize("K,dist", [(512, "uniform"), (4096, "uniform"), (2048, "normal")])
def test_error_against_exact_sum_is_far_below_gate(K, dist):
    M, N = 6, 5
    A = synthgen.fill(np.empty((M, K)), 11, "A", dist)
    B = synthgen.fill(np.empty((K, N)), 11, "B", dist)
    C0 = synthgen.fill(np.empty((M, N)), 11, "C", dist)
    alpha, beta = 1.0, 0.5        # powers of two: the epilogue scaling is exact, so fsum is THE answer
    C = C0.copy()
    D = oracle.dgemm(alpha, A, B, beta, C, want_denominator=True)
    from fractions import Fraction
    for i in range(M):
        for j in range(N):
            exact = sum((Fraction(float(A[i, k])) * Fraction(float(B[k, j])) for k in range(K)), Fraction(0))
            exact = alpha * exact + Fraction(beta) * Fraction(float(C0[i, j]))
            dexact = sum((abs(Fraction(float(A[i, k])) * Fraction(float(B[k, j]))) for k in range(K)), Fraction(0))
            dexact = dexact + Fraction(beta) * abs(Fraction(float(C0[i, j])))
            err = abs(Fraction(float(C[i, j])) - exact)
            u = Fraction(1, 2 ** 53)
            assert err <= (K + 2) * u * dexact * Fraction(101, 100)      # classical gamma_K bound
            assert float(err) <= 2e-15 * float(dexact)                   # ~50x below the 1e-13 gate
            assert abs(float(D[i, j]) - float(dexact)) <= 1e-12 * float(dexact)   # pins D itself


def test_library_matmul_agrees_within_gate():
    M, N, K = 150, 170, 700
    A = synthgen.fill(np.empty((M, K)), 12, "A", "uniform")
    B = synthgen.fill(np.empty((K, N)), 12, "B", "uniform")
    C0 = synthgen.fill(np.empty((M, N)), 12, "C", "uniform")
    C = C0.copy()
    D = oracle.dgemm(2.0, A, B, -1.0, C, want_denominator=True)
    ok, worst = oracle.within_gate(2.0 * (A @ B) - C0, C, D)
    assert ok and worst < 1e-14
    # the denominator is what it says
    assert np.allclose(D, 2.0 * (np.abs(A) @ np.abs(B)) + np.abs(C0), rtol=1e-12, atol=0)
    # and the gate is sharp enough to see one dropped k term
    Cbad = 2.0 * (A[:, :-1] @ B[:-1]) - C0
    ok_bad, _ = oracle.within_gate(Cbad, C, D)
    assert not ok_bad


# ---------------------------------------------------------------- sampled form == full form
def test_sub_matches_full_bit_for_bit():
    M, N, K = 45, 52, 301
    rng = np.random.default_rng(8)
    _, A = padded(rng, M, K, 2); _, B = padded(rng, K, N, 1); _, C0 = padded(rng, M, N, 4)
    C = C0.copy()
    D = oracle.dgemm(1.0, A, B, 0.5, C, want_denominator=True)
    rows = np.array([0, 44, 31, 32, 7]); cols = np.array([51, 0, 13])
    s, d = oracle.dgemm_sub(1.0, A, B, 0.5, C0, rows=rows, cols=None)
    assert np.array_equal(bits(s), bits(C[rows])) and np.array_equal(bits(d), bits(D[rows]))
    s, d = oracle.dgemm_sub(1.0, A, B, 0.5, C0, rows=None, cols=cols)
    assert np.array_equal(bits(s), bits(C[:, cols])) and np.array_equal(bits(d), bits(D[:, cols]))
    s, d = oracle.dgemm_sub(1.0, A, B, 0.5, C0, rows=rows, cols=cols)
    assert np.array_equal(bits(s), bits(C[np.ix_(rows, cols)]))
    s, _ = oracle.dgemm_sub(1.0, A, B, 0.0, None, rows=rows, cols=cols)      # beta == 0: C0 not needed
    assert np.array_equal(bits(s), bits(naive_ijk(1.0, A, B, 0.0, np.zeros((M, N)))[np.ix_(rows, cols)]))


# ---------------------------------------------------------------- the paper's partition example
def test_paper_partition_example_golden():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "paper_partition_example.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 1
    M, N, K, S, total, h, w, blocks, steps = map(int, rows[0])
    assert M * K + K * N + M * N == total and total > S             # "80 exceeds 44"
    assert oracle.partition(M, N, K, S) == (h, w)                   # Figure 3
    assert h * w == blocks == steps                                  # "w x h main steps"
    # the reading is discriminating: both rival readings of PAPER.md:289 contradict Figure 3
    feas = [(hh, ww) for hh in (1, 2, 4) for ww in (1, 2, 4)
            if K * (N // ww) + 2 * (M // hh) * K + 2 * (M // hh) * (N // ww) <= S]
    assert sorted(feas) == [(2, 4), (4, 2), (4, 4)]
    assert oracle.partition(M, N, K, 19) is None                     # (4,4) needs 8+16+2 = 26 > 19
    assert oracle.partition(M, N, K, 80 * 2) == (1, 1)               # everything fits: in-core


# ---------------------------------------------------------------- generator twins agree
@pytest.mark.parametrize("dist", ["uniform", "int", "normal"])
def test_generator_c_and_numpy_twins_agree(dist):
    a = np.full((9, 20), np.nan)
    synthgen.fill(a, 99, "C", dist, cols=17, row0=5, col0=3, logical_cols=1000)
    b = synthgen.fill_numpy(9, 17, 99, "C", dist, row0=5, col0=3, logical_cols=1000)
    if dist == "normal":
        assert np.allclose(a[:, :17], b, rtol=1e-14, atol=1e-15)      # libm vs numpy log/cos: last ulps
    else:
        assert np.array_equal(a[:, :17], b)
    assert np.isnan(a[:, 17:]).all()
    # a sub-block regenerates the same values as the whole
    whole = synthgen.fill(np.empty((14, 1000)), 99, "C", dist)
    assert np.array_equal(a[:, :17], whole[5:14, 3:20])
    if dist == "uniform":
        assert whole.min() >= -1.0 and whole.max() < 1.0 and abs(whole.mean()) < 0.02
    if dist == "normal":
        assert abs(whole.mean()) < 0.03 and abs(whole.std() - 1.0) < 0.03


# ------------------------------------------------------------------ dsyrk (the definition restricted to a triangle)
@pytest.mark.parametrize("uplo", [0, 1])
@pytest.mark.parametrize("trans", [0, 1])
def test_dsyrk_brute_force_and_untouched_triangle(uplo, trans):
    """Pure-Python loops over the referenced triangle in the order of the definition (in-order sum of separately rounded
    products, then alpha*acc + beta*c): bit-identical; the other triangle keeps its bits (NaN there stays NaN and is never
    computed with)."""
    rng = np.random.default_rng(7 + 2 * uplo + trans)
    for N, K in ((1, 1), (4, 3), (5, 9), (7, 2), (6, 0)):
        A = rng.uniform(-1, 1, (K, N) if trans else (N, K))
        C0 = rng.uniform(-1, 1, (N, N))
        other = np.triu(np.ones((N, N), bool), 1) if uplo == 0 else np.tril(np.ones((N, N), bool), -1)
        C0[other] = np.nan
        C = C0.copy()
        oracle.dsyrk(uplo, trans, 1.5, A, -0.5, C)
        for i in range(N):
            for j in range(N):
                if other[i, j]:
                    assert np.isnan(C[i, j])
                    continue
                acc = 0.0
                for k in range(K):
                    acc = acc + ((A[k, i] * A[k, j]) if trans else (A[i, k] * A[j, k]))
                want = 1.5 * acc + (-0.5) * C0[i, j]
                assert C[i, j] == want and np.signbit(C[i, j]) == np.signbit(want), (N, K, i, j)


def test_dsyrk_symmetry_integers_and_closed_forms():
    rng = np.random.default_rng(11)
    N, K = 37, 53
    A = rng.integers(-4, 5, (N, K)).astype(np.float64)
    S = rng.integers(-4, 5, (N, N)).astype(np.float64)
    S = np.tril(S) + np.tril(S, -1).T                                   # symmetric C0
    lo, up = S.copy(), S.copy()
    oracle.dsyrk(0, 0, 2.0, A, 0.5, lo)
    oracle.dsyrk(1, 0, 2.0, A, 0.5, up)
    # exact in int64 (scaled by 2 for the half-integer beta), and lower == upper^T: a_ik*a_jk commutes, same k order
    exact2 = 4 * (A.astype(np.int64) @ A.astype(np.int64).T) + S.astype(np.int64)
    assert np.array_equal(np.tril(lo) * 2, np.tril(exact2).astype(np.float64))
    assert np.array_equal(np.tril(lo), np.triu(up).T)
    assert np.array_equal(np.triu(lo, 1), np.triu(S, 1)) and np.array_equal(np.tril(up, -1), np.tril(S, -1))
    # trans: A^T A of the K x N matrix A^T is the same product
    lo_t = S.copy()
    oracle.dsyrk(0, 1, 2.0, np.ascontiguousarray(A.T), 0.5, lo_t)
    assert np.array_equal(lo_t, lo)
    # rows of A orthonormal (a permutation of unit vectors): A A^T = I
    P = np.eye(9)[rng.permutation(9)][:6]
    C = np.full((6, 6), 3.0)
    oracle.dsyrk(0, 0, 2.0, P, 1.0, C)
    assert np.array_equal(np.tril(C), np.tril(2.0 * np.eye(6) + 3.0)) and np.array_equal(np.triu(C, 1), np.triu(np.full((6, 6), 3.0), 1))
    # rank 1: C_ij = alpha*u_i*u_j with exactly that rounding sequence; float symmetry holds bit for bit
    u = rng.uniform(-1, 1, (8, 1))
    lo1, up1 = np.zeros((8, 8)), np.zeros((8, 8))
    oracle.dsyrk(0, 0, 1.25, u, 0.0, lo1); oracle.dsyrk(1, 0, 1.25, u, 0.0, up1)
    assert np.array_equal(np.tril(lo1), np.tril(1.25 * (u * u.T))) and np.array_equal(np.tril(lo1), np.triu(up1).T)


def test_dsyr2k_brute_force_symmetry_and_integers():
    rng = np.random.default_rng(13)
    for uplo in (0, 1):
        for trans in (0, 1):
            N, K = 6, 5
            A = rng.uniform(-1, 1, (K, N) if trans else (N, K)); B = rng.uniform(-1, 1, (K, N) if trans else (N, K))
            C0 = rng.uniform(-1, 1, (N, N))
            other = np.triu(np.ones((N, N), bool), 1) if uplo == 0 else np.tril(np.ones((N, N), bool), -1)
            C0[other] = np.nan
            C = C0.copy()
            oracle.dsyr2k(uplo, trans, 1.5, A, B, -0.5, C)
            a = A.T if trans else A
            b = B.T if trans else B
            for i in range(N):
                for j in range(N):
                    if other[i, j]:
                        assert np.isnan(C[i, j])
                        continue
                    s1 = 0.0
                    for k in range(K):
                        s1 = s1 + a[i, k] * b[j, k]
                    first = 1.5 * s1 + (-0.5) * C0[i, j]
                    s2 = 0.0
                    for k in range(K):
                        s2 = s2 + b[i, k] * a[j, k]
                    assert C[i, j] == 1.5 * s2 + 1.0 * first, (uplo, trans, i, j)
    # integers: exact; beta == 0: alpha*S1 + alpha*S2 commutes, so lower == upper^T bit for bit even in floating point
    N, K = 23, 31
    A = rng.integers(-4, 5, (N, K)).astype(np.float64); B = rng.integers(-4, 5, (N, K)).astype(np.float64)
    lo, up = np.zeros((N, N)), np.zeros((N, N))
    oracle.dsyr2k(0, 0, 2.0, A, B, 0.0, lo); oracle.dsyr2k(1, 0, 2.0, A, B, 0.0, up)
    Ai, Bi = A.astype(np.int64), B.astype(np.int64)
    assert np.array_equal(np.tril(lo), np.tril(2 * (Ai @ Bi.T + Bi @ Ai.T)).astype(np.float64))
    assert np.array_equal(np.tril(lo), np.triu(up).T)
    Af, Bf = rng.uniform(-1, 1, (N, K)), rng.uniform(-1, 1, (N, K))
    lo, up = np.zeros((N, N)), np.zeros((N, N))
    oracle.dsyr2k(0, 0, 1.25, Af, Bf, 0.0, lo); oracle.dsyr2k(1, 0, 1.25, Af, Bf, 0.0, up)
    assert np.array_equal(np.tril(lo), np.triu(up).T)
    # B == A: dsyr2k(alpha) == dsyrk(2 alpha) on integers
    s1, s2 = np.zeros((N, N)), np.zeros((N, N))
    oracle.dsyr2k(0, 0, 1.0, A, A, 0.0, s1); oracle.dsyrk(0, 0, 2.0, A, 0.0, s2)
    assert np.array_equal(s1, s2)


def test_dsyrk_and_dsyr2k_denominators_against_the_absolute_value_products():
    """The D these oracles return is the tolerance denominator of the DSYRK / DSYR2K float parity tests:
        dsyrk:  D_ij = |alpha| sum_k |a_ik||a_jk| + |beta||C0_ij|
        dsyr2k: D_ij = |alpha| sum_k (|a_ik||b_jk| + |b_ik||a_jk|) + |beta||C0_ij|
    on the referenced triangle and 0 elsewhere -- compared here with numpy's |A||B|^T products (an independent routine; the sums
    of positive terms agree to a few ulps), with a case where the signed result cancels (D must not), and with a wrong formula
    (a dropped term, |beta| forgotten, the signed instead of the absolute intermediate) shown to fall outside the band."""
    rng = np.random.default_rng(17)
    for uplo in (0, 1):
        for trans in (0, 1):
            N, K, alpha, beta = 19, 45, -1.75, 2.5
            A = rng.uniform(-1, 1, (K, N) if trans else (N, K)); B = rng.uniform(-1, 1, (K, N) if trans else (N, K))
            C0 = rng.uniform(-1, 1, (N, N))
            a, b = np.abs(A.T if trans else A), np.abs(B.T if trans else B)
            keep = np.tril(np.ones((N, N), bool)) if uplo == 0 else np.triu(np.ones((N, N), bool))
            D1 = oracle.dsyrk(uplo, trans, alpha, A, beta, C0.copy(), want_denominator=True)
            want1 = abs(alpha) * (a @ a.T) + abs(beta) * np.abs(C0)
            assert np.allclose(D1[keep], want1[keep], rtol=1e-13, atol=0) and (D1[~keep] == 0).all()
            D2 = oracle.dsyr2k(uplo, trans, alpha, A, B, beta, C0.copy(), want_denominator=True)
            want2 = abs(alpha) * (a @ b.T + b @ a.T) + abs(beta) * np.abs(C0)
            assert np.allclose(D2[keep], want2[keep], rtol=1e-13, atol=0) and (D2[~keep] == 0).all()
            # plausible mistakes are far outside that band
            for wrong in (abs(alpha) * (a @ b.T) + abs(beta) * np.abs(C0),              # second product dropped
                          abs(alpha) * (a @ b.T + b @ a.T),                              # |beta||C0| dropped
                          abs(alpha) * (a @ b.T + b @ a.T) + abs(beta) * np.abs(C0) +
                          np.abs(alpha * ((A.T if trans else A) @ (B if trans else B.T)) + beta * C0)):  # |mid| not removed
                assert not np.allclose(D2[keep], wrong[keep], rtol=1e-6, atol=0)
    # cancellation: B = -A on integers gives C = 0 exactly while D stays the full absolute sum
    N, K = 9, 14
    A = rng.integers(-4, 5, (N, K)).astype(np.float64)
    C = np.zeros((N, N))
    D = oracle.dsyr2k(0, 0, 1.0, A, -A, 0.0, C, want_denominator=True)
    assert np.array_equal(np.tril(D), np.tril(2.0 * (np.abs(A) @ np.abs(A).T)))
    C1 = np.zeros((N, N)); C2 = np.zeros((N, N))
    oracle.dsyr2k(0, 0, 1.0, A, A, 0.0, C1); oracle.dsyr2k(0, 0, 1.0, A, -A, 0.0, C2)
    assert np.array_equal(np.tril(C1), -np.tril(C2)) and np.tril(C1).any()


# ------------------------------------------------------------------ oracle/checksum.py: the whole-matrix checker of configs 3-5
def test_checksum_identities_are_exact_on_integers_and_see_one_wrong_element():
    """oracle.checksum.before / expected against the full oracle on a case small enough to run it (60 x 70 x 50): on integer
    inputs C x and y^T C are EXACTLY the row / column sums of oracle.dgemm's C (half-integer beta included); the gate
    denominators Dx, yD equal the oracle's elementwise D summed with |x|, |y|; and a single wrong element of C -- by one unit --
    flips exactly one row sum and one column sum."""
    import oracle.checksum as cks
    M, N, K, alpha, beta = 60, 70, 50, 2.0, -0.5
    A = synthgen.fill_numpy(M, K, 91, "A", "int"); B = synthgen.fill_numpy(K, N, 91, "B", "int"); C0 = synthgen.fill_numpy(M, N, 91, "C", "int")
    x = synthgen.fill_numpy(N, 1, 77, "A", "int")[:, 0]; y = synthgen.fill_numpy(1, M, 77, "B", "int")[0]
    assert x.any() and y.any() and np.abs(x).max() <= 4
    pre = cks.before(C0, x, y)
    C = C0.copy()
    D = oracle.dgemm(alpha, A, B, beta, C, want_denominator=True)
    Cx, yC, Dx, yD = cks.expected(alpha, A, B, beta, pre, x, y)
    assert np.array_equal(Cx, C @ x) and np.array_equal(yC, y @ C)
    # independent exact value: int64 arithmetic, scaled by 2 for the half-integer beta
    Ci2 = 2 * int(alpha) * (A.astype(np.int64) @ B.astype(np.int64)) + int(2 * beta) * C0.astype(np.int64)
    assert np.array_equal(2 * Cx, (Ci2 @ x.astype(np.int64)).astype(np.float64))
    assert np.array_equal(2 * yC, (y.astype(np.int64) @ Ci2).astype(np.float64))
    assert np.allclose(Dx, D @ np.abs(x), rtol=1e-12, atol=0) and np.allclose(yD, np.abs(y) @ D, rtol=1e-12, atol=0)
    # one wrong element: exactly its row sum and its column sum move (x_j, y_i nonzero there)
    i, j = 17, int(np.flatnonzero(x)[3])
    assert y[i] != 0
    bad = C.copy(); bad[i, j] += 1.0
    assert list(np.flatnonzero(bad @ x != Cx)) == [i] and list(np.flatnonzero(y @ bad != yC)) == [j]


def test_checksum_gate_on_floats_is_tight_enough_to_see_a_dropped_term():
    """On float inputs the identities hold within sum_j RTOL*D_ij*|x_j| (and the column form): the oracle's own C passes with
    three orders of magnitude to spare, a C with one k term dropped in one element fails, and Dx, yD are the elementwise D
    summed (so the float leg is neither vacuous nor looser than the element gate it stands in for)."""
    import oracle.checksum as cks
    rng = np.random.default_rng(19)
    M, N, K, alpha, beta = 60, 70, 50, 1.0, 0.5
    A, B, C0 = rng.uniform(-1, 1, (M, K)), rng.uniform(-1, 1, (K, N)), rng.uniform(-1, 1, (M, N))
    x = synthgen.fill_numpy(N, 1, 77, "A", "int")[:, 0]; y = synthgen.fill_numpy(1, M, 77, "B", "int")[0]
    pre = cks.before(C0, x, y)
    C = C0.copy()
    D = oracle.dgemm(alpha, A, B, beta, C, want_denominator=True)
    Cx, yC, Dx, yD = cks.expected(alpha, A, B, beta, pre, x, y)
    assert np.allclose(Dx, D @ np.abs(x), rtol=1e-12, atol=0) and np.allclose(yD, np.abs(y) @ D, rtol=1e-12, atol=0)
    assert (np.abs(C @ x - Cx) <= 1e-3 * oracle.RTOL * Dx).all() and (np.abs(y @ C - yC) <= 1e-3 * oracle.RTOL * yD).all()
    i, j = 5, int(np.flatnonzero(x)[0])
    bad = C.copy(); bad[i, j] -= alpha * A[i, 7] * B[7, j]                       # one k term of one element dropped
    assert not (np.abs(bad @ x - Cx) <= oracle.RTOL * Dx).all()
    # exactly-representable closed form: A = I, so C = B + beta*C0 and the sums are plain
    I = np.eye(M)
    Bs = rng.integers(-4, 5, (M, N)).astype(np.float64); Cs = rng.integers(-4, 5, (M, N)).astype(np.float64)
    pre = cks.before(Cs, x, y)
    Cx, yC, _, _ = cks.expected(1.0, I, Bs, 0.5, pre, x, y)
    assert np.array_equal(Cx, (Bs + 0.5 * Cs) @ x) and np.array_equal(yC, y @ (Bs + 0.5 * Cs))


# ---------------------------------------------------------------------------------------------------------------------
# DTRSM (side = Left), the routine PAPER.md:412 names as future work: op(T) X = alpha B by substitution
ALL_TRSM = list(itertools.product((0, 1), (0, 1), (0, 1)))          # uplo, trans, unit


def tri_inputs(rng, M, N, pad=0, ints=False):
    """A (M x M, NaN in the padding), B (M x N): well conditioned (rows of the off-diagonal part sum to < 1 in magnitude,
    diagonal in [1, 2)) or small integers with a unit-friendly diagonal of +-1."""
    abuf = np.full((max(M, 1), M + pad), np.nan); A = abuf[:M, :M]
    bbuf = np.full((max(M, 1), N + pad), np.nan); B = bbuf[:M, :N]
    if ints:
        A[...] = rng.integers(-2, 3, (M, M)).astype(np.float64)
        A[np.arange(M), np.arange(M)] = rng.choice([-1.0, 1.0], M)
        B[...] = rng.integers(-4, 5, (M, N)).astype(np.float64)
    else:
        A[...] = rng.uniform(-1, 1, (M, M)) / max(M, 1)
        A[np.arange(M), np.arange(M)] = rng.uniform(1, 2, M) * rng.choice([-1.0, 1.0], M)
        B[...] = rng.uniform(-1, 1, (M, N))
    return A, B


def op_tri(A, uplo, trans, unit):
    """op(T) written out densely (zeros outside the triangle, ones on a unit diagonal)."""
    T = np.tril(A) if uplo == 0 else np.triu(A)
    if unit:
        T = T - np.diag(np.diag(T)) + np.eye(A.shape[0])
    return T.T.copy() if trans else T


@pytest.mark.parametrize("uplo,trans,unit", ALL_TRSM)
def test_dtrsm_exact_rational_arithmetic_on_tiny_cases(uplo, trans, unit):
    """Brute force: the solution in exact rational arithmetic (fractions), rounded once, against the oracle within the
    substitution bound gamma_M cond-free residual gate AND to a few ulps on these well conditioned 5 x 5 cases."""
    from fractions import Fraction
    rng = np.random.default_rng(7)
    M, N, alpha = 5, 3, -1.5
    A, B = tri_inputs(rng, M, N, pad=2)
    other = np.triu(np.ones((M, M), bool), 1) if uplo == 0 else np.tril(np.ones((M, M), bool), -1)
    A[other] = np.nan                                              # the other triangle must not be read
    if unit:
        A[np.arange(M), np.arange(M)] = np.nan                     # nor a unit diagonal
    X = B.copy()
    oracle.dtrsm(uplo, trans, unit, alpha, A, X)
    T = op_tri(np.nan_to_num(A), uplo, trans, unit)
    Tf = [[Fraction(float(T[i, k])) for k in range(M)] for i in range(M)]
    lower = (uplo == 0) != bool(trans)
    order = range(M) if lower else range(M - 1, -1, -1)
    for j in range(N):
        x = [None] * M
        for i in order:
            s = Fraction(alpha) * Fraction(float(B[i, j]))
            for k in (range(i) if lower else range(i + 1, M)):
                s -= Tf[i][k] * x[k]
            x[i] = s / Tf[i][i]
        for i in range(M):
            assert abs(X[i, j] - float(x[i])) <= 8 * np.spacing(abs(float(x[i]))), (i, j)


@pytest.mark.parametrize("uplo,trans,unit", ALL_TRSM)
def test_dtrsm_against_scipy_and_residual_gate(uplo, trans, unit):
    import scipy.linalg as sl
    rng = np.random.default_rng(11)
    M, N, alpha = 61, 17, 0.75
    A, B = tri_inputs(rng, M, N, pad=3)
    X = B.copy()
    oracle.dtrsm(uplo, trans, unit, alpha, A, X)
    ref = sl.solve_triangular(A, alpha * B, lower=(uplo == 0), trans=trans, unit_diagonal=bool(unit))
    assert np.abs(X - ref).max() <= 1e-13 * np.abs(ref).max()
    res, den = oracle.dtrsm_residual(uplo, trans, unit, alpha, A, B, X)
    assert (res <= oracle.dtrsm_gate(M) * den).all()
    # the residual function itself, against the dense product in numpy (longdouble) -- and it does notice a wrong X
    T = op_tri(A, uplo, trans, unit).astype(np.longdouble)
    r2 = np.abs(np.longdouble(alpha) * B.astype(np.longdouble) - T @ X.astype(np.longdouble))
    assert np.allclose(res, r2.astype(np.float64), rtol=0, atol=1e-18)
    Xbad = X.copy(); Xbad[M // 2, N // 2] *= 1.0 + 1e-9
    res, den = oracle.dtrsm_residual(uplo, trans, unit, alpha, A, B, Xbad)
    assert not (res <= oracle.dtrsm_gate(M) * den).all()
    # sampled rows / columns pick the same numbers
    rows, cols = np.array([0, 5, M - 1]), np.array([N - 1, 2])
    rs, ds = oracle.dtrsm_residual(uplo, trans, unit, alpha, A, B, X, rows, cols)
    rf, df = oracle.dtrsm_residual(uplo, trans, unit, alpha, A, B, X)
    assert np.array_equal(rs, rf[np.ix_(rows, cols)]) and np.array_equal(ds, df[np.ix_(rows, cols)])


def test_dtrsm_closed_forms():
    rng = np.random.default_rng(3)
    M, N = 19, 7
    B = rng.uniform(-1, 1, (M, N))
    for uplo, trans, unit in ALL_TRSM:
        # identity: X = alpha*B exactly (one multiplication, a division by 1)
        X = B.copy(); oracle.dtrsm(uplo, trans, unit, 2.5, np.eye(M), X)
        assert np.array_equal(X, 2.5 * B)
        # diagonal: x_ij = (alpha*b_ij)/d_i, or alpha*b_ij when the diagonal is declared unit
        d = rng.uniform(1, 2, M)
        X = B.copy(); oracle.dtrsm(uplo, trans, unit, -0.5, np.diag(d), X)
        assert np.array_equal(X, (-0.5 * B) if unit else (-0.5 * B) / d[:, None])
        # alpha == 0: zeros, A not read (NaN), NaN in B not propagated (BLAS convention)
        X = B.copy(); X[3, 2] = np.nan
        oracle.dtrsm(uplo, trans, unit, 0.0, np.full((M, M), np.nan), X)
        assert np.array_equal(X, np.zeros((M, N)))
    # all-ones lower triangle: T X = cumulative sums of X, so X = first differences of B (exact on integers)
    Bi = rng.integers(-50, 51, (M, N)).astype(np.float64)
    ones = np.ones((M, M))
    X = Bi.copy(); oracle.dtrsm(0, 0, 0, 1.0, ones, X)
    assert np.array_equal(X, np.diff(Bi, axis=0, prepend=0.0))
    X = Bi.copy(); oracle.dtrsm(1, 0, 1, 1.0, ones, X)                # upper: differences from below
    assert np.array_equal(X, Bi - np.vstack([Bi[1:], np.zeros((1, N))]))
    # M == 0, N == 0
    oracle.dtrsm(0, 0, 0, 1.0, np.zeros((0, 0)), np.zeros((0, 5)))
    oracle.dtrsm(0, 0, 0, 1.0, np.eye(4), np.zeros((4, 0)))


@pytest.mark.parametrize("uplo,trans,unit", ALL_TRSM)
def test_dtrsm_integers_are_exact(uplo, trans, unit):
    """B := op(T) X0 in int64, then the solve must return X0 bit for bit (every intermediate is a small integer; the
    diagonal is +-1, so the divisions are exact too)."""
    rng = np.random.default_rng(5)
    M, N = 67, 9
    A, _ = tri_inputs(rng, M, N, ints=True)
    X0 = rng.integers(-3, 4, (M, N))
    T = op_tri(A, uplo, trans, unit).astype(np.int64)
    B = (T @ X0).astype(np.float64)
    X = B.copy()
    oracle.dtrsm(uplo, trans, unit, 1.0, A, X)
    assert np.array_equal(X, X0.astype(np.float64))
    X = B.copy()
    oracle.dtrsm(uplo, trans, unit, 2.0, A, X)
    assert np.array_equal(X, 2.0 * X0)


def test_dtrsm_transposed_storage_identity():
    """(uplo, trans = 1) on A is the same computation as (other uplo, trans = 0) on the written-out transpose."""
    rng = np.random.default_rng(9)
    M, N = 33, 5
    A, B = tri_inputs(rng, M, N)
    At = A.T.copy()
    for uplo in (0, 1):
        for unit in (0, 1):
            X1 = B.copy(); oracle.dtrsm(uplo, 1, unit, 1.25, A, X1)
            X2 = B.copy(); oracle.dtrsm(1 - uplo, 0, unit, 1.25, At, X2)
            assert np.array_equal(X1, X2)


def test_dtrsm_gate_is_gamma_m_plus_2():
    """oracle.dtrsm_gate(M) = gamma_(M+2) = (M+2)u / (1 - (M+2)u), u = 2^-53 (Higham, Accuracy and Stability, thm 8.5 plus the
    two extra roundings of DESIGN.md G23), checked in exact rational arithmetic; it grows with M, and the oracle's own solution of
    an ILL-CONDITIONED system (forward error large) still sits inside the backward gate -- which is why only that gate is asserted
    on such systems -- while a solution that is off by a relative 1e-12 in one element does not."""
    from fractions import Fraction
    u = Fraction(1, 2 ** 53)
    for M in (1, 5, 128, 4096, 32768):
        want = (M + 2) * u / (1 - (M + 2) * u)
        assert abs(Fraction(oracle.dtrsm_gate(M)) - want) <= want * Fraction(1, 2 ** 50)
    assert oracle.dtrsm_gate(10) < oracle.dtrsm_gate(11)
    # ill conditioned: unit lower triangle with -2 below the diagonal everywhere near it (condition number ~ 3^M)
    rng = np.random.default_rng(23)
    M, N = 48, 6
    A = np.eye(M) + np.tril(rng.uniform(-2.0, -1.0, (M, M)), -1)
    B = rng.uniform(-1, 1, (M, N))
    X = B.copy()
    oracle.dtrsm(0, 0, 0, 1.0, A, X)
    assert np.abs(X).max() > 1e8                                          # the solution blows up: forward error is hopeless
    res, den = oracle.dtrsm_residual(0, 0, 0, 1.0, A, B, X)
    assert (res <= oracle.dtrsm_gate(M) * den).all()
    Xbad = X.copy(); Xbad[M - 1, 0] *= 1.0 + 1e-12
    res, den = oracle.dtrsm_residual(0, 0, 0, 1.0, A, B, Xbad)
    assert not (res <= oracle.dtrsm_gate(M) * den).all()
