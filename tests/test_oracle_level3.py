"""Pins for oracle/level3_oracle.c (DTRSM side = Right, DTRMM, DSYMM, DPOTRF) -- `-m "not gpu"`.

The paper names these routines only as future work, so what fixes them is mathematics: every oracle is compared
with a pure-Python restatement of the definition in the same operation order (bit for bit), with exact integer / rational
arithmetic, with scipy / numpy routines (independent implementations), with closed forms and textbook worked examples, and the
parts of the operands the definitions do not reference are NaN-poisoned.
"""
import itertools
from fractions import Fraction

import numpy as np
import pytest

import oracle

ALL = list(itertools.product((0, 1), (0, 1), (0, 1)))          # uplo, trans, unit


def tri_operand(rng, n, ints=False):
    """A square matrix whose triangles are both usable: well conditioned (off-diagonal / n, |diagonal| in [1, 2)); integers: +-1
    diagonal."""
    if ints:
        A = rng.integers(-3, 4, (n, n)).astype(np.float64)
        A[np.arange(n), np.arange(n)] = rng.choice([-1.0, 1.0], n)
        return A
    A = rng.uniform(-1, 1, (n, n)) / max(n, 1)
    A[np.arange(n), np.arange(n)] = rng.uniform(1, 2, n) * rng.choice([-1.0, 1.0], n)
    return A


def op_tri(A, uplo, trans, unit):
    T = np.tril(A) if uplo == 0 else np.triu(A)
    if unit:
        T = T - np.diag(np.diag(T)) + np.eye(A.shape[0])
    return T.T if trans else T


def poison(A, uplo, unit):
    A = A.copy()
    n = A.shape[0]
    other = np.triu(np.ones((n, n), bool), 1) if uplo == 0 else np.tril(np.ones((n, n), bool), -1)
    A[other] = np.nan
    if unit:
        A[np.arange(n), np.arange(n)] = np.nan
    return A


# ------------------------------------------------------------------------------------------------ DTRSM, side = Right
@pytest.mark.parametrize("uplo,trans,unit", ALL)
def test_dtrsm_right_brute_force_scipy_and_exact_integers(uplo, trans, unit):
    rng = np.random.default_rng(100 + 4 * uplo + 2 * trans + unit)
    M, N, alpha = 7, 13, -0.75
    A = tri_operand(rng, N)
    B = rng.uniform(-1, 1, (M, N))
    X = B.copy()
    oracle.dtrsm_right(uplo, trans, unit, alpha, poison(A, uplo, unit), X)
    # (1) pure-Python loops in the order of the definition: bit for bit
    T = op_tri(A, uplo, trans, unit)
    upper = (uplo == 1) != bool(trans)
    for i in range(M):
        x = [0.0] * N
        for j in (range(N) if upper else range(N - 1, -1, -1)):
            s = alpha * B[i, j]
            for k in (range(j) if upper else range(N - 1, j, -1)):
                s = s - x[k] * T[k, j]
            x[j] = s if unit else s / T[j, j]
        assert list(X[i]) == x
    # (2) an independent routine: X op(T) = alpha B  <=>  op(T)^T X^T = alpha B^T
    import scipy.linalg as sl
    ref = sl.solve_triangular(T.T, alpha * B.T, lower=upper).T
    assert np.abs(X - ref).max() <= 1e-13 * np.abs(ref).max()
    # (3) the identity with the LEFT-side oracle on written-out transposes: same operations in the same order, same bits
    Xt = np.ascontiguousarray(B.T)
    oracle.dtrsm(uplo, 1 - trans, unit, alpha, A, Xt)
    assert np.array_equal(Xt.T, X)
    # (4) integers with a +-1 diagonal: B := X0 op(T) in int64, solved back bit for bit
    Ai = tri_operand(rng, N, ints=True)
    X0 = rng.integers(-3, 4, (M, N))
    Bi = (X0 @ op_tri(Ai, uplo, trans, unit).astype(np.int64)).astype(np.float64)
    oracle.dtrsm_right(uplo, trans, unit, 2.0, poison(Ai, uplo, unit), Bi)
    assert np.array_equal(Bi, 2.0 * X0)


def test_dtrsm_right_closed_forms_and_degenerate_cases():
    rng = np.random.default_rng(5)
    M, N = 6, 9
    B = rng.uniform(-1, 1, (M, N))
    for uplo, trans, unit in ALL:
        X = B.copy(); oracle.dtrsm_right(uplo, trans, unit, 2.5, np.eye(N), X)
        assert np.array_equal(X, 2.5 * B)
        d = rng.uniform(1, 2, N)
        X = B.copy(); oracle.dtrsm_right(uplo, trans, unit, -0.5, np.diag(d), X)
        assert np.array_equal(X, (-0.5 * B) if unit else (-0.5 * B) / d[None, :])
        X = B.copy(); X[1, 2] = np.nan
        oracle.dtrsm_right(uplo, trans, unit, 0.0, np.full((N, N), np.nan), X)       # alpha == 0: zeros, A not read
        assert np.array_equal(X, np.zeros((M, N)))
    # all-ones upper triangle: X T = cumulative sums along the row, so X = first differences of B along the row (integers)
    Bi = rng.integers(-50, 51, (M, N)).astype(np.float64)
    X = Bi.copy(); oracle.dtrsm_right(1, 0, 0, 1.0, np.ones((N, N)), X)
    assert np.array_equal(X, np.diff(Bi, axis=1, prepend=0.0))
    oracle.dtrsm_right(0, 0, 0, 1.0, np.zeros((0, 0)), np.zeros((4, 0)))
    oracle.dtrsm_right(0, 0, 0, 1.0, np.eye(3), np.zeros((0, 3)))


# ------------------------------------------------------------------------------------------------ DTRMM
@pytest.mark.parametrize("side", [0, 1])
@pytest.mark.parametrize("uplo,trans,unit", ALL)
def test_dtrmm_brute_force_numpy_and_integers(side, uplo, trans, unit):
    rng = np.random.default_rng(200 + 8 * side + 4 * uplo + 2 * trans + unit)
    M, N, alpha = 8, 11, 1.25
    n = M if side == 0 else N
    A = tri_operand(rng, n)
    B0 = rng.uniform(-1, 1, (M, N))
    B = B0.copy()
    oracle.dtrmm(side, uplo, trans, unit, alpha, poison(A, uplo, unit), B)
    T = op_tri(A, uplo, trans, unit)
    lower = (uplo == 0) != bool(trans)
    for i in range(M):
        for j in range(N):
            acc = 0.0
            if side == 0:
                for k in (range(0, i + 1) if lower else range(i, M)):
                    acc = acc + (B0[k, j] if (k == i and unit) else T[i, k] * B0[k, j])
            else:
                for k in (range(j, N) if lower else range(0, j + 1)):
                    acc = acc + (B0[i, k] if (k == j and unit) else B0[i, k] * T[k, j])
            assert B[i, j] == alpha * acc, (i, j)
    ref = alpha * (T @ B0 if side == 0 else B0 @ T)
    assert np.abs(B - ref).max() <= 1e-14 * np.abs(ref).max()
    # integers: exact against int64; and DTRSM undoes DTRMM bit for bit there (+-1 diagonal)
    Ai = tri_operand(rng, n, ints=True)
    Bi0 = rng.integers(-3, 4, (M, N))
    Bi = Bi0.astype(np.float64)
    oracle.dtrmm(side, uplo, trans, unit, 2.0, poison(Ai, uplo, unit), Bi)
    Ti = op_tri(Ai, uplo, trans, unit).astype(np.int64)
    assert np.array_equal(Bi, 2.0 * (Ti @ Bi0 if side == 0 else Bi0 @ Ti))
    back = Bi.copy()
    (oracle.dtrsm if side == 0 else oracle.dtrsm_right)(uplo, trans, unit, 0.5, Ai, back)
    assert np.array_equal(back, Bi0.astype(np.float64))
    # alpha == 0 and identity
    Z = B0.copy(); Z[0, 0] = np.nan
    oracle.dtrmm(side, uplo, trans, unit, 0.0, np.full((n, n), np.nan), Z)
    assert np.array_equal(Z, np.zeros((M, N)))
    I = B0.copy(); oracle.dtrmm(side, uplo, trans, unit, 1.0, np.eye(n), I)
    assert np.array_equal(I, B0)


# ------------------------------------------------------------------------------------------------ DSYMM
@pytest.mark.parametrize("side", [0, 1])
@pytest.mark.parametrize("uplo", [0, 1])
def test_dsymm_is_dgemm_on_the_mirrored_triangle(side, uplo):
    rng = np.random.default_rng(300 + 2 * side + uplo)
    M, N, alpha, beta = 9, 7, 1.5, -0.5
    n = M if side == 0 else N
    S = rng.uniform(-1, 1, (n, n)); S = np.tril(S) + np.tril(S, -1).T              # symmetric
    A = poison(S, uplo, 0)                                                          # only the triangle is stored
    B = rng.uniform(-1, 1, (M, N)); C0 = rng.uniform(-1, 1, (M, N))
    C = C0.copy()
    D = oracle.dsymm(side, uplo, alpha, A, B, beta, C, want_denominator=True)
    for i in range(M):
        for j in range(N):
            acc = 0.0
            for k in range(n):
                acc = acc + ((S[i, k] * B[k, j]) if side == 0 else (B[i, k] * S[k, j]))
            assert C[i, j] == alpha * acc + beta * C0[i, j], (i, j)
    ref = alpha * (S @ B if side == 0 else B @ S) + beta * C0
    assert np.abs(C - ref).max() <= 1e-14
    want_D = abs(alpha) * (np.abs(S) @ np.abs(B) if side == 0 else np.abs(B) @ np.abs(S)) + abs(beta) * np.abs(C0)
    assert np.allclose(D, want_D, rtol=1e-13, atol=0)
    # both triangles of the same symmetric matrix give the same bits; integers are exact
    C2 = C0.copy(); oracle.dsymm(side, 1 - uplo, alpha, poison(S, 1 - uplo, 0), B, beta, C2)
    assert np.array_equal(C, C2)
    Si = rng.integers(-4, 5, (n, n)); Si = np.tril(Si) + np.tril(Si, -1).T
    Bi = rng.integers(-4, 5, (M, N)); Ci = rng.integers(-4, 5, (M, N))
    Cf = Ci.astype(np.float64)
    oracle.dsymm(side, uplo, 2.0, poison(Si.astype(np.float64), uplo, 0), Bi.astype(np.float64), 3.0, Cf)
    assert np.array_equal(Cf, (2 * (Si @ Bi if side == 0 else Bi @ Si) + 3 * Ci).astype(np.float64))
    # a NON-symmetric stored matrix: only the named triangle counts (catches reading the other one)
    R = rng.uniform(-1, 1, (n, n))
    Sym = np.tril(R) + np.tril(R, -1).T if uplo == 0 else np.triu(R) + np.triu(R, 1).T
    C3, C4 = C0.copy(), C0.copy()
    oracle.dsymm(side, uplo, alpha, R, B, beta, C3); oracle.dsymm(side, uplo, alpha, Sym, B, beta, C4)
    assert np.array_equal(C3, C4)


# ------------------------------------------------------------------------------------------------ DPOTRF
def spd(rng, n):
    G = rng.uniform(-1, 1, (n, n + 3))
    return G @ G.T + n * np.eye(n) * 0.05


@pytest.mark.parametrize("uplo", [0, 1])
def test_dpotrf_brute_force_bit_for_bit_and_untouched_triangle(uplo):
    """Pure-Python Cholesky-Banachiewicz in the order of the definition: identical bits; the other triangle (NaN) is neither
    read nor written."""
    rng = np.random.default_rng(400 + uplo)
    for n in (1, 2, 5, 12):
        S = spd(rng, n)
        A = poison(S, uplo, 0)
        info = oracle.dpotrf(uplo, A)
        assert info == 0
        f = [[0.0] * n for _ in range(n)]
        for i in range(n):
            for j in range(i):
                s = S[i, j]
                for k in range(j):
                    s = s - f[i][k] * f[j][k]
                f[i][j] = s / f[j][j]
            s = S[i, i]
            for k in range(i):
                s = s - f[i][k] * f[i][k]
            f[i][i] = float(np.sqrt(s))
        F = np.array(f)
        got = np.tril(A) if uplo == 0 else np.triu(A).T
        assert np.array_equal(np.nan_to_num(got), F)
        other = np.triu(np.ones((n, n), bool), 1) if uplo == 0 else np.tril(np.ones((n, n), bool), -1)
        assert np.isnan(A[other]).all()


def test_dpotrf_textbook_example_integers_and_closed_forms():
    # the classic worked example (e.g. the Cholesky decomposition article of Wikipedia): exact in floating point
    A = np.array([[4.0, 12, -16], [12, 37, -43], [-16, -43, 98]])
    L = A.copy()
    assert oracle.dpotrf(0, L) == 0
    assert np.array_equal(np.tril(L), np.array([[2.0, 0, 0], [6, 1, 0], [-8, 5, 3]]))
    U = A.copy()
    assert oracle.dpotrf(1, U) == 0
    assert np.array_equal(np.triu(U), np.tril(L).T)
    # integer L0 with positive diagonal, A := L0 L0^T in int64: the factorization returns L0 bit for bit (square roots of
    # perfect squares and the divisions are exact)
    rng = np.random.default_rng(7)
    n = 40
    L0 = np.tril(rng.integers(-3, 4, (n, n)), -1) + np.diag(rng.integers(1, 5, n))
    Ai = (L0 @ L0.T).astype(np.float64)
    for uplo in (0, 1):
        F = poison(Ai, uplo, 0)
        assert oracle.dpotrf(uplo, F) == 0
        got = np.tril(F) if uplo == 0 else np.triu(F).T
        assert np.array_equal(np.nan_to_num(got), L0.astype(np.float64))
    # identity and diagonal
    I = np.eye(6); assert oracle.dpotrf(0, I) == 0 and np.array_equal(I, np.eye(6))
    d = rng.uniform(0.5, 4, 9)
    Dm = np.diag(d * d); assert oracle.dpotrf(1, Dm) == 0
    assert np.array_equal(np.diag(Dm), np.sqrt(d * d)) and np.array_equal(Dm - np.diag(np.diag(Dm)), np.zeros((9, 9)))
    # rank-one plus identity: A = I + v v^T has the closed form l_ij = v_i v_j / sqrt(s_{j-1} s_j), s_j = 1 + sum_{k<=j} v_k^2
    v = rng.uniform(-1, 1, 8)
    A1 = np.eye(8) + np.outer(v, v)
    F = A1.copy(); assert oracle.dpotrf(0, F) == 0
    s = 1.0 + np.cumsum(v * v); sm1 = np.concatenate([[1.0], s[:-1]])
    want = np.tril(np.outer(v, v) / np.sqrt(sm1 * s)[None, :], -1) + np.diag(np.sqrt(s / sm1))
    assert np.abs(np.tril(F) - want).max() <= 1e-14
    assert oracle.dpotrf(0, np.zeros((0, 0))) == 0


@pytest.mark.parametrize("uplo", [0, 1])
def test_dpotrf_against_scipy_and_the_backward_gate(uplo):
    import scipy.linalg as sl
    rng = np.random.default_rng(410 + uplo)
    n = 90
    S = spd(rng, n)
    F = poison(S, uplo, 0)
    assert oracle.dpotrf(uplo, F) == 0
    ref = sl.cholesky(S, lower=(uplo == 0))
    got = np.nan_to_num(F)
    assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()
    res, den = oracle.dpotrf_residual(uplo, S, got)
    assert (res <= oracle.dpotrf_gate(n) * den).all()
    # the gate itself: gamma_(n+2) in exact rational arithmetic, and the residual function against exact rationals
    u = Fraction(1, 2 ** 53)
    want = (n + 2) * u / (1 - (n + 2) * u)
    assert abs(Fraction(oracle.dpotrf_gate(n)) - want) <= want * Fraction(1, 2 ** 50)
    Lm = got if uplo == 0 else got.T
    for (i, j) in ((0, 0), (5, 3), (n - 1, n - 1), (n - 1, 0), (17, 60)):
        exact = Fraction(float(S[max(i, j), min(i, j)])) - sum(Fraction(float(Lm[i, k])) * Fraction(float(Lm[j, k])) for k in range(min(i, j) + 1))
        # long double carries a 64-bit significand: each of its min(i, j) + 2 operations errs by at most 2^-64 of the running size
        assert abs(float(abs(exact)) - res[i, j]) <= (min(i, j) + 3) * 2.0 ** -64 * (den[i, j] + abs(S[i, j]))
        dd = sum(abs(Fraction(float(Lm[i, k])) * Fraction(float(Lm[j, k]))) for k in range(min(i, j) + 1))
        assert abs(float(dd) - den[i, j]) <= 1e-15 * den[i, j]
    # sampled rows / columns pick the same numbers; a factor that is off by 1e-9 in one entry fails the gate
    rows, cols = np.array([0, 7, n - 1]), np.array([n - 1, 2])
    rs, ds = oracle.dpotrf_residual(uplo, S, got, rows, cols)
    assert np.array_equal(rs, res[np.ix_(rows, cols)]) and np.array_equal(ds, den[np.ix_(rows, cols)])
    bad = got.copy()
    if uplo == 0:
        bad[n // 2, n // 3] *= 1.0 + 1e-9
    else:
        bad[n // 3, n // 2] *= 1.0 + 1e-9
    res, den = oracle.dpotrf_residual(uplo, S, bad)
    assert not (res <= oracle.dpotrf_gate(n) * den).all()


def test_dpotrf_reports_the_first_minor_that_is_not_positive_definite():
    rng = np.random.default_rng(9)
    n = 12
    S = spd(rng, n)
    ok = S.copy(); assert oracle.dpotrf(0, ok) == 0
    for k in (0, 4, n - 1):
        A = S.copy()
        A[k, k] = -1.0 if k == 0 else float(np.sum(ok[k, :k] ** 2)) * (1.0 - 1e-3)        # the k-th pivot becomes negative
        F = A.copy()
        assert oracle.dpotrf(0, F) == k + 1
        assert np.array_equal(F[:k, :], ok[:k, :])                       # the rows before it are the factor's
        assert np.array_equal(np.tril(F[k:k + 1, :k]), np.tril(ok[k:k + 1, :k])) and F[k, k] == A[k, k]
        assert np.array_equal(F[k + 1:, :], A[k + 1:, :])                # nothing below was touched
        U = A.T.copy()
        assert oracle.dpotrf(1, U) == k + 1
    Z = np.zeros((3, 3)); assert oracle.dpotrf(0, Z) == 1                # a zero pivot is "not positive"
    Nn = np.eye(3); Nn[1, 1] = np.nan; assert oracle.dpotrf(0, Nn) == 2  # and so is NaN
