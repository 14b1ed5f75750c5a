"""Pins for oracle_dgetrf / oracle_dgetrf_residual (oracle/level3_oracle.c) -- `-m "not gpu"`.

The paper names LU only as future work, so what fixes the oracle is mathematics: a pure-Python restatement of
Gaussian elimination with partial pivoting in the same operation order (bit for bit), exact rational arithmetic, scipy's
lu_factor (LAPACK, an independent implementation), matrices built from known factors that must come back bit for bit, closed
forms (identity, permutations, triangular inputs, ties, zero columns), a textbook worked example, and -- for the residual
function -- a long-double numpy product and single-element perturbations.
"""
from fractions import Fraction

import numpy as np
import pytest
import scipy.linalg

import oracle
from _lu_inputs import apply_interchanges, exact_lu_case, split_lu


def brute_force_lu(A):
    """Gaussian elimination with partial pivoting on a list of lists of Python floats, the definition in the oracle's header."""
    M, N = len(A), len(A[0]) if A else 0
    A = [row[:] for row in A]
    ipiv, info = [], 0
    for j in range(min(M, N)):
        p, best = j, abs(A[j][j])
        for i in range(j + 1, M):
            if abs(A[i][j]) > best:
                p, best = i, abs(A[i][j])
        ipiv.append(p)
        A[j], A[p] = A[p], A[j]
        if A[j][j] == 0.0:
            info = info or j + 1
            continue
        for i in range(j + 1, M):
            l = A[i][j] / A[j][j]
            A[i][j] = l
            for k in range(j + 1, N):
                prod = l * A[j][k]
                A[i][k] = A[i][k] - prod
    return A, ipiv, info


@pytest.mark.parametrize("M,N", [(m, n) for m in range(1, 7) for n in range(1, 7)] + [(23, 9), (9, 23), (40, 40)])
def test_dgetrf_brute_force_bit_for_bit(M, N):
    rng = np.random.default_rng(1000 * M + N)
    A = rng.uniform(-1, 1, (M, N))
    ref, ipiv_ref, info_ref = brute_force_lu(A.tolist())
    F = A.copy()
    ipiv, info = oracle.dgetrf(F)
    assert info == info_ref == 0
    assert ipiv.tolist() == ipiv_ref
    assert np.array_equal(F, np.array(ref))


def test_dgetrf_rounds_the_product_before_it_subtracts():
    # l = 1 - e, u = 1 + e, e = 2^-27: l * u = 1 - 2^-54 rounds to 1, so a - l*u = 1 - 1 = 0 exactly (and the zero pivot is
    # reported); a fused multiply-add would leave 2^-54 and no info
    e = 2.0 ** -27
    A = np.array([[1.0, 1.0 + e], [1.0 - e, 1.0]])
    F = A.copy()
    ipiv, info = oracle.dgetrf(F)
    assert ipiv.tolist() == [0, 1]
    assert F[1, 0] == 1.0 - e and F[1, 1] == 0.0 and info == 2


def exact_rational_lu(A):
    """The same elimination in exact rational arithmetic (pivots: first maximum of the exact values)."""
    M, N = A.shape
    R = [[Fraction(float(x)) for x in row] for row in A]
    ipiv = []
    for j in range(min(M, N)):
        p = max(range(j, M), key=lambda i: (abs(R[i][j]), -i))
        ipiv.append(p)
        R[j], R[p] = R[p], R[j]
        if R[j][j] == 0:
            continue
        for i in range(j + 1, M):
            l = R[i][j] / R[j][j]
            R[i][j] = l
            for k in range(j + 1, N):
                R[i][k] -= l * R[j][k]
    return R, ipiv


def test_dgetrf_pivot_sequence_of_the_3x3_case():
    A = np.array([[1.0, 4.0, 2.0], [3.0, 5.0, 7.0], [6.0, 2.0, 1.0]])
    F = A.copy()
    ipiv, info = oracle.dgetrf(F)
    # by hand: pivot 6 (row 2); rows become [6,2,1],[3,5,7],[1,4,2]; multipliers 1/2, 1/6; Schur complement [[4, 13/2], [11/3, 11/6]];
    # pivot 4 (no interchange); multiplier 11/12; last pivot 11/6 - 11/12 * 13/2 = -33/8
    assert ipiv.tolist() == [2, 1, 2] and info == 0
    want = np.array([[6.0, 2.0, 1.0], [0.5, 4.0, 6.5], [1.0 / 6.0, 11.0 / 12.0, -33.0 / 8.0]])
    assert np.allclose(F, want, rtol=4e-16, atol=0)


@pytest.mark.parametrize("M,N", [(5, 5), (7, 4), (4, 7)])
def test_dgetrf_against_exact_rational_arithmetic(M, N):
    rng = np.random.default_rng(7 * M + N)
    A = rng.integers(-9, 10, (M, N)).astype(np.float64) + rng.uniform(-0.25, 0.25, (M, N))
    F = A.copy()
    ipiv, info = oracle.dgetrf(F)
    Fr, ip = exact_rational_lu(A)
    assert info == 0 and ipiv.tolist() == ip
    exact = np.array([[float(x) for x in row] for row in Fr])
    assert np.allclose(F, exact, rtol=1e-12, atol=1e-13)
    # and the exact factors multiply back to P A exactly (the rational elimination itself is right)
    n = min(M, N)
    PA = apply_interchanges(A, ip)
    for i in range(M):
        for j in range(N):
            s = sum((Fraction(1) if k == i else Fr[i][k]) * Fr[k][j] for k in range(min(i, j, n - 1) + 1))
            assert s == Fraction(float(PA[i, j]))


@pytest.mark.parametrize("M,N,seed", [(64, 64, 1), (200, 120, 2), (120, 200, 3), (301, 301, 4)])
def test_dgetrf_against_scipy_lapack(M, N, seed):
    rng = np.random.default_rng(seed)
    A = rng.uniform(-1, 1, (M, N))
    F = A.copy()
    ipiv, info = oracle.dgetrf(F)
    lu, piv = scipy.linalg.lu_factor(A) if M == N else scipy.linalg.lapack.dgetrf(A)[:2]
    assert info == 0
    assert ipiv.tolist() == piv.tolist()                   # scipy's pivots are 0-based row indices, like ours
    assert np.allclose(F, lu, rtol=1e-10, atol=1e-12)
    # backward gate (Higham thm 9.3) through the residual function, on every element
    res, den = oracle.dgetrf_residual(A, F, ipiv)
    assert (res <= oracle.dgetrf_gate(min(M, N)) * den).all()


@pytest.mark.parametrize("M,N,seed", [(1, 1, 0), (8, 8, 1), (37, 37, 2), (50, 20, 3), (20, 50, 4), (130, 130, 5)])
def test_dgetrf_returns_known_factors_bit_for_bit(M, N, seed):
    A, F_want, ipiv_want = exact_lu_case(M, N, seed)
    F = A.copy()
    ipiv, info = oracle.dgetrf(F)
    assert info == 0
    assert np.array_equal(ipiv, ipiv_want)
    assert np.array_equal(F, F_want)
    L, U = split_lu(F_want)
    assert np.array_equal(L @ U, apply_interchanges(A, ipiv_want))      # the case itself: P A = L U exactly
    res, den = oracle.dgetrf_residual(A, F, ipiv)
    assert (res == 0).all()


def test_dgetrf_closed_forms_ties_and_singular_inputs():
    n = 6
    I = np.eye(n)
    F = I.copy()
    ipiv, info = oracle.dgetrf(F)
    assert info == 0 and ipiv.tolist() == list(range(n)) and np.array_equal(F, I)
    # an upper triangular matrix with a dominant diagonal is its own U, no interchange
    U = np.triu(np.arange(1.0, n * n + 1).reshape(n, n)) + 100 * np.eye(n)
    F = U.copy()
    ipiv, info = oracle.dgetrf(F)
    assert info == 0 and ipiv.tolist() == list(range(n)) and np.array_equal(F, U)
    # a permutation matrix: L = U = I, and the interchanges sort the rows
    perm = np.array([3, 0, 5, 1, 2, 4])
    P = np.zeros((n, n)); P[np.arange(n), perm] = 1.0
    F = P.copy()
    ipiv, info = oracle.dgetrf(F)
    assert info == 0 and np.array_equal(F, I) and np.array_equal(apply_interchanges(P, ipiv), I)
    # ties: the FIRST maximum is the pivot (IDAMAX), also between +x and -x
    A = np.array([[1.0, 2.0], [-1.0, 5.0], [1.0, 7.0]])
    F = A.copy()
    ipiv, info = oracle.dgetrf(F)
    assert ipiv.tolist() == [0, 1] and info == 0            # Schur complement: 5 + 2 = 7, 7 - 2 = 5
    assert np.array_equal(F, np.array([[1.0, 2.0], [-1.0, 7.0], [1.0, 5.0 / 7.0]]))
    A = np.array([[-3.0, 1.0], [3.0, 2.0], [3.0, 4.0]])     # three equal magnitudes: row 0 stays; then 3 and 5: row 2 comes up
    F = A.copy()
    ipiv, info = oracle.dgetrf(F)
    assert ipiv.tolist() == [0, 2] and np.array_equal(F, np.array([[-3.0, 1.0], [-1.0, 5.0], [-1.0, 3.0 / 5.0]]))
    # a zero column: info = that column + 1 (first one only), the factorization still completes and P A = L U holds
    A = np.array([[2.0, 4.0, 1.0, 3.0], [1.0, 2.0, 5.0, 1.0], [4.0, 8.0, 2.0, 2.0], [2.0, 4.0, 7.0, 9.0]])    # column 1 = 2 * column 0
    F = A.copy()
    ipiv, info = oracle.dgetrf(F)
    assert info == 2 and F[1, 1] == 0.0
    L, Uf = split_lu(F)
    assert np.allclose(L @ Uf, apply_interchanges(A, ipiv), rtol=0, atol=1e-14)
    Z = np.zeros((3, 3))
    ipiv, info = oracle.dgetrf(Z)
    assert info == 1 and ipiv.tolist() == [0, 1, 2] and not Z.any()
    # empty shapes
    for shape in ((0, 5), (5, 0), (0, 0)):
        ipiv, info = oracle.dgetrf(np.zeros(shape))
        assert info == 0 and ipiv.size == 0


def test_dgetrf_textbook_example():
    # Trefethen & Bau, Numerical Linear Algebra, lecture 21: the 4 x 4 example of Gaussian elimination with partial pivoting
    with open(__file__.rsplit("/", 1)[0] + "/golden/lu_textbook_example.txt") as f:
        rows = [[Fraction(x) for x in line.split()] for line in f if line.strip() and not line.startswith("#")]
    A = np.array([[float(x) for x in r] for r in rows[0:4]])
    Lw, Uw, Pw = rows[4:8], rows[8:12], rows[12:16]
    # the printed factors are consistent: P A = L U in exact arithmetic
    for i in range(4):
        for j in range(4):
            assert sum(Lw[i][k] * Uw[k][j] for k in range(4)) == sum(Pw[i][k] * rows[k][j] for k in range(4))
    F = A.copy()
    ipiv, info = oracle.dgetrf(F)
    assert info == 0
    L, U = split_lu(F)
    assert np.allclose(L, np.array([[float(x) for x in r] for r in Lw]), rtol=1e-15, atol=1e-16)
    assert np.allclose(U, np.array([[float(x) for x in r] for r in Uw]), rtol=1e-15, atol=1e-16)
    assert np.array_equal(apply_interchanges(A, ipiv), np.array([[float(x) for x in r] for r in Pw]) @ A)


def test_dgetrf_residual_against_long_double_numpy_and_perturbations():
    rng = np.random.default_rng(11)
    for (M, N) in ((30, 30), (45, 20), (20, 45)):
        A = rng.uniform(-1, 1, (M, N))
        F = A.copy()
        ipiv, info = oracle.dgetrf(F)
        L, U = split_lu(F)
        PA = apply_interchanges(A, ipiv).astype(np.longdouble)
        want_res = np.abs(PA - L.astype(np.longdouble) @ U.astype(np.longdouble))
        want_den = np.abs(L).astype(np.longdouble) @ np.abs(U).astype(np.longdouble)
        res, den = oracle.dgetrf_residual(A, F, ipiv)
        assert np.allclose(res, want_res.astype(np.float64), rtol=1e-9, atol=4e-18)      # long double: 2^-64 per operation on sums of O(10)
        assert np.allclose(den, want_den.astype(np.float64), rtol=1e-15, atol=0)
        gate = oracle.dgetrf_gate(min(M, N))
        assert (res <= gate * den).all()
        # sampled rows / columns are the same numbers
        rows, cols = np.array([0, M - 1, M // 2]), np.array([N - 1, 0, N // 3])
        rs, ds = oracle.dgetrf_residual(A, F, ipiv, rows, cols)
        assert np.array_equal(rs, res[np.ix_(rows, cols)]) and np.array_equal(ds, den[np.ix_(rows, cols)])
        # one perturbed element of L, of U, or one wrong interchange is noticed
        for (i, j) in ((M - 1, 0), (0, N - 1), (min(M, N) // 2, min(M, N) // 2)):
            G = F.copy()
            G[i, j] += 1e-9
            r2, d2 = oracle.dgetrf_residual(A, G, ipiv)
            assert not (r2 <= gate * d2).all()
        ip2 = ipiv.copy()
        j = 3
        ip2[j] = ip2[j] + 1 if ip2[j] + 1 < M else j
        r2, d2 = oracle.dgetrf_residual(A, F, ip2)
        assert not (r2 <= gate * d2).all()
    with pytest.raises(ValueError):
        oracle.dgetrf_residual(A, F, np.zeros_like(ipiv) - 1)


def test_dgetrf_gate_is_gamma_n():
    for n in (1, 5, 1000, 32768):
        u = Fraction(1, 2 ** 53)
        assert abs(Fraction(oracle.dgetrf_gate(n)) - n * u / (1 - n * u)) < Fraction(1, 2 ** 80)
