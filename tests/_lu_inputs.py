"""Inputs for the LU tests (CPU pins and GPU parity) -- no arithmetic of the method: matrices with a KNOWN factorization, built
from the factors by exact products.

exact_lu_case(M, N, seed): A = P^T (L U) where L is unit lower trapezoidal with entries in {-1/2, 0, 1/2} below the diagonal, U is
upper trapezoidal with small integer entries and a non-zero diagonal, and P is a sequence of row interchanges (ipiv[j] >= j).
Every intermediate quantity of Gaussian elimination on A -- in any blocking -- is a multiple of 1/2 of modest size, hence exact in
FP64, and at step j the pivot candidates are u_jj (once) and +-u_jj/2 or 0 (all other rows): the pivot is unique, so ipiv, L and U
must be reproduced BIT FOR BIT by any correct implementation.
"""
import numpy as np


def exact_lu_case(M, N, seed, umax=3):
    rng = np.random.default_rng(seed)
    n = min(M, N)
    L2 = rng.integers(-1, 2, (M, n)).astype(np.int64)            # 2 * L below the diagonal
    L2 = np.tril(L2, -1)
    L2[np.arange(n), np.arange(n)] = 2                            # unit diagonal
    U = np.triu(rng.integers(-umax, umax + 1, (n, N)).astype(np.int64))
    d = rng.integers(1, umax + 1, n) * rng.choice([-1, 1], n)
    U[np.arange(n), np.arange(n)] = d
    # 2 * (L U): integers below 2^53 at every partial sum, so the FP64 product is exact in any order of summation
    LU2 = L2.astype(np.float64) @ U.astype(np.float64)
    assert np.abs(LU2).max() < 2.0 ** 50
    # a fourth of the steps need no interchange (ipiv[j] = j), as in real matrices with a dominant diagonal
    keep = rng.random(n) < 0.25
    ipiv = np.where(keep, np.arange(n), np.array([rng.integers(j, M) for j in range(n)], dtype=np.int64)).astype(np.int64)
    PA2 = LU2.copy()
    for j in range(n - 1, -1, -1):                                # undo the interchanges, last one first:  A = P^T (L U)
        p = int(ipiv[j])
        if p != j:
            PA2[[j, p]] = PA2[[p, j]]
    A = PA2 / 2.0
    F = np.zeros((M, N))                                          # the factors as DGETRF stores them
    Lf = L2.astype(np.float64) / 2.0
    for i in range(M):
        k = min(i, n)
        F[i, :k] = Lf[i, :k]
    F[:n, :] += U.astype(np.float64)
    return A, F, ipiv


def apply_interchanges(A, ipiv):
    """P A: the interchanges row j <-> row ipiv[j], j = 0, 1, ..., applied in that order (a copy)."""
    B = A.copy()
    for j, p in enumerate(ipiv):
        p = int(p)
        if p != j:
            B[[j, p]] = B[[p, j]]
    return B


def split_lu(F):
    """(L, U) of the packed factors: L  M x n unit lower trapezoidal, U  n x N upper trapezoidal, n = min(M, N)."""
    M, N = F.shape
    n = min(M, N)
    L = np.tril(F[:, :n], -1)
    L[np.arange(n), np.arange(n)] = 1.0
    U = np.triu(F[:n, :])
    return L, U
