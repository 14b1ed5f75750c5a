"""TEST INFRASTRUCTURE ONLY -- the CPU oracle for out-of-core DGEMM (C = alpha*A*B + beta*C, FP64).

Plain C (oracle/dgemm_oracle.c, see its header for the definition and the PAPER.md citations),
compiled with `gcc -O2 -ffp-contract=off -fopenmp` and called through ctypes.  It shares nothing
with the CUDA path in paper_1808_05056_b200/ and must never be imported by it: only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs use it.

Pinned by tests/test_oracle_pins.py (brute force, int64 exactness, closed forms, exact-sum error
bound, numpy cross-check, the paper's 44-element partition example; dsyrk: brute force on the triangle,
exact symmetry, int64 exactness, untouched other triangle; dtrsm: scipy's solve_triangular, exact rational
arithmetic on tiny cases, identity / diagonal / all-ones closed forms, int64 exactness, transposed-storage identity; the D returned
by dsyrk / dsyr2k against numpy's |A||B|^T products; dtrsm_gate against gamma_(M+2) in exact arithmetic; oracle/checksum.py
against the full oracle, int64 arithmetic and single-element mutations; dtrsm_right / dtrmm / dsymm / dpotrf (level3_oracle.c) in
tests/test_oracle_level3.py; dgetrf and its residual in tests/test_oracle_lu.py) -- nothing here is "parity unpinned".
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dgemm_oracle.c")
_SRC3 = os.path.join(_HERE, "level3_oracle.c")          # DTRSM (right), DTRMM, DPOTRF: the routines PAPER.md:412 names
_LIB = os.path.join(_HERE, "liboracle.so")

# the gate of BASELINE.json north_star as read in DESIGN.md (G14): |C - C_ref| <= RTOL * D
RTOL = 1e-13


def build(force: bool = False) -> str:
    """Compile liboracle.so if missing or stale.  Never -ffast-math, never contraction."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_SRC3)):
        subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
                               "-o", _LIB, _SRC, _SRC3, "-lm"])
    return _LIB


_lib = None
_i64 = ctypes.c_int64
_dbl = ctypes.c_double
_ptr = ctypes.c_void_p


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.oracle_dgemm.restype = ctypes.c_int
        lib.oracle_dgemm.argtypes = [_i64, _i64, _i64, _dbl, _ptr, _i64, _ptr, _i64, _dbl, _ptr, _i64, _ptr, _i64]
        lib.oracle_dgemm_sub.restype = ctypes.c_int
        lib.oracle_dgemm_sub.argtypes = [_i64, _i64, _i64, _dbl, _ptr, _i64, _ptr, _i64, _dbl, _ptr, _i64,
                                         _i64, _ptr, _i64, _ptr, _ptr, _ptr]
        lib.oracle_partition.restype = ctypes.c_int
        lib.oracle_partition.argtypes = [_i64, _i64, _i64, _i64, ctypes.POINTER(_i64), ctypes.POINTER(_i64)]
        lib.oracle_dtrsm.restype = ctypes.c_int
        lib.oracle_dtrsm.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, _i64, _i64, _dbl, _ptr, _i64, _ptr, _i64]
        lib.oracle_dtrsm_residual.restype = ctypes.c_int
        lib.oracle_dtrsm_residual.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, _i64, _i64, _dbl, _ptr, _i64, _ptr, _i64,
                                              _ptr, _i64, _i64, _ptr, _i64, _ptr, _ptr, _ptr]
        lib.oracle_dtrsm_right.restype = ctypes.c_int
        lib.oracle_dtrsm_right.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, _i64, _i64, _dbl, _ptr, _i64, _ptr, _i64]
        lib.oracle_dtrmm.restype = ctypes.c_int
        lib.oracle_dtrmm.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, _i64, _i64, _dbl, _ptr, _i64, _ptr, _i64]
        lib.oracle_dpotrf.restype = ctypes.c_int
        lib.oracle_dpotrf.argtypes = [ctypes.c_int, _i64, _ptr, _i64, ctypes.POINTER(_i64)]
        lib.oracle_dpotrf_residual.restype = ctypes.c_int
        lib.oracle_dpotrf_residual.argtypes = [ctypes.c_int, _i64, _ptr, _i64, _ptr, _i64, _i64, _ptr, _i64, _ptr, _ptr, _ptr]
        lib.oracle_dgetrf.restype = ctypes.c_int
        lib.oracle_dgetrf.argtypes = [_i64, _i64, _ptr, _i64, _ptr, ctypes.POINTER(_i64)]
        lib.oracle_dgetrf_residual.restype = ctypes.c_int
        lib.oracle_dgetrf_residual.argtypes = [_i64, _i64, _ptr, _i64, _ptr, _i64, _ptr, _i64, _ptr, _i64, _ptr, _ptr, _ptr]
        _lib = lib
    return _lib


def _chk2d(x, name):
    assert isinstance(x, np.ndarray) and x.dtype == np.float64 and x.ndim == 2 and x.strides[1] == 8 \
        and x.strides[0] % 8 == 0, f"{name}: need a row-major float64 2-D array"
    return x.ctypes.data, x.strides[0] // 8


def dgemm_ptr(M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, D=0, ldd=0) -> None:
    """Raw-address form (host pointers as ints), for multi-GB buffers not owned by numpy."""
    rc = _load().oracle_dgemm(M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, D or None, ldd)
    if rc != 0:
        raise RuntimeError(f"oracle_dgemm failed: {rc}")


def dgemm(alpha, A, B, beta, C, want_denominator=False):
    """C <- alpha*A*B + beta*C in place (numpy row-major views; M, N, K from C and A).
    Returns D (the tolerance denominator) when asked, else None."""
    M, N = C.shape
    K = A.shape[1] if A is not None else 0
    cp, ldc = _chk2d(C, "C")
    ap, lda = _chk2d(A, "A") if A is not None and A.size else (None, max(K, 1))
    bp, ldb = _chk2d(B, "B") if B is not None and B.size else (None, max(N, 1))
    if A is not None and A.size:
        assert A.shape[0] == M and B.shape == (K, N)
    D = np.empty((M, N)) if want_denominator else None
    rc = _load().oracle_dgemm(M, N, K, alpha, ap, lda, bp, ldb, beta, cp, ldc,
                              D.ctypes.data if D is not None else None, N)
    if rc != 0:
        raise RuntimeError(f"oracle_dgemm failed: {rc}")
    return D


def dgemm_sub_ptr(M, N, K, alpha, A, lda, B, ldb, beta, C0, ldc, rows=None, cols=None,
                  want_denominator=True):
    """Sampled outputs from raw host addresses: the sub-matrix rows x cols of the updated C (dense),
    plus its denominator.  rows/cols: 1-D int arrays or None for all."""
    rows_a = None if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
    cols_a = None if cols is None else np.ascontiguousarray(cols, dtype=np.int64)
    nr = M if rows_a is None else rows_a.size
    nc = N if cols_a is None else cols_a.size
    out = np.empty((nr, nc))
    dout = np.empty((nr, nc)) if want_denominator else None
    rc = _load().oracle_dgemm_sub(M, N, K, alpha, A or None, lda, B or None, ldb, beta, C0 or None, ldc,
                                  nr, rows_a.ctypes.data if rows_a is not None else None,
                                  nc, cols_a.ctypes.data if cols_a is not None else None,
                                  out.ctypes.data, dout.ctypes.data if dout is not None else None)
    if rc != 0:
        raise RuntimeError(f"oracle_dgemm_sub failed: {rc}")
    return out, dout


def dgemm_sub(alpha, A, B, beta, C0, rows=None, cols=None, want_denominator=True):
    """numpy-view form of dgemm_sub_ptr; C0 may be None when beta == 0."""
    M, K = A.shape
    N = B.shape[1]
    ap, lda = _chk2d(A, "A") if A.size else (0, max(K, 1))
    bp, ldb = _chk2d(B, "B") if B.size else (0, max(N, 1))
    cp, ldc = _chk2d(C0, "C0") if C0 is not None else (0, N)
    return dgemm_sub_ptr(M, N, K, alpha, ap, lda, bp, ldb, beta, cp, ldc, rows, cols, want_denominator)


def dsyrk(uplo, trans, alpha, A, beta, C, want_denominator=False):
    """The DSYRK definition on one triangle of C, in place (the BLAS operation the paper names as future work):
        trans = 0: C_ij <- alpha * sum_k A_ik A_jk + beta * C_ij   (A is N x K)
        trans = 1: C_ij <- alpha * sum_k A_ki A_kj + beta * C_ij   (A is K x N)
    for j <= i (uplo = 0, lower) or j >= i (uplo = 1, upper); the other triangle is not referenced and keeps its bits.
    It IS the DGEMM definition with op(B) = op(A)^T restricted to a triangle, so the step is `dgemm` above on a written-out
    transpose (a copy, no arithmetic), then the triangle is taken.  Returns D on the triangle (0 elsewhere) when asked."""
    N = C.shape[0]
    assert C.shape == (N, N)
    opA = np.empty((N, A.shape[0] if trans else A.shape[1]))
    opA[...] = A.T if trans else A
    opAt = np.empty((opA.shape[1], N))
    opAt[...] = opA.T
    full = C.copy()
    D = dgemm(alpha, opA, opAt, beta, full, want_denominator=want_denominator)
    keep = np.tril(np.ones((N, N), dtype=bool)) if uplo == 0 else np.triu(np.ones((N, N), dtype=bool))
    C[keep] = full[keep]
    if D is not None:
        D[~keep] = 0.0
    return D


def dsyr2k(uplo, trans, alpha, A, B, beta, C, want_denominator=False):
    """The DSYR2K definition on one triangle of C, in place, as two DGEMM definitions in sequence:
        C_ij <- (alpha * sum_k a_ik b_jk + beta * C_ij),  then  C_ij <- alpha * sum_k b_ik a_jk + C_ij      (trans = 0)
    (A, B are N x K; trans = 1: A, B are K x N and the sums run over a_ki b_kj, b_ki a_kj).  The other triangle keeps its bits.
    D = |alpha| sum_k (|a_ik||b_jk| + |b_ik||a_jk|) + |beta||C0_ij| on the triangle when asked."""
    N = C.shape[0]
    opA, opB = np.empty((N, A.shape[0] if trans else A.shape[1])), np.empty((N, B.shape[0] if trans else B.shape[1]))
    opA[...] = A.T if trans else A
    opB[...] = B.T if trans else B
    opAt, opBt = np.empty(opA.shape[::-1]), np.empty(opB.shape[::-1])
    opAt[...] = opA.T
    opBt[...] = opB.T
    full = C.copy()
    D1 = dgemm(alpha, opA, opBt, beta, full, want_denominator=want_denominator)
    mid = full.copy() if want_denominator else None
    D2 = dgemm(alpha, opB, opAt, 1.0, full, want_denominator=want_denominator)
    keep = np.tril(np.ones((N, N), dtype=bool)) if uplo == 0 else np.triu(np.ones((N, N), dtype=bool))
    C[keep] = full[keep]
    if not want_denominator:
        return None
    D = D1 + (D2 - np.abs(mid))          # D2 = |alpha| sum |b||a| + |1||mid|: take the product part, keep D1's |beta||C0|
    D[~keep] = 0.0
    return D


def dtrsm(uplo, trans, unit, alpha, A, B):
    """Solve op(T) X = alpha B by substitution (oracle_dtrsm: the definition, PAPER.md:412 names the routine), X overwrites B.
    T = the `uplo` (0 lower, 1 upper) triangle of the square row-major A, op = transpose when trans, unit diagonal when unit."""
    M, N = B.shape
    assert A.shape == (M, M) or alpha == 0.0
    ap, lda = _chk2d(A, "A") if A is not None and A.size else (0, max(M, 1))
    bp, ldb = _chk2d(B, "B") if B.size else (0, max(N, 1))
    rc = _load().oracle_dtrsm(int(uplo), int(trans), int(unit), M, N, float(alpha), ap, lda, bp, ldb)
    if rc != 0:
        raise ValueError("oracle_dtrsm: bad argument")


# gate for a triangular solve of order M (reading G23): substitution in any summation order leaves a residual
# |b' - op(T) x| <= gamma_M |op(T)||x| elementwise, gamma_n = n u / (1 - n u), u = 2^-53 (Higham thm 8.5); forming b' = alpha*b
# is one more rounding and the kernel multiplies by a rounded reciprocal of t_ii instead of dividing (one more), so the gate is
#     |alpha b - op(T) x| <= gamma_(M+2) (|alpha b| + |op(T)||x|)        -- this function returns gamma_(M+2).
# Pinned by tests/test_oracle_pins.py::test_dtrsm_gate_is_gamma_m_plus_2 (the closed form in exact rational arithmetic, and
# that oracle.dtrsm's own solutions sit inside it while a one-ulp-per-row perturbation of a long solve does not).
def dtrsm_gate(M: int) -> float:
    u = 2.0 ** -53
    return (M + 2) * u / (1.0 - (M + 2) * u)


def dtrsm_residual(uplo, trans, unit, alpha, A, B0, X, rows=None, cols=None):
    """(res, den) of oracle_dtrsm_residual on the sampled rows x cols (None: all), computed in long double."""
    M, N = B0.shape
    ap, lda = _chk2d(A, "A")
    bp, ldb = _chk2d(B0, "B0")
    xp, ldx = _chk2d(X, "X")
    r = None if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
    c = None if cols is None else np.ascontiguousarray(cols, dtype=np.int64)
    nr, nc = (M if r is None else r.size), (N if c is None else c.size)
    res, den = np.empty((nr, nc)), np.empty((nr, nc))
    rc = _load().oracle_dtrsm_residual(int(uplo), int(trans), int(unit), M, N, float(alpha), ap, lda, bp, ldb, xp, ldx,
                                       nr, 0 if r is None else r.ctypes.data, nc, 0 if c is None else c.ctypes.data,
                                       res.ctypes.data, den.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_dtrsm_residual: bad argument")
    return res, den


def dtrsm_right(uplo, trans, unit, alpha, A, B):
    """Solve X op(T) = alpha B by substitution along each row (oracle_dtrsm_right: the definition), X overwrites B (M x N);
    T = the `uplo` (0 lower, 1 upper) triangle of the N x N row-major A."""
    M, N = B.shape
    assert A.shape == (N, N) or alpha == 0.0
    ap, lda = _chk2d(A, "A") if A is not None and A.size else (0, max(N, 1))
    bp, ldb = _chk2d(B, "B") if B.size else (0, max(N, 1))
    rc = _load().oracle_dtrsm_right(int(uplo), int(trans), int(unit), M, N, float(alpha), ap, lda, bp, ldb)
    if rc != 0:
        raise ValueError("oracle_dtrsm_right: bad argument")


def dtrmm(side, uplo, trans, unit, alpha, A, B):
    """B <- alpha op(T) B (side = 0) or alpha B op(T) (side = 1), in place (oracle_dtrmm: the definition from the original B)."""
    M, N = B.shape
    n = M if side == 0 else N
    assert A.shape == (n, n) or alpha == 0.0
    ap, lda = _chk2d(A, "A") if A is not None and A.size else (0, max(n, 1))
    bp, ldb = _chk2d(B, "B") if B.size else (0, max(N, 1))
    rc = _load().oracle_dtrmm(int(side), int(uplo), int(trans), int(unit), M, N, float(alpha), ap, lda, bp, ldb)
    if rc != 0:
        raise ValueError(f"oracle_dtrmm failed: {rc}")


def dsymm(side, uplo, alpha, A, B, beta, C, want_denominator=False):
    """The DSYMM definition, in place:  C <- alpha*S*B + beta*C (side = 0, S is M x M) or alpha*B*S + beta*C (side = 1, S is
    N x N), where S is the symmetric matrix whose `uplo` triangle is stored in A (the other triangle of A is never read).
    It IS the DGEMM definition on the written-out symmetric matrix (mirroring the triangle is a copy, no arithmetic), so the step
    is `dgemm` above: sums over k in increasing order, s_ik taken from the triangle at (max, min) or (min, max)."""
    n = A.shape[0]
    tri = np.tril(A) if uplo == 0 else np.triu(A)
    other = np.tril(A, -1).T if uplo == 0 else np.triu(A, 1).T
    S = np.empty((n, n))
    S[...] = tri
    mask = np.triu(np.ones((n, n), dtype=bool), 1) if uplo == 0 else np.tril(np.ones((n, n), dtype=bool), -1)
    S[mask] = other[mask]
    Bc = np.ascontiguousarray(B)
    return dgemm(alpha, S, Bc, beta, C, want_denominator) if side == 0 else dgemm(alpha, Bc, S, beta, C, want_denominator)


def dpotrf(uplo, A):
    """Cholesky-Banachiewicz on the `uplo` triangle of the square row-major A, in place (oracle_dpotrf: the definition).
    Returns LAPACK's info: 0, or i+1 when the leading minor of order i+1 is not positive definite (the routine stops there)."""
    N = A.shape[0]
    assert A.shape == (N, N)
    ap, lda = _chk2d(A, "A") if A.size else (0, 1)
    info = _i64(0)
    rc = _load().oracle_dpotrf(int(uplo), N, ap, lda, ctypes.byref(info))
    if rc != 0:
        raise ValueError("oracle_dpotrf: bad argument")
    return int(info.value)


# gate for a Cholesky factorization of order N (reading G24): the computed factor of ANY summation order satisfies
# |A - L L^T| <= gamma_(N+1) |L||L^T| elementwise (Higham thm 10.3); the CUDA path multiplies by a rounded reciprocal of l_jj
# instead of dividing (one more rounding per element), so the gate is gamma_(N+2) -- this function returns gamma_(N+2).
def dpotrf_gate(N: int) -> float:
    u = 2.0 ** -53
    return (N + 2) * u / (1.0 - (N + 2) * u)


def dpotrf_residual(uplo, A0, F, rows=None, cols=None):
    """(res, den) of oracle_dpotrf_residual on the sampled rows x cols (None: all): |a_ij - sum_k f_ik f_jk| and
    sum_k |f_ik||f_jk| in long double, A0 = the original matrix (its `uplo` triangle), F = the candidate factor."""
    N = A0.shape[0]
    ap, lda = _chk2d(A0, "A0")
    fp, ldf = _chk2d(F, "F")
    r = None if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
    c = None if cols is None else np.ascontiguousarray(cols, dtype=np.int64)
    nr, nc = (N if r is None else r.size), (N if c is None else c.size)
    res, den = np.empty((nr, nc)), np.empty((nr, nc))
    rc = _load().oracle_dpotrf_residual(int(uplo), N, ap, lda, fp, ldf, nr, 0 if r is None else r.ctypes.data,
                                        nc, 0 if c is None else c.ctypes.data, res.ctypes.data, den.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_dpotrf_residual: bad argument")
    return res, den


def dgetrf(A):
    """LU factorization with partial pivoting of the row-major M x N matrix A, in place (oracle_dgetrf: Gaussian elimination
    column by column, first maximum as the pivot).  Returns (ipiv, info): ipiv[j] = the row (0-based) exchanged with row j,
    j < min(M, N); info = 0, or j+1 for the first exactly-zero pivot."""
    M, N = A.shape
    ap, lda = _chk2d(A, "A") if A.size else (0, 1)
    ipiv = np.zeros(min(M, N), dtype=np.int64)
    info = _i64(0)
    rc = _load().oracle_dgetrf(M, N, ap, lda, ipiv.ctypes.data if ipiv.size else 0, ctypes.byref(info))
    if rc != 0:
        raise ValueError("oracle_dgetrf: bad argument")
    return ipiv, int(info.value)


# gate for an LU factorization with n = min(M, N) pivots (reading G27): the computed factors of Gaussian elimination in
# ANY order of its operations satisfy |P A - L U| <= gamma_n |L||U| elementwise (Higham thm 9.3; partitioned LU with conventional
# matrix products keeps the bound, Higham section 13.2).
def dgetrf_gate(n: int) -> float:
    u = 2.0 ** -53
    return n * u / (1.0 - n * u)


def dgetrf_residual(A0, F, ipiv, rows=None, cols=None):
    """(res, den) of oracle_dgetrf_residual on the sampled rows x cols (None: all): |(P A0)_ij - sum_k l_ik u_kj| and
    sum_k |l_ik||u_kj| in long double; A0 = the original matrix, F = the candidate factors (L below the diagonal, unit diagonal
    not stored, U on and above it), ipiv = the candidate interchanges (0-based)."""
    M, N = A0.shape
    ap, lda = _chk2d(A0, "A0")
    fp, ldf = _chk2d(F, "F")
    ip = np.ascontiguousarray(ipiv, dtype=np.int64)
    assert ip.size == min(M, N)
    r = None if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
    c = None if cols is None else np.ascontiguousarray(cols, dtype=np.int64)
    nr, nc = (M if r is None else r.size), (N if c is None else c.size)
    res, den = np.empty((nr, nc)), np.empty((nr, nc))
    rc = _load().oracle_dgetrf_residual(M, N, ap, lda, fp, ldf, ip.ctypes.data, nr, 0 if r is None else r.ctypes.data,
                                        nc, 0 if c is None else c.ctypes.data, res.ctypes.data, den.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_dgetrf_residual: bad argument (an interchange out of range?)")
    return res, den


def partition(M, N, K, S):
    """(h, w) of the paper's hclMatrixPartitioner rule by enumeration, or None if nothing fits."""
    h, w = _i64(), _i64()
    rc = _load().oracle_partition(M, N, K, S, ctypes.byref(h), ctypes.byref(w))
    if rc == 1:
        return None
    if rc != 0:
        raise ValueError("oracle_partition: bad argument")
    return h.value, w.value


def within_gate(C_test: np.ndarray, C_ref: np.ndarray, D: np.ndarray, rtol: float = RTOL):
    """Elementwise gate |C_test - C_ref| <= rtol * D (G14).  Returns (ok, worst ratio)."""
    err = np.abs(C_test - C_ref)
    bad = ~(err <= rtol * D)          # NaN-safe: NaN fails
    with np.errstate(divide="ignore", invalid="ignore"):
        ratio = np.where(D > 0, err / D, np.where(err == 0, 0.0, np.inf))
    return (not bad.any()), float(np.nanmax(ratio)) if ratio.size else 0.0
