/* level3_oracle.c -- TEST INFRASTRUCTURE ONLY.  CPU oracles for the routines the paper names as future work on top of
 * the out-of-core DGEMM ("full support for level-3 BLAS kernels" and "out-of-core factorizations (LU, QR,
 * Cholesky) that use the out-of-core matrix-matrix multiplication (DGEMM) as a fundamental building block"):
 *
 *     oracle_dtrsm_right   X * op(T) = alpha * B                                  (DTRSM, side = Right)
 *     oracle_dtrmm         B := alpha * op(T) * B   or   B := alpha * B * op(T)    (DTRMM, both sides)
 *     oracle_dpotrf        A = L * L^T  or  A = U^T * U                            (Cholesky factorization, DPOTRF)
 *     oracle_dpotrf_residual   |A - L L^T| and |L||L^T| on sampled entries, in long double
 *     oracle_dgetrf        P * A = L * U                                           (LU factorization with partial pivoting, DGETRF)
 *     oracle_dgetrf_residual   |P A - L U| and |L||U| on sampled entries, in long double
 *
 * The paper gives no algorithm for any of them, so each oracle is the plain textbook DEFINITION written out element by element
 * (row-major storage, leading dimensions in elements, FP64, every product rounded and then added or subtracted: compiled with
 * -ffp-contract=off, never -ffast-math), in the BLAS / LAPACK argument conventions the names imply (readings G24-G26):
 * only the `uplo` triangle of a triangular or symmetric operand is referenced; a unit diagonal is not read; the part of a
 * matrix an operation does not define keeps its bits.
 *
 * Independence: shares no code, header, constant or helper with the CUDA path under paper_1808_05056_b200/; only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.  Pins: tests/test_oracle_level3.py
 * (pure-Python brute force in the same operation order, exact integer / rational cases, scipy cross-checks, closed forms,
 * textbook worked examples, NaN-poisoned unreferenced parts) -- nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* op(T)[i][k] of the triangular operand stored row-major in A */
static inline double l3_tri_at(const double* A, int64_t lda, int trans, int64_t i, int64_t k) {
    return trans ? A[k * lda + i] : A[i * lda + k];
}

/* ------------------------------------------------------------------------------------------------------------------
 * DTRSM, side = Right:  solve  X * op(T) = alpha * B  for X  (B is M x N row-major and is overwritten by X; T = the `uplo`
 * triangle of the N x N matrix A, lda >= N; op(T) = T or T^T; unit = 1: the diagonal is taken as 1 and not read).
 * Every row of B is an independent system  op(T)^T x^T = alpha b^T; substitution along the row (Golub & Van Loan 3.1):
 *     op(T) upper:  x_ij = (alpha*b_ij - sum_{k<j} x_ik t_kj) / t_jj,   j = 0 .. N-1,   k increasing
 *     op(T) lower:  x_ij = (alpha*b_ij - sum_{k>j} x_ik t_kj) / t_jj,   j = N-1 .. 0,   k decreasing from N-1
 * with t_kj = op(T)_kj.  alpha == 0: X = 0, A not read.  Returns 0, -1 on a bad argument. */
int oracle_dtrsm_right(int uplo, int trans, int unit, int64_t M, int64_t N, double alpha, const double* A, int64_t lda,
                       double* B, int64_t ldb) {
    if ((uplo != 0 && uplo != 1) || (trans != 0 && trans != 1) || (unit != 0 && unit != 1)) return -1;
    if (M < 0 || N < 0) return -1;
    if (M == 0 || N == 0) return 0;
    if (!B || ldb < N) return -1;
    if (alpha == 0.0) {
        for (int64_t i = 0; i < M; ++i) for (int64_t j = 0; j < N; ++j) B[i * ldb + j] = 0.0;
        return 0;
    }
    if (!A || lda < N) return -1;
    const int upper = (uplo == 1) != (trans != 0);          /* op(T) is upper triangular */
    #pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < M; ++i) {
        double* b = B + i * ldb;
        if (upper) {
            for (int64_t j = 0; j < N; ++j) {
                double x = alpha * b[j];
                for (int64_t k = 0; k < j; ++k) { const double p = b[k] * l3_tri_at(A, lda, trans, k, j); x = x - p; }
                if (!unit) x = x / l3_tri_at(A, lda, trans, j, j);
                b[j] = x;
            }
        } else {
            for (int64_t j = N - 1; j >= 0; --j) {
                double x = alpha * b[j];
                for (int64_t k = N - 1; k > j; --k) { const double p = b[k] * l3_tri_at(A, lda, trans, k, j); x = x - p; }
                if (!unit) x = x / l3_tri_at(A, lda, trans, j, j);
                b[j] = x;
            }
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------------
 * DTRMM:  B := alpha * op(T) * B  (side = 0, Left: T is M x M)  or  B := alpha * B * op(T)  (side = 1, Right: T is N x N),
 * B is M x N row-major, T = the `uplo` triangle of A (the other triangle is never read, nor the diagonal when unit = 1).
 * The definition element by element, from the ORIGINAL B:
 *     left :  b'_ij = alpha * sum_k op(T)_ik b_kj     right:  b'_ij = alpha * sum_k b_ik op(T)_kj
 * the sum over the k inside the triangle in increasing order, every product rounded and then added to an accumulator that
 * starts at +0.0; a unit diagonal contributes b itself (no multiplication); then one multiplication by alpha.
 * alpha == 0: B = 0, A not read.  Returns 0, -1 on a bad argument, -2 if scratch memory is unavailable. */
int oracle_dtrmm(int side, int uplo, int trans, int unit, int64_t M, int64_t N, double alpha, const double* A, int64_t lda,
                 double* B, int64_t ldb) {
    if ((side != 0 && side != 1) || (uplo != 0 && uplo != 1) || (trans != 0 && trans != 1) || (unit != 0 && unit != 1)) return -1;
    if (M < 0 || N < 0) return -1;
    if (M == 0 || N == 0) return 0;
    if (!B || ldb < N) return -1;
    if (alpha == 0.0) {
        for (int64_t i = 0; i < M; ++i) for (int64_t j = 0; j < N; ++j) B[i * ldb + j] = 0.0;
        return 0;
    }
    const int64_t n = side == 0 ? M : N;
    if (!A || lda < n) return -1;
    double* B0 = (double*)malloc((size_t)M * (size_t)N * sizeof(double));
    if (!B0) return -2;
    for (int64_t i = 0; i < M; ++i) memcpy(B0 + i * N, B + i * ldb, (size_t)N * sizeof(double));
    const int lower = (uplo == 0) != (trans != 0);          /* op(T) is lower triangular */
    #pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < M; ++i) {
        for (int64_t j = 0; j < N; ++j) {
            double acc = 0.0;
            if (side == 0) {       /* sum_k op(T)_ik b_kj: k <= i (lower) or k >= i (upper) */
                const int64_t k0 = lower ? 0 : i, k1 = lower ? i : M - 1;
                for (int64_t k = k0; k <= k1; ++k) {
                    const double p = (k == i && unit) ? B0[k * N + j] : l3_tri_at(A, lda, trans, i, k) * B0[k * N + j];
                    acc = acc + p;
                }
            } else {               /* sum_k b_ik op(T)_kj: k >= j (lower) or k <= j (upper) */
                const int64_t k0 = lower ? j : 0, k1 = lower ? N - 1 : j;
                for (int64_t k = k0; k <= k1; ++k) {
                    const double p = (k == j && unit) ? B0[i * N + k] : B0[i * N + k] * l3_tri_at(A, lda, trans, k, j);
                    acc = acc + p;
                }
            }
            B[i * ldb + j] = alpha * acc;
        }
    }
    free(B0);
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------------
 * DPOTRF: the Cholesky factorization of a symmetric positive definite N x N matrix held in its `uplo` triangle,
 *     uplo = 0 (lower):  A = L * L^T,  L lower triangular with positive diagonal, overwrites the lower triangle
 *     uplo = 1 (upper):  A = U^T * U,  U upper triangular with positive diagonal, overwrites the upper triangle
 * (the other triangle is neither read nor written).  The Cholesky-Banachiewicz definition, row by row (lower) -- for upper
 * the same recurrences with the roles of the two indices exchanged, i.e. column by column of U^T:
 *     lower:  for i = 0 .. N-1:   for j = 0 .. i-1:  l_ij = (a_ij - sum_{k<j} l_ik l_jk) / l_jj
 *                                 s = a_ii - sum_{k<i} l_ik^2;   l_ii = sqrt(s)
 *     upper:  for i = 0 .. N-1:   for j = 0 .. i-1:  u_ji = (a_ji - sum_{k<j} u_ki u_kj) / u_jj
 *                                 s = a_ii - sum_{k<i} u_ki^2;   u_ii = sqrt(s)
 * sums over k in increasing order, every product rounded and then subtracted.  LAPACK's `info` convention: if some s is not
 * positive (s <= 0, or NaN) the leading minor of order i+1 is not positive definite: *info = i+1 and the routine stops, leaving
 * rows 0 .. i-1 of the factor (and the off-diagonal part of row i) in place; otherwise *info = 0.
 * Returns 0 (also when *info > 0), -1 on a bad argument. */
int oracle_dpotrf(int uplo, int64_t N, double* A, int64_t lda, int64_t* info) {
    if ((uplo != 0 && uplo != 1) || N < 0 || !info) return -1;
    *info = 0;
    if (N == 0) return 0;
    if (!A || lda < N) return -1;
    #define F(i, j) (uplo == 0 ? A[(i) * lda + (j)] : A[(j) * lda + (i)])      /* factor entry (i, j), j <= i, as stored */
    for (int64_t i = 0; i < N; ++i) {
        for (int64_t j = 0; j < i; ++j) {
            double s = F(i, j);
            for (int64_t k = 0; k < j; ++k) { const double p = F(i, k) * F(j, k); s = s - p; }
            s = s / F(j, j);
            if (uplo == 0) A[i * lda + j] = s; else A[j * lda + i] = s;
        }
        double s = A[i * lda + i];
        for (int64_t k = 0; k < i; ++k) { const double p = F(i, k) * F(i, k); s = s - p; }
        if (!(s > 0.0)) { *info = i + 1; return 0; }
        A[i * lda + i] = sqrt(s);
    }
    #undef F
    return 0;
}

/* Backward residual of a candidate Cholesky factor on sampled entries of the referenced triangle, in long double:
 *     res[r*nc + c] = | a_ij - sum_k f_ik f_jk |,    den[r*nc + c] = sum_k |f_ik||f_jk|,     k = 0 .. min(i, j)
 * for i = rows[r] (NULL: r), j = cols[c] (NULL: c), with f = L (uplo = 0; f_ik = F[i][k]) or f = U^T (uplo = 1; f_ik = F[k][i]),
 * and a_ij read from the `uplo` triangle of A0 (the entry (max, min) or (min, max)).  Cholesky in ANY order of summation
 * satisfies |A - L L^T| <= gamma_(n+1) |L||L^T| elementwise (Higham, Accuracy and Stability, thm 10.3), which is the gate of
 * the parity tests (G24). */
int oracle_dpotrf_residual(int uplo, int64_t N, const double* A0, int64_t lda, const double* F, int64_t ldf,
                           int64_t nr, const int64_t* rows, int64_t nc, const int64_t* cols, double* res, double* den) {
    if ((uplo != 0 && uplo != 1) || N < 0 || nr < 0 || nc < 0) return -1;
    if (nr == 0 || nc == 0) return 0;
    if (!A0 || !F || !res || !den || lda < N || ldf < N) return -1;
    for (int64_t r = 0; r < nr; ++r) { int64_t i = rows ? rows[r] : r; if (i < 0 || i >= N) return -1; }
    for (int64_t c = 0; c < nc; ++c) { int64_t j = cols ? cols[c] : c; if (j < 0 || j >= N) return -1; }
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t r = 0; r < nr; ++r) {
        const int64_t i = rows ? rows[r] : r;
        for (int64_t c = 0; c < nc; ++c) {
            const int64_t j = cols ? cols[c] : c;
            const int64_t hi = i > j ? i : j, lo = i > j ? j : i;
            const long double a = uplo == 0 ? (long double)A0[hi * lda + lo] : (long double)A0[lo * lda + hi];
            long double s = a, d = 0.0L;
            for (int64_t k = 0; k <= lo; ++k) {
                const long double fi = uplo == 0 ? (long double)F[i * ldf + k] : (long double)F[k * ldf + i];
                const long double fj = uplo == 0 ? (long double)F[j * ldf + k] : (long double)F[k * ldf + j];
                s -= fi * fj;
                d += fabsl(fi) * fabsl(fj);
            }
            res[r * nc + c] = (double)fabsl(s);
            den[r * nc + c] = (double)d;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------------
 * DGETRF: the LU factorization with partial pivoting (row interchanges) of a general M x N matrix (PAPER.md:412 names
 * "LU" first among the out-of-core factorizations to be built on the DGEMM; reading G27 in DESIGN.md):
 *     P * A = L * U,    L  M x min(M,N) unit lower trapezoidal (|l_ij| <= 1),   U  min(M,N) x N upper trapezoidal,
 * L (without its unit diagonal) and U overwrite A.  The textbook definition, Gaussian elimination column by column
 * (Golub & Van Loan, Matrix Computations, alg. 3.4.1; LAPACK's unblocked DGETF2 is the same recurrences):
 *     for j = 0 .. min(M,N)-1:
 *         p = the SMALLEST i >= j with |a_ij| = max_{i >= j} |a_ij|                 (the first maximum, as IDAMAX)
 *         ipiv[j] = p  (0-based; LAPACK's is 1-based);  exchange rows j and p of the whole matrix (all N columns)
 *         if a_jj == 0:  *info = j+1 unless it is set already; next j   (the column is zero from row j down: nothing to eliminate)
 *         for i > j:   a_ij = a_ij / a_jj;    for k > j:  a_ik = a_ik - a_ij * a_jk     (product rounded, then subtracted)
 * *info = 0, or j+1 for the first exactly-zero pivot u_jj (the factorization is completed all the same, as in LAPACK; U is
 * then singular).  NaN entries: unspecified.  Returns 0 (also when *info > 0), -1 on a bad argument. */
int oracle_dgetrf(int64_t M, int64_t N, double* A, int64_t lda, int64_t* ipiv, int64_t* info) {
    if (M < 0 || N < 0 || !info) return -1;
    *info = 0;
    if (M == 0 || N == 0) return 0;
    if (!A || lda < N || !ipiv) return -1;
    const int64_t n = M < N ? M : N;
    for (int64_t j = 0; j < n; ++j) {
        int64_t p = j;
        double best = fabs(A[j * lda + j]);
        for (int64_t i = j + 1; i < M; ++i) {
            const double v = fabs(A[i * lda + j]);
            if (v > best) { best = v; p = i; }
        }
        ipiv[j] = p;
        if (p != j)
            for (int64_t k = 0; k < N; ++k) { const double t = A[j * lda + k]; A[j * lda + k] = A[p * lda + k]; A[p * lda + k] = t; }
        const double piv = A[j * lda + j];
        if (piv == 0.0) { if (*info == 0) *info = j + 1; continue; }
        for (int64_t i = j + 1; i < M; ++i) {
            const double l = A[i * lda + j] / piv;
            A[i * lda + j] = l;
            for (int64_t k = j + 1; k < N; ++k) { const double prod = l * A[j * lda + k]; A[i * lda + k] = A[i * lda + k] - prod; }
        }
    }
    return 0;
}

/* Backward residual of a candidate LU factorization on sampled entries, in long double:
 *     res[r*nc + c] = | (P A0)_ij - sum_k l_ik u_kj |,    den[r*nc + c] = sum_k |l_ik||u_kj|,    k = 0 .. min(i, j, min(M,N)-1)
 * for i = rows[r] (NULL: r), j = cols[c] (NULL: c); l_ik = F[i][k] for k < i, l_ii = 1, u_kj = F[k][j] for k <= j; P A0 is A0 with
 * the interchanges ipiv[0], ipiv[1], ... applied in that order (row j <-> row ipiv[j]).  Gaussian elimination in ANY order of
 * the operations satisfies |P A - L U| <= gamma_n |L||U| elementwise, n = min(M,N) (Higham, Accuracy and Stability of Numerical
 * Algorithms, thm 9.3), which is the gate of the parity tests (G27).  Returns -1 on a bad argument (also an
 * interchange out of range: ipiv[j] < j or >= M). */
int oracle_dgetrf_residual(int64_t M, int64_t N, const double* A0, int64_t lda, const double* F, int64_t ldf, const int64_t* ipiv,
                           int64_t nr, const int64_t* rows, int64_t nc, const int64_t* cols, double* res, double* den) {
    if (M < 0 || N < 0 || nr < 0 || nc < 0) return -1;
    if (nr == 0 || nc == 0) return 0;
    if (!A0 || !F || !ipiv || !res || !den || lda < N || ldf < N) return -1;
    const int64_t n = M < N ? M : N;
    for (int64_t r = 0; r < nr; ++r) { int64_t i = rows ? rows[r] : r; if (i < 0 || i >= M) return -1; }
    for (int64_t c = 0; c < nc; ++c) { int64_t j = cols ? cols[c] : c; if (j < 0 || j >= N) return -1; }
    int64_t* perm = (int64_t*)malloc((size_t)M * sizeof(int64_t));      /* row i of P A0 is row perm[i] of A0 */
    if (!perm) return -1;
    for (int64_t i = 0; i < M; ++i) perm[i] = i;
    for (int64_t j = 0; j < n; ++j) {
        const int64_t p = ipiv[j];
        if (p < j || p >= M) { free(perm); return -1; }
        const int64_t t = perm[j]; perm[j] = perm[p]; perm[p] = t;
    }
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t r = 0; r < nr; ++r) {
        const int64_t i = rows ? rows[r] : r;
        for (int64_t c = 0; c < nc; ++c) {
            const int64_t j = cols ? cols[c] : c;
            int64_t top = i < j ? i : j;
            if (top > n - 1) top = n - 1;
            long double s = (long double)A0[perm[i] * lda + j], d = 0.0L;
            for (int64_t k = 0; k <= top; ++k) {
                const long double l = k == i ? 1.0L : (long double)F[i * ldf + k];
                const long double u = (long double)F[k * ldf + j];
                s -= l * u;
                d += fabsl(l) * fabsl(u);
            }
            res[r * nc + c] = (double)fabsl(s);
            den[r * nc + c] = (double)d;
        }
    }
    free(perm);
    return 0;
}
