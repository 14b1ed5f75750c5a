/* dgemm_oracle.c -- TEST INFRASTRUCTURE ONLY.  The CPU oracle for the out-of-core DGEMM path.
 *
 * What it is: the plain definition of the operation the paper's MMOOC computes,
 *     C = alpha * A * B + beta * C,   A is M x K, B is K x N, C is M x N, FP64
 * (section V; the per-block form c_ij = alpha * a_i b_j + beta * c_ij is
 * the paper prints "a_i b_i", a typo, reading G3).  The method is exact up
 * to rounding order, so the oracle is the definition written out:
 *
 *     acc = +0.0;  for k = 0 .. K-1 in increasing order:  acc = acc + (A[i][k] * B[k][j])
 *         (product rounded to FP64, then the sum rounded to FP64; never fused)
 *     beta == 0 :  C[i][j] = alpha * acc                       (C is not read: NaN is overwritten)
 *     otherwise :  C[i][j] = alpha * acc + beta * C[i][j]      (two products and one sum, each rounded)
 *     D[i][j]   = |alpha| * sum_k |A[i][k]| * |B[k][j]| + |beta| * |C0[i][j]|   (tolerance denominator)
 *
 * Row-major storage, leading dimensions in elements, no transposes (readings G1, G2).
 * Quick returns follow the BLAS convention (readings G8-G10): M == 0 or N == 0 touches nothing;
 * alpha == 0 or K == 0 gives C = beta * C (or +0 when beta == 0) without reading A or B.
 *
 * Form: a blocked triple loop (row blocks x k panels, j innermost) accumulating into a separate
 * acc array, so every element still sums in increasing k -- bit-identical to the naive i-j-k loop.
 * OpenMP runs over row blocks only, which changes no element's operation order.  Must be compiled
 * with -ffp-contract=off and without -ffast-math (oracle/__init__.py does).
 *
 * Independence: shares no code, header, constant or helper with the CUDA path under
 * paper_1808_05056_b200/; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.  Pins: tests/test_oracle_pins.py (all functions pinned; none
 * is "parity unpinned").
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_IB 32   /* rows per block  */
#define ORACLE_KB 128  /* k per panel     */

/* epilogue for one element */
static inline double oracle_epilogue(double alpha, double acc, double beta, double c0) {
    if (beta == 0.0) return alpha * acc;
    {
        double t1 = alpha * acc;
        double t2 = beta * c0;
        return t1 + t2;
    }
}

/* Full problem.  C is updated in place.  D (M x N, leading dimension ldd) receives the tolerance
 * denominator when non-NULL.  Returns 0, -1 on bad arguments, -2 if scratch memory is unavailable. */
int oracle_dgemm(int64_t M, int64_t N, int64_t K, double alpha, const double* A, int64_t lda,
                 const double* B, int64_t ldb, double beta, double* C, int64_t ldc, double* D,
                 int64_t ldd) {
    if (M < 0 || N < 0 || K < 0) return -1;
    if (M == 0 || N == 0) return 0;
    if (!C || ldc < N || (D && ldd < N)) return -1;
    const int noab = (alpha == 0.0 || K == 0);
    if (!noab && (!A || !B || lda < K || ldb < N)) return -1;
    int err = 0;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i0 = 0; i0 < M; i0 += ORACLE_IB) {
        const int64_t ib = (M - i0 < ORACLE_IB) ? (M - i0) : ORACLE_IB;
        double* acc = (double*)malloc((size_t)ib * (size_t)N * sizeof(double));
        double* dab = D ? (double*)malloc((size_t)ib * (size_t)N * sizeof(double)) : NULL;
        if (!acc || (D && !dab)) {
            #pragma omp atomic write
            err = 1;
            free(acc); free(dab);
            continue;
        }
        for (int64_t t = 0; t < ib * N; ++t) acc[t] = 0.0;
        if (dab) for (int64_t t = 0; t < ib * N; ++t) dab[t] = 0.0;
        if (!noab) {
            for (int64_t k0 = 0; k0 < K; k0 += ORACLE_KB) {
                const int64_t kb = (K - k0 < ORACLE_KB) ? (K - k0) : ORACLE_KB;
                for (int64_t i = 0; i < ib; ++i) {
                    const double* arow = A + (i0 + i) * lda;
                    double* accrow = acc + i * N;
                    for (int64_t k = k0; k < k0 + kb; ++k) {
                        const double a = arow[k];
                        const double* brow = B + k * ldb;
                        for (int64_t j = 0; j < N; ++j) {
                            const double p = a * brow[j];
                            accrow[j] = accrow[j] + p;
                        }
                        if (dab) {
                            const double aa = fabs(a);
                            double* drow = dab + i * N;
                            for (int64_t j = 0; j < N; ++j) drow[j] = drow[j] + aa * fabs(brow[j]);
                        }
                    }
                }
            }
        }
        for (int64_t i = 0; i < ib; ++i) {
            double* crow = C + (i0 + i) * ldc;
            for (int64_t j = 0; j < N; ++j) {
                const double c0 = (beta == 0.0) ? 0.0 : crow[j];
                if (D) D[(i0 + i) * ldd + j] = fabs(alpha) * dab[i * N + j] + ((beta == 0.0) ? 0.0 : fabs(beta) * fabs(c0));
                crow[j] = oracle_epilogue(alpha, acc[i * N + j], beta, c0);
            }
        }
        free(acc); free(dab);
    }
    return err ? -2 : 0;
}

/* Sampled outputs: the nr x nc sub-matrix {rows[r]} x {cols[c]} of the updated C, written DENSE
 * (leading dimension nc) to `out`, with the denominator to `dout` when non-NULL.  rows == NULL means
 * rows 0..nr-1, cols == NULL means columns 0..nc-1.  C0 is read (when beta != 0) and not modified.
 * Same per-element operation order as oracle_dgemm. */
int oracle_dgemm_sub(int64_t M, int64_t N, int64_t K, double alpha, const double* A, int64_t lda,
                     const double* B, int64_t ldb, double beta, const double* C0, int64_t ldc,
                     int64_t nr, const int64_t* rows, int64_t nc, const int64_t* cols, double* out,
                     double* dout) {
    if (M < 0 || N < 0 || K < 0 || nr < 0 || nc < 0) return -1;
    if (nr == 0 || nc == 0) return 0;
    if (!out || (beta != 0.0 && (!C0 || ldc < N))) return -1;
    const int noab = (alpha == 0.0 || K == 0);
    if (!noab && (!A || !B || lda < K || ldb < N)) return -1;
    for (int64_t r = 0; r < nr; ++r) { int64_t i = rows ? rows[r] : r; if (i < 0 || i >= M) return -1; }
    for (int64_t c = 0; c < nc; ++c) { int64_t j = cols ? cols[c] : c; if (j < 0 || j >= N) return -1; }
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t r = 0; r < nr; ++r) {
        const int64_t i = rows ? rows[r] : r;
        double* acc = out + r * nc;
        double* dab = dout ? dout + r * nc : NULL;
        for (int64_t c = 0; c < nc; ++c) acc[c] = 0.0;
        if (dab) for (int64_t c = 0; c < nc; ++c) dab[c] = 0.0;
        if (!noab) {
            for (int64_t k = 0; k < K; ++k) {
                const double a = A[i * lda + k];
                const double* brow = B + k * ldb;
                if (cols) {
                    for (int64_t c = 0; c < nc; ++c) { const double p = a * brow[cols[c]]; acc[c] = acc[c] + p; }
                    if (dab) for (int64_t c = 0; c < nc; ++c) dab[c] = dab[c] + fabs(a) * fabs(brow[cols[c]]);
                } else {
                    for (int64_t c = 0; c < nc; ++c) { const double p = a * brow[c]; acc[c] = acc[c] + p; }
                    if (dab) for (int64_t c = 0; c < nc; ++c) dab[c] = dab[c] + fabs(a) * fabs(brow[c]);
                }
            }
        }
        for (int64_t c = 0; c < nc; ++c) {
            const int64_t j = cols ? cols[c] : c;
            const double c0 = (beta == 0.0) ? 0.0 : C0[i * ldc + j];
            if (dab) dab[c] = fabs(alpha) * dab[c] + ((beta == 0.0) ? 0.0 : fabs(beta) * fabs(c0));
            acc[c] = oracle_epilogue(alpha, acc[c], beta, c0);
        }
    }
    return 0;
}

/* The paper's hclMatrixPartitioner rule, written out by enumeration (PAPER.md:289 and the worked
 * example at :301 / Figure 3 at :281; reading G6): among EQUAL partitions (h | M, w | N)
 * whose working set  K*nb + 2*mb*K + 2*mb*nb  (one B slice, two A slices, two C blocks -- "any two
 * blocks of C in the same column") fits in S elements, take the least host-to-device traffic
 * w*M*K + K*N + M*N; ties go to the fewest steps h*w, then the smallest h.  Returns 0 and (h, w),
 * or 1 when nothing fits. */
int oracle_partition(int64_t M, int64_t N, int64_t K, int64_t S, int64_t* h_out, int64_t* w_out) {
    if (M <= 0 || N <= 0 || K <= 0 || !h_out || !w_out) return -1;
    int found = 0;
    int64_t best_h = 0, best_w = 0;
    long double best_t = 0;
    for (int64_t h = 1; h <= M; ++h) {
        if (M % h) continue;
        for (int64_t w = 1; w <= N; ++w) {
            if (N % w) continue;
            const int64_t mb = M / h, nb = N / w;
            const long double need = (long double)K * nb + 2.0L * mb * K + 2.0L * mb * nb;
            if (need > (long double)S) continue;
            const long double t = (long double)w * M * K + (long double)K * N + (long double)M * N;
            if (!found || t < best_t || (t == best_t && (h * w < best_h * best_w || (h * w == best_h * best_w && h < best_h)))) {
                found = 1; best_t = t; best_h = h; best_w = w;
            }
        }
    }
    if (!found) return 1;
    *h_out = best_h; *w_out = best_w;
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------------
 * DTRSM, side = Left (the level-3 BLAS routine the paper names as future work):
 *     solve  op(T) * X = alpha * B  for X,   T = the `uplo` triangle of the M x M matrix A (row-major, lda >= M),
 *     op(T) = T (trans = 0) or T^T (trans = 1), unit = 1: the diagonal of T is taken as 1 and not read.
 * B is M x N row-major and is overwritten by X.  Only the `uplo` triangle of A is read.  alpha == 0: X = 0, A not read.
 * The definition by substitution, written out (Golub & Van Loan alg. 3.1.1 / 3.1.2 applied to each column of B):
 *     op(T) lower:  x_ij = (alpha*b_ij - sum_{k<i} t_ik x_kj) / t_ii,   i = 0 .. M-1
 *     op(T) upper:  x_ij = (alpha*b_ij - sum_{k>i} t_ik x_kj) / t_ii,   i = M-1 .. 0
 * with t_ik = op(T)_ik; the sum runs over k in increasing order (lower) or decreasing order from M-1 (upper), each product
 * rounded, then subtracted (no FMA: compiled with -ffp-contract=off). */
static inline double tri_at(const double* A, int64_t lda, int trans, int64_t i, int64_t k) {
    return trans ? A[k * lda + i] : A[i * lda + k];
}

int oracle_dtrsm(int uplo, int trans, int unit, int64_t M, int64_t N, double alpha, const double* A, int64_t lda,
                 double* B, int64_t ldb) {
    if ((uplo != 0 && uplo != 1) || (trans != 0 && trans != 1) || (unit != 0 && unit != 1)) return -1;
    if (M < 0 || N < 0) return -1;
    if (M == 0 || N == 0) return 0;
    if (!B || ldb < N) return -1;
    if (alpha == 0.0) {
        for (int64_t i = 0; i < M; ++i) for (int64_t j = 0; j < N; ++j) B[i * ldb + j] = 0.0;
        return 0;
    }
    if (!A || lda < M) return -1;
    /* op(T) is lower when (lower, no transpose) or (upper, transpose) */
    const int lower = (uplo == 0) != (trans != 0);
    #pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < N; ++j) {
        if (lower) {
            for (int64_t i = 0; i < M; ++i) {
                double x = alpha * B[i * ldb + j];
                for (int64_t k = 0; k < i; ++k) { const double p = tri_at(A, lda, trans, i, k) * B[k * ldb + j]; x = x - p; }
                if (!unit) x = x / tri_at(A, lda, trans, i, i);
                B[i * ldb + j] = x;
            }
        } else {
            for (int64_t i = M - 1; i >= 0; --i) {
                double x = alpha * B[i * ldb + j];
                for (int64_t k = M - 1; k > i; --k) { const double p = tri_at(A, lda, trans, i, k) * B[k * ldb + j]; x = x - p; }
                if (!unit) x = x / tri_at(A, lda, trans, i, i);
                B[i * ldb + j] = x;
            }
        }
    }
    return 0;
}

/* Residual of a candidate solution X of op(T) X = alpha B on sampled entries, in long double (64-bit significand):
 *     res[r*nc + c] = | alpha*b_ij - sum_k op(T)_ik x_kj |,   den[r*nc + c] = |alpha||b_ij| + sum_k |op(T)_ik||x_kj|
 * for i = rows[r] (NULL: r), j = cols[c] (NULL: c), k over the triangle (diagonal term: 1*x_ij when unit).  Substitution in
 * ANY order of summation satisfies res <= gamma_M * sum_k|t_ik||x_kj| (Higham, Accuracy and Stability, thm 8.5), which is the
 * gate the parity tests apply to the GPU result at sizes where oracle_dtrsm itself would take too long. */
int oracle_dtrsm_residual(int uplo, int trans, int unit, int64_t M, int64_t N, double alpha, const double* A, int64_t lda,
                          const double* B0, int64_t ldb, const double* X, int64_t ldx,
                          int64_t nr, const int64_t* rows, int64_t nc, const int64_t* cols, double* res, double* den) {
    if ((uplo != 0 && uplo != 1) || (trans != 0 && trans != 1) || (unit != 0 && unit != 1)) return -1;
    if (M < 0 || N < 0 || nr < 0 || nc < 0) return -1;
    if (nr == 0 || nc == 0) return 0;
    if (!A || !B0 || !X || !res || !den || lda < M || ldb < N || ldx < N) return -1;
    const int lower = (uplo == 0) != (trans != 0);
    for (int64_t r = 0; r < nr; ++r) { int64_t i = rows ? rows[r] : r; if (i < 0 || i >= M) return -1; }
    for (int64_t c = 0; c < nc; ++c) { int64_t j = cols ? cols[c] : c; if (j < 0 || j >= N) return -1; }
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t r = 0; r < nr; ++r) {
        const int64_t i = rows ? rows[r] : r;
        const int64_t k0 = lower ? 0 : i, k1 = lower ? i : M - 1;
        for (int64_t c = 0; c < nc; ++c) {
            const int64_t j = cols ? cols[c] : c;
            long double s = (long double)alpha * (long double)B0[i * ldb + j];
            long double d = fabsl(s);
            for (int64_t k = k0; k <= k1; ++k) {
                const long double t = (k == i && unit) ? 1.0L : (long double)tri_at(A, lda, trans, i, k);
                const long double x = (long double)X[k * ldx + j];
                s -= t * x;
                d += fabsl(t) * fabsl(x);
            }
            res[r * nc + c] = (double)fabsl(s);
            den[r * nc + c] = (double)d;
        }
    }
    return 0;
}
