// blas3_ooc.cu -- the level-3 BLAS routines whose operand is a TRIANGLE of a stored matrix, on the out-of-core DGEMM pipeline
// ("full support for level-3 BLAS kernels" is the paper's future work):
//
//     hclooc_dtrmm   B := alpha * op(T) * B   or   B := alpha * B * op(T)          T = the `uplo` triangle of A
//     hclooc_dsymm   C := alpha * S * B + beta * C   or   alpha * B * S + beta * C   S symmetric, its `uplo` triangle stored in A
//
// Nothing is copied into a dense triangle or mirrored: the pipeline streams the stored matrix as it is and the tile kernel is told
// which part of op(A) or op(B) counts (dgemm_sm100.cu, MASK): a tile runs only over the k blocks that can hold counted elements
// and zeroes the rest of the blocks that cross the diagonal by a select in registers, so whatever the other triangle holds (NaN
// included) never reaches a product.  DSYMM is two such passes -- the stored triangle, then its strict part read transposed -- like
// DSYR2K; DTRMM works in place: a step reads device copies of its operands that were made before the first block of its column
// was stored, which is safe as long as K is not split into panels (a plan with K panels is refused).
#include <algorithm>
#include <chrono>
#include <cstring>
#include "executor.h"

using namespace hclooc;

namespace {

struct Reserve {
    hclooc_ctx* ctx;
    Reserve(hclooc_ctx* c, size_t bytes) : ctx(c) { c->reserved_bytes = bytes; }
    ~Reserve() { ctx->reserved_bytes = 0; }
};

void add_stats(hclooc_stats& acc, const hclooc_stats& one) {
    acc.bytes_h2d += one.bytes_h2d; acc.bytes_d2h += one.bytes_d2h; acc.n_kernels += one.n_kernels;
    acc.n_copies_h2d += one.n_copies_h2d; acc.n_copies_d2h += one.n_copies_d2h; acc.t_enqueue_s += one.t_enqueue_s;
    acc.plan = one.plan;
}

}  // namespace

extern "C" int hclooc_dtrmm(hclooc_ctx* ctx, int side, int uplo, int trans, int diag, int64_t M, int64_t N, double alpha,
                            const double* A, int64_t lda, double* B, int64_t ldb, size_t device_budget_bytes, hclooc_stats* stats) {
    const auto t_begin = std::chrono::steady_clock::now();
    if (side != HCL_SIDE_LEFT && side != HCL_SIDE_RIGHT) return -2;
    if (uplo != HCL_UPLO_LOWER && uplo != HCL_UPLO_UPPER) return -3;
    if (trans != HCL_OP_N && trans != HCL_OP_T) return -4;
    if (diag != HCL_DIAG_NONUNIT && diag != HCL_DIAG_UNIT) return -5;
    if (M < 0) return -6;
    if (N < 0) return -7;
    if (stats) std::memset(stats, 0, sizeof(*stats));
    if (M == 0 || N == 0) return HCLOOC_OK;
    const int64_t n = side == HCL_SIDE_LEFT ? M : N;
    if (alpha != 0.0) {
        if (!A) return -9;
        if (lda < n) return -10;
    }
    if (!B) return -11;
    if (ldb < N) return -12;
    if (alpha != 0.0 && overlaps(B, M, N, ldb, A, n, n, lda)) return -11;
    int rc;
    if (alpha == 0.0) {                                              // B = 0, A not referenced, NaN in B not propagated
        rc = dgemm_core(ctx, 0, 0, M, N, 0, 0.0, nullptr, 1, nullptr, 1, 0.0, B, ldb, device_budget_bytes, stats);
        return rc == -10 ? -11 : rc;
    }
    if (!ctx && (rc = default_ctx(&ctx))) return rc;
    std::lock_guard<std::mutex> lk(ctx->mu);
    HCL_CUDA(cudaSetDevice(ctx->device));
    bool dummy = true;
    if ((rc = check_resident(A, &dummy)) || (rc = check_resident(B, &dummy))) return rc;
    size_t budget = 0;
    bool own = false;
    if ((rc = resolve_budget(ctx, device_budget_bytes, &budget, &own))) return rc;
    const bool lower_op = (uplo == HCL_UPLO_LOWER) != (trans == HCL_OP_T);     // op(T) is lower triangular
    const bool unit = diag == HCL_DIAG_UNIT;
    // a unit diagonal is not read: the strict triangle multiplies, and B itself comes in as beta * C with beta = alpha
    const double beta = unit ? alpha : 0.0;
    hclooc_stats acc;
    std::memset(&acc, 0, sizeof(acc));
    DgemmExtra ex;
    if (side == HCL_SIDE_LEFT) {
        ex.in_place = true;                                                    // C is B itself
        // B := alpha op(T) B: op(A) = op(T) (M x M), op(B) = B; op(T)[r][k] counts iff k <= r (lower) / k >= r (upper), strictly for unit
        ex.amask = lower_op ? 1 : 2;
        ex.adiag = unit ? (lower_op ? -1 : 1) : 0;
        hclooc_stats one;
        rc = dgemm_core_locked(ctx, trans ? 1 : 0, 0, M, N, M, alpha, A, lda, B, ldb, beta, B, ldb, budget, &one, 0, &ex);
        if (rc) return rc == -10 ? -11 : rc;
        add_stats(acc, one);
    } else {
        // B := alpha B op(T): op(A) = B, op(B) = op(T) (N x N).  The row slices of B are operands of every column of blocks and are
        // overwritten by the first one, so B goes through the device in row bands: a band is copied up once (at most a quarter of
        // the budget) and the pipeline reads ITS rows from that copy while it stores the results over the host rows.
        ex.bmask = lower_op ? 1 : 2;                                           // op(T)[k][c] counts iff c <= k (lower) / c >= k (upper)
        ex.bdiag = unit ? (lower_op ? -1 : 1) : 0;
        const int64_t ldx = (N + 1) & ~(int64_t)1;
        int64_t Mb = (int64_t)((budget / 4) / ((size_t)ldx * 8));
        if (Mb >= 128) Mb = Mb / 128 * 128;
        if (Mb < 1) return HCLOOC_ERR_BUDGET;
        if (Mb > M) Mb = M;
        const size_t band_bytes = (((size_t)Mb * ldx * 8) + 1023) & ~(size_t)1023;
        if (own) { if ((rc = ensure_workspace(ctx, budget))) return rc; }
        uint8_t* base = (uint8_t*)ctx->workspace;
        const uintptr_t mis = (uintptr_t)base & 1023u;
        const size_t shift = mis ? 1024 - mis : 0;
        if (band_bytes + shift > ctx->workspace_bytes) return HCLOOC_ERR_BUDGET;
        double* dBand = (double*)(base + shift);
        Reserve guard(ctx, band_bytes + shift);
        for (int64_t m0 = 0; m0 < M; m0 += Mb) {
            const int64_t mb = std::min(Mb, M - m0);
            if ((rc = copy2d(dBand, (size_t)ldx * 8, B + m0 * ldb, (size_t)ldb * 8, (size_t)N * 8, (size_t)mb, ctx->s_h2d))) return rc;
            acc.bytes_h2d += (uint64_t)mb * N * 8; ++acc.n_copies_h2d;
            HCL_CUDA(cudaStreamSynchronize(ctx->s_h2d));
            hclooc_stats one;
            rc = dgemm_core_locked(ctx, 0, trans ? 1 : 0, mb, N, N, alpha, dBand, ldx, A, lda, beta, B + m0 * ldb, ldb, budget, &one, 0, &ex);
            if (rc) return rc == -10 ? -11 : rc;
            add_stats(acc, one);
        }
    }
    if (stats) {
        *stats = acc;
        stats->plan.flops = (double)M * (double)N * (double)n;
        stats->bytes_h2d = acc.bytes_h2d; stats->bytes_d2h = acc.bytes_d2h;
        stats->t_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
    }
    return HCLOOC_OK;
}

extern "C" int hclooc_dsymm(hclooc_ctx* ctx, int side, int uplo, int64_t M, int64_t N, double alpha, const double* A, int64_t lda,
                            const double* B, int64_t ldb, double beta, double* C, int64_t ldc, size_t device_budget_bytes,
                            hclooc_stats* stats) {
    const auto t_begin = std::chrono::steady_clock::now();
    if (side != HCL_SIDE_LEFT && side != HCL_SIDE_RIGHT) return -2;
    if (uplo != HCL_UPLO_LOWER && uplo != HCL_UPLO_UPPER) return -3;
    if (M < 0) return -4;
    if (N < 0) return -5;
    if (stats) std::memset(stats, 0, sizeof(*stats));
    if (M == 0 || N == 0) return HCLOOC_OK;
    const int64_t n = side == HCL_SIDE_LEFT ? M : N;
    const bool scale_only = alpha == 0.0;
    if (!scale_only) {
        if (!A) return -7;
        if (lda < n) return -8;
        if (!B) return -9;
        if (ldb < N) return -10;
    }
    if (!C) return -12;
    if (ldc < N) return -13;
    if (!scale_only && (overlaps(C, M, N, ldc, A, n, n, lda) || overlaps(C, M, N, ldc, B, M, N, ldb))) return -12;
    int rc;
    if (scale_only) {
        rc = dgemm_core(ctx, 0, 0, M, N, 0, 0.0, nullptr, 1, nullptr, 1, beta, C, ldc, device_budget_bytes, stats);
        return rc == -10 ? -12 : rc;
    }
    if (!ctx && (rc = default_ctx(&ctx))) return rc;
    std::lock_guard<std::mutex> lk(ctx->mu);
    const bool lower = uplo == HCL_UPLO_LOWER;
    hclooc_stats one, two;
    DgemmExtra ex1, ex2;
    if (side == HCL_SIDE_LEFT) {
        // pass 1: C = alpha * tri(A) * B + beta * C        (the stored triangle, diagonal included)
        // pass 2: C = alpha * stri(A)^T * B + C            (its strict part read transposed: the other half of S)
        ex1.amask = lower ? 1 : 2;
        ex2.amask = lower ? 2 : 1; ex2.adiag = lower ? 1 : -1;                  // A^T[r][k] = A[k][r] counts iff k > r (lower stored) / k < r
        rc = dgemm_core_locked(ctx, 0, 0, M, N, M, alpha, A, lda, B, ldb, beta, C, ldc, device_budget_bytes, &one, 0, &ex1);
        if (!rc) rc = dgemm_core_locked(ctx, 1, 0, M, N, M, alpha, A, lda, B, ldb, 1.0, C, ldc, device_budget_bytes, &two, 0, &ex2);
    } else {
        // C = alpha * B * S + beta * C: the triangle is op(B):  tri(A)[k][c] counts iff c <= k (lower stored) / c >= k
        ex1.bmask = lower ? 1 : 2;
        ex2.bmask = lower ? 2 : 1; ex2.bdiag = lower ? 1 : -1;                  // A^T[k][c] = A[c][k] counts iff c > k (lower stored) / c < k
        rc = dgemm_core_locked(ctx, 0, 0, M, N, N, alpha, B, ldb, A, lda, beta, C, ldc, device_budget_bytes, &one, 0, &ex1);
        if (!rc) rc = dgemm_core_locked(ctx, 0, 1, M, N, N, alpha, B, ldb, A, lda, 1.0, C, ldc, device_budget_bytes, &two, 0, &ex2);
    }
    if (rc) return rc == -10 ? -12 : rc;
    if (stats) {
        *stats = one;
        stats->bytes_h2d += two.bytes_h2d; stats->bytes_d2h += two.bytes_d2h;
        stats->n_kernels += two.n_kernels; stats->n_copies_h2d += two.n_copies_h2d; stats->n_copies_d2h += two.n_copies_d2h;
        stats->t_enqueue_s += two.t_enqueue_s;
        stats->plan.flops = 2.0 * (double)M * (double)N * (double)n;
        stats->t_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
    }
    return HCLOOC_OK;
}
