// factor.cu -- routines built ON the out-of-core DGEMM ("out-of-core factorizations (LU, QR, Cholesky) that use the
// out-of-core matrix-matrix multiplication (DGEMM) as a fundamental building block", and "full support for level-3 BLAS
// kernels"):
//
//     hclooc_dpotrf      Cholesky factorization  A = L L^T  /  A = U^T U  of a host-resident symmetric positive definite matrix
//     hclooc_dtrsm_side  DTRSM with a side argument; side = Right:  X op(T) = alpha B  (side = Left is hclooc_dtrsm)
//
// Both are LEFT-LOOKING at the out-of-core level: a panel (a block column of NB columns, or a block row for the upper factor)
// lives in device memory from its upload to the download of its final values; it first receives the contribution of everything
// factored / solved before it as ONE out-of-core DGEMM through the pipeline of executor.cu (C in device memory, the operands
// streamed from the host: 2*NB flops per 8 bytes read, so NB = 4096 is compute bound on a 55 GB/s link), then its diagonal
// block is factored / solved in device memory by recursive halving down to 128 x 128 blocks -- the flops of the recursion sit in
// tile-kernel launches (DGEMM, DSYRK with the triangle mask) and only the 128 x 128 blocks go to the latency-bound block kernels
// (potrf_sm100.cu, trsm_sm100.cu).  Right-looking would move the whole trailing matrix over the link at every step.
#include <algorithm>
#include <chrono>
#include <cstdlib>
#include <cstring>
#include <vector>
#include "executor.h"

using namespace hclooc;

namespace {

int64_t split_point(int64_t lo, int64_t hi) { return lo + ((hi - lo + 127) / 128 + 1) / 2 * 128; }

// X <- op(T)^-1 (scale X) (right = 0: X is n x w) or X <- (scale X) op(T)^-1 (right = 1: X is w x n) in device memory, T the
// n x n triangle at dT (row-major as stored, ldt even), lower = op(T) is lower triangular, trans = op(T)[r][c] is stored at
// T[c][r].  Recursive halving over 128-blocks of the triangular dimension: solve the half that comes first in the order of
// substitution, subtract its contribution from the other half with ONE tile-kernel launch, solve the other half; `scale`
// reaches every element exactly once (as beta of the first update that touches it, or in the block kernel).
int dev_trsm(int right, const double* dT, int64_t ldt, int lower, int trans, int unit, double* X, int64_t ld, int64_t w, int64_t n,
             double scale, cudaStream_t st, uint64_t* n_kernels) {
    struct Range { int64_t lo, hi; double scale; int stage; };
    std::vector<Range> stack;
    stack.push_back({0, n, scale, 0});
    // the half solved first: rows [lo, mid) of a lower op(T) on the left; on the right x_j depends on the columns BEFORE j when
    // op(T) is upper, so the first half is [lo, mid) for an upper op(T) there
    const bool low_first = right ? !lower : (lower != 0);
    while (!stack.empty()) {
        const Range r = stack.back();
        stack.pop_back();
        const int64_t len = r.hi - r.lo;
        if (len <= 128) {
            int e = launch_trsm_block(dT + r.lo * ldt + r.lo, ldt, (int)len, right ? X + r.lo : X + r.lo * ld, ld, w, lower, trans, unit, r.scale, st, right);
            if (e) return e;
            ++*n_kernels;
            continue;
        }
        const int64_t mid = split_point(r.lo, r.hi);
        const int64_t f0 = low_first ? r.lo : mid, f1 = low_first ? mid : r.hi, s0 = low_first ? mid : r.lo, s1 = low_first ? r.hi : mid;
        if (r.stage == 0) {
            stack.push_back({r.lo, r.hi, r.scale, 1});
            stack.push_back({f0, f1, r.scale, 0});
            continue;
        }
        int e;
        if (!right) {      // X[second] <- scale * X[second] - op(T)[second, first] X[first]
            const double* Tp = trans ? dT + f0 * ldt + s0 : dT + s0 * ldt + f0;
            e = launch_dgemm_tiles(s1 - s0, w, f1 - f0, -1.0, Tp, ldt, X + f0 * ld, ld, r.scale, X + s0 * ld, ld, st, 1, nullptr, trans ? 1 : 0, 0);
        } else {           // X[:, second] <- scale * X[:, second] - X[:, first] op(T)[first, second]
            const double* Tp = trans ? dT + s0 * ldt + f0 : dT + f0 * ldt + s0;
            e = launch_dgemm_tiles(w, s1 - s0, f1 - f0, -1.0, X + f0, ld, Tp, ldt, r.scale, X + s0, ld, st, 1, nullptr, 0, trans ? 1 : 0);
        }
        if (e) return e;
        ++*n_kernels;
        stack.push_back({s0, s1, 1.0, 0});
    }
    return HCLOOC_OK;
}

// Cholesky factorization of the n x n block at dA (device, ld even) on its lower (lower = 1: A = L L^T) or upper (A = U^T U)
// triangle, by recursive halving:  factor A11;  A21 <- A21 L11^-T (a right-side solve; upper: A12 <- U11^-T A12, a left-side one);
// A22 <- A22 - A21 A21^T on its triangle (the tile kernel with the triangle mask);  factor A22.
int dev_potrf(double* dA, int64_t ld, int64_t n, int lower, long long* d_info, long long info_base, cudaStream_t st, uint64_t* n_kernels) {
    if (n <= 128) {
        ++*n_kernels;
        return launch_potrf_block(dA, ld, (int)n, lower, d_info, info_base, st);
    }
    const int64_t n1 = split_point(0, n), n2 = n - n1;
    int e = dev_potrf(dA, ld, n1, lower, d_info, info_base, st, n_kernels);
    if (e) return e;
    double* A22 = dA + n1 * ld + n1;
    if (lower) {
        double* A21 = dA + n1 * ld;
        if ((e = dev_trsm(1, dA, ld, /*op(T) = L11^T is upper*/ 0, /*stored transposed*/ 1, 0, A21, ld, n2, n1, 1.0, st, n_kernels))) return e;
        e = launch_dgemm_tiles(n2, n2, n1, -1.0, A21, ld, A21, ld, 1.0, A22, ld, st, 0, nullptr, 0, 1, /*tri*/ 1, 0);
    } else {
        double* A12 = dA + n1;
        if ((e = dev_trsm(0, dA, ld, /*op(T) = U11^T is lower*/ 1, 1, 0, A12, ld, n2, n1, 1.0, st, n_kernels))) return e;
        e = launch_dgemm_tiles(n2, n2, n1, -1.0, A12, ld, A12, ld, 1.0, A22, ld, st, 0, nullptr, 1, 0, /*tri*/ 2, 0);
    }
    if (e) return e;
    ++*n_kernels;
    return dev_potrf(A22, ld, n2, lower, d_info, info_base + n1, st, n_kernels);
}

// resets ctx->reserved_bytes when the routine that set it leaves
struct Reserve {
    hclooc_ctx* ctx;
    Reserve(hclooc_ctx* c, size_t bytes) : ctx(c) { c->reserved_bytes = bytes; }
    ~Reserve() { ctx->reserved_bytes = 0; }
};

void add_stats(hclooc_stats& acc, const hclooc_stats& one, double* t_enq) {
    acc.bytes_h2d += one.bytes_h2d; acc.bytes_d2h += one.bytes_d2h; acc.n_kernels += one.n_kernels;
    acc.n_copies_h2d += one.n_copies_h2d; acc.n_copies_d2h += one.n_copies_d2h; *t_enq += one.t_enqueue_s;
}

int64_t round_even(int64_t x) { return (x + 1) & ~(int64_t)1; }
size_t round_1k(size_t x) { return (x + 1023) & ~(size_t)1023; }

// Panel width NB of hclooc_dpotrf under `budget` for an N x N matrix: the resident panel (N x NB, the tallest one) takes at
// most half the budget; 4096 where that fits, else the largest multiple of 128 (of 32 below 128) that does.
int potrf_nb(int64_t N, size_t budget, int64_t* nb_out) {
    static const int64_t nb_env = [] { const char* e = std::getenv("HCLOOC_POTRF_NB"); const long v = e ? std::atol(e) : 0; return v >= 32 ? (int64_t)(v / 32 * 32) : (int64_t)0; }();
    int64_t NB = nb_env ? nb_env : 4096;
    auto fits = [&](int64_t nb) { return round_1k((size_t)N * round_even(nb) * 8) + 2048 <= budget / 2; };
    while (NB > 128 && !fits(NB)) NB -= 128;
    while (NB > 32 && !fits(NB)) NB -= 32;
    if (!fits(NB)) return HCLOOC_ERR_BUDGET;
    if (NB > N) NB = N;
    *nb_out = NB;
    return HCLOOC_OK;
}

}  // namespace

extern "C" int hclooc_dpotrf_plan(int64_t N, size_t device_budget_bytes, int64_t* NB, uint64_t* panel_bytes) {
    if (N < 1) return -1;
    if (!NB || !panel_bytes) return -3;
    int rc = potrf_nb(N, device_budget_bytes, NB);
    if (rc) return rc;
    *panel_bytes = round_1k((size_t)N * round_even(*NB) * 8) + 1024;
    return HCLOOC_OK;
}

extern "C" int hclooc_dpotrf(hclooc_ctx* ctx, int uplo, int64_t N, double* A, int64_t lda, size_t device_budget_bytes,
                             int64_t* info, hclooc_stats* stats) {
    const auto t_begin = std::chrono::steady_clock::now();
    if (uplo != HCL_UPLO_LOWER && uplo != HCL_UPLO_UPPER) return -2;
    if (N < 0) return -3;
    if (!info) return -7;
    *info = 0;
    if (stats) std::memset(stats, 0, sizeof(*stats));
    if (N == 0) return HCLOOC_OK;
    if (!A) return -4;
    if (lda < N) return -5;
    int rc;
    if (!ctx && (rc = default_ctx(&ctx))) return rc;
    std::lock_guard<std::mutex> lk(ctx->mu);
    HCL_CUDA(cudaSetDevice(ctx->device));
    bool dummy = true;
    if ((rc = check_resident(A, &dummy))) return rc;
    size_t budget = 0;
    bool own = false;
    if ((rc = resolve_budget(ctx, device_budget_bytes, &budget, &own))) return rc;
    int64_t NB = 0;
    if ((rc = potrf_nb(N, budget, &NB))) return rc;
    const bool lower = uplo == HCL_UPLO_LOWER;
    // the resident panel: (N - c0) x nbj for the lower factor (a block column), nbj x (N - c0) for the upper one (a block row)
    const size_t panel_bytes = lower ? round_1k((size_t)N * round_even(NB) * 8) : round_1k((size_t)NB * round_even(N) * 8);
    const size_t reserved = panel_bytes + 1024;                   // + the info word
    if (own) { if ((rc = ensure_workspace(ctx, budget))) return rc; }
    uint8_t* base = (uint8_t*)ctx->workspace;
    const uintptr_t mis = (uintptr_t)base & 1023u;
    const size_t shift = mis ? 1024 - mis : 0;
    if (reserved + shift > ctx->workspace_bytes) return HCLOOC_ERR_BUDGET;
    double* dP = (double*)(base + shift);
    long long* d_info = (long long*)(base + shift + panel_bytes);
    Reserve guard(ctx, reserved + shift);
    while (ctx->events.size() < 3) {
        cudaEvent_t e;
        HCL_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        ctx->events.push_back(e);
    }
    cudaStream_t sc = ctx->s_compute[0];
    HCL_CUDA(cudaMemsetAsync(d_info, 0, sizeof(long long), sc));
    hclooc_stats acc;
    std::memset(&acc, 0, sizeof(acc));
    double t_enq = 0.0;
    size_t ws_max = reserved;
    const int64_t nblk = (N + NB - 1) / NB;
    long long h_info = 0;
    for (int64_t bj = 0; bj < nblk; ++bj) {
        const int64_t c0 = bj * NB, nbj = std::min(NB, N - c0), rest = N - c0;
        // panel on the host: lower: A[c0:N, c0:c0+nbj] (rest x nbj); upper: A[c0:c0+nbj, c0:N] (nbj x rest)
        double* hP = A + c0 * lda + c0;
        const int64_t prow = lower ? rest : nbj, pcol = lower ? nbj : rest, ldp = round_even(pcol);
        if ((rc = copy2d(dP, (size_t)ldp * 8, hP, (size_t)lda * 8, (size_t)pcol * 8, (size_t)prow, ctx->s_h2d))) return rc;
        acc.bytes_h2d += (uint64_t)prow * pcol * 8; ++acc.n_copies_h2d;
        HCL_CUDA(cudaStreamSynchronize(ctx->s_h2d));               // the DGEMM's own streams do not wait for this one
        if (c0 > 0) {
            // the contribution of the block columns (rows) already factored, on the referenced triangle of the panel only:
            //   lower:  P <- P - L[c0:N, 0:c0] * L[c0:c0+nbj, 0:c0]^T          upper:  P <- P - U[0:c0, c0:c0+nbj]^T * U[0:c0, c0:N]
            hclooc_stats one;
            if (lower) rc = dgemm_core_locked(ctx, 0, 1, rest, nbj, c0, -1.0, A + c0 * lda, lda, A + c0 * lda, lda, 1.0, dP, ldp, budget, &one, 1);
            else rc = dgemm_core_locked(ctx, 1, 0, nbj, rest, c0, -1.0, A + c0, lda, A + c0, lda, 1.0, dP, ldp, budget, &one, 2);
            if (rc) return rc;
            add_stats(acc, one, &t_enq);
            ws_max = std::max(ws_max, reserved + (size_t)one.plan.workspace_bytes);
        }
        const auto te0 = std::chrono::steady_clock::now();
        // the diagonal block, then the rest of the panel:  lower: P21 <- P21 L_jj^-T;  upper: P12 <- U_jj^-T P12
        if ((rc = dev_potrf(dP, ldp, nbj, lower ? 1 : 0, d_info, (long long)c0, sc, &acc.n_kernels))) return rc;
        if (rest > nbj) {
            if (lower) rc = dev_trsm(1, dP, ldp, 0, 1, 0, dP + nbj * ldp, ldp, rest - nbj, nbj, 1.0, sc, &acc.n_kernels);
            else rc = dev_trsm(0, dP, ldp, 1, 1, 0, dP + nbj, ldp, rest - nbj, nbj, 1.0, sc, &acc.n_kernels);
            if (rc) return rc;
        }
        HCL_CUDA(cudaMemcpyAsync(&h_info, d_info, sizeof(long long), cudaMemcpyDeviceToHost, sc));
        HCL_CUDA(cudaStreamSynchronize(sc));
        t_enq += std::chrono::duration<double>(std::chrono::steady_clock::now() - te0).count();
        if (h_info != 0) break;                                     // not positive definite: the panel is not written back
        if ((rc = copy2d(hP, (size_t)lda * 8, dP, (size_t)ldp * 8, (size_t)pcol * 8, (size_t)prow, ctx->s_d2h))) return rc;
        acc.bytes_d2h += (uint64_t)prow * pcol * 8; ++acc.n_copies_d2h;
        HCL_CUDA(cudaStreamSynchronize(ctx->s_d2h));
    }
    *info = (int64_t)h_info;
    if (stats) {
        *stats = acc;
        stats->plan.M = N; stats->plan.N = N; stats->plan.K = N;
        stats->plan.mb = lower ? N : NB; stats->plan.nb = lower ? NB : N; stats->plan.kb = 128;
        stats->plan.h = lower ? 1 : nblk; stats->plan.w = lower ? nblk : 1; stats->plan.kpanels = 1; stats->plan.n_steps = nblk;
        stats->plan.workspace_bytes = ws_max;
        stats->plan.n_sets = 1;
        stats->plan.bytes_h2d = acc.bytes_h2d; stats->plan.bytes_d2h = acc.bytes_d2h;
        stats->plan.n_copies_h2d = acc.n_copies_h2d; stats->plan.n_copies_d2h = acc.n_copies_d2h;
        stats->plan.flops = (double)N * (double)N * (double)N / 3.0;
        stats->t_enqueue_s = t_enq;
        stats->t_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
    }
    return HCLOOC_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// DTRSM with a side argument.  side = Right:  X op(T) = alpha B,  B is M x N (host), T the `uplo` triangle of the N x N host
// matrix A.  Every row of B is an independent system, so (a) the rows are cut into bands small enough for a band of one block
// column to sit in device memory, and (b) inside a band the block columns are solved in the order of substitution (ascending
// when op(T) is upper), each one first receiving   B_j <- alpha*B_j - X[:, solved] op(T)[solved, j]   as one out-of-core DGEMM.
extern "C" int hclooc_dtrsm_side(hclooc_ctx* ctx, int side, int uplo, int trans, int diag, int64_t M, int64_t N, double alpha,
                                 const double* A, int64_t lda, double* B, int64_t ldb, size_t device_budget_bytes, hclooc_stats* stats) {
    if (side == HCL_SIDE_LEFT) {
        int rc = hclooc_dtrsm(ctx, uplo, trans, diag, M, N, alpha, A, lda, B, ldb, device_budget_bytes, stats);
        return rc < -1 ? rc - 1 : rc;                               // argument numbers shift by one (the side argument)
    }
    const auto t_begin = std::chrono::steady_clock::now();
    if (side != HCL_SIDE_RIGHT) return -2;
    if (uplo != HCL_UPLO_LOWER && uplo != HCL_UPLO_UPPER) return -3;
    if (trans != HCL_OP_N && trans != HCL_OP_T) return -4;
    if (diag != HCL_DIAG_NONUNIT && diag != HCL_DIAG_UNIT) return -5;
    if (M < 0) return -6;
    if (N < 0) return -7;
    if (stats) std::memset(stats, 0, sizeof(*stats));
    if (M == 0 || N == 0) return HCLOOC_OK;
    if (alpha != 0.0) {
        if (!A) return -9;
        if (lda < N) return -10;
    }
    if (!B) return -11;
    if (ldb < N) return -12;
    if (alpha != 0.0 && overlaps(B, M, N, ldb, A, N, N, lda)) return -11;
    int rc;
    if (alpha == 0.0) {                                              // X = 0, A not referenced, NaN in B not propagated
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
    // block-column width NB: the triangle buffer (NB x NB) takes at most a quarter of the budget; band height Mb: a band of one
    // block column (Mb x NB) takes at most a quarter as well; the out-of-core DGEMM keeps the other half
    int64_t NB = 4096;
    while (NB > 128 && (size_t)NB * NB * 8 + 1024 > budget / 4) NB -= 128;
    while (NB > 32 && (size_t)NB * NB * 8 + 1024 > budget / 4) NB -= 32;
    if ((size_t)NB * NB * 8 + 1024 > budget / 4) return HCLOOC_ERR_BUDGET;
    if (NB > N) NB = N;
    const int64_t ldt = round_even(NB), ldp = round_even(NB);
    const size_t tbytes = round_1k((size_t)NB * ldt * 8);
    int64_t Mb = (int64_t)((budget / 4 - 1024) / ((size_t)ldp * 8));
    if (Mb >= 128) Mb = Mb / 128 * 128;
    if (Mb < 1) return HCLOOC_ERR_BUDGET;
    if (Mb > M) Mb = M;
    const size_t pbytes = round_1k((size_t)Mb * ldp * 8);
    const size_t reserved = tbytes + pbytes;
    if (own) { if ((rc = ensure_workspace(ctx, budget))) return rc; }
    uint8_t* base = (uint8_t*)ctx->workspace;
    const uintptr_t mis = (uintptr_t)base & 1023u;
    const size_t shift = mis ? 1024 - mis : 0;
    if (reserved + shift > ctx->workspace_bytes) return HCLOOC_ERR_BUDGET;
    double* dT = (double*)(base + shift);
    double* dP = (double*)(base + shift + tbytes);
    Reserve guard(ctx, reserved + shift);
    const bool lower_op = (uplo == HCL_UPLO_LOWER) != (trans == HCL_OP_T);     // op(T) is lower triangular
    const int64_t nblk = (N + NB - 1) / NB;
    cudaStream_t sc = ctx->s_compute[0];
    hclooc_stats acc;
    std::memset(&acc, 0, sizeof(acc));
    double t_enq = 0.0;
    size_t ws_max = reserved;
    for (int64_t m0 = 0; m0 < M; m0 += Mb) {
        const int64_t mb = std::min(Mb, M - m0);
        for (int64_t bq = 0; bq < nblk; ++bq) {
            const int64_t j = lower_op ? nblk - 1 - bq : bq;                    // x_j depends on the columns after j when op(T) is lower
            const int64_t c0 = j * NB, nbj = std::min(NB, N - c0), c1 = c0 + nbj;
            const int64_t k0 = lower_op ? c1 : 0, kk = lower_op ? N - c1 : c0;    // columns already solved
            double* hB = B + m0 * ldb + c0;
            if ((rc = copy2d(dP, (size_t)ldp * 8, hB, (size_t)ldb * 8, (size_t)nbj * 8, (size_t)mb, ctx->s_h2d))) return rc;
            if ((rc = copy2d(dT, (size_t)ldt * 8, A + c0 * lda + c0, (size_t)lda * 8, (size_t)nbj * 8, (size_t)nbj, ctx->s_h2d))) return rc;
            acc.bytes_h2d += (uint64_t)mb * nbj * 8 + (uint64_t)nbj * nbj * 8; acc.n_copies_h2d += 2;
            HCL_CUDA(cudaStreamSynchronize(ctx->s_h2d));
            double scale = alpha;
            if (kk > 0) {
                // op(T)[solved, j]: stored at A[k0.., c0..] (kk x nbj), or, transposed, at A[c0.., k0..] (nbj x kk)
                const double* Tp = trans ? A + c0 * lda + k0 : A + k0 * lda + c0;
                hclooc_stats one;
                rc = dgemm_core_locked(ctx, 0, trans ? 1 : 0, mb, nbj, kk, -1.0, B + m0 * ldb + k0, ldb, Tp, lda, alpha, dP, ldp, budget, &one);
                if (rc) return rc;
                add_stats(acc, one, &t_enq);
                ws_max = std::max(ws_max, reserved + (size_t)one.plan.workspace_bytes);
                scale = 1.0;
            }
            if ((rc = dev_trsm(1, dT, ldt, lower_op ? 1 : 0, trans, diag, dP, ldp, mb, nbj, scale, sc, &acc.n_kernels))) return rc;
            HCL_CUDA(cudaStreamSynchronize(sc));
            if ((rc = copy2d(hB, (size_t)ldb * 8, dP, (size_t)ldp * 8, (size_t)nbj * 8, (size_t)mb, ctx->s_d2h))) return rc;
            acc.bytes_d2h += (uint64_t)mb * nbj * 8; ++acc.n_copies_d2h;
            HCL_CUDA(cudaStreamSynchronize(ctx->s_d2h));
        }
    }
    if (stats) {
        *stats = acc;
        stats->plan.M = M; stats->plan.N = N; stats->plan.K = N;
        stats->plan.mb = Mb; stats->plan.nb = NB; stats->plan.kb = 128;
        stats->plan.h = (M + Mb - 1) / Mb; stats->plan.w = nblk; stats->plan.kpanels = 1; stats->plan.n_steps = stats->plan.h * nblk;
        stats->plan.workspace_bytes = ws_max;
        stats->plan.n_sets = 1;
        stats->plan.bytes_h2d = acc.bytes_h2d; stats->plan.bytes_d2h = acc.bytes_d2h;
        stats->plan.n_copies_h2d = acc.n_copies_h2d; stats->plan.n_copies_d2h = acc.n_copies_d2h;
        stats->plan.flops = (double)M * (double)N * (double)N;
        stats->t_enqueue_s = t_enq;
        stats->t_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
    }
    return HCLOOC_OK;
}
