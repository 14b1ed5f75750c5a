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
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>
#include "executor.h"

using namespace hclooc;

namespace {

// the context whose debug shaker (executor.h) applies to the device recursions below: set by the routine that runs them
thread_local hclooc_ctx* t_dbg = nullptr;
struct DbgScope {
    hclooc_ctx* prev;
    explicit DbgScope(hclooc_ctx* c) : prev(t_dbg) { t_dbg = c; }
    ~DbgScope() { t_dbg = prev; }
};

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
        debug_jitter(t_dbg, st);
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
            e = launch_dgemm_tiles(s1 - s0, w, f1 - f0, -1.0, Tp, ldt, X + f0 * ld, ld, r.scale, X + s0 * ld, ld, st, 0, nullptr, trans ? 1 : 0, 0);
        } else {           // X[:, second] <- scale * X[:, second] - X[:, first] op(T)[first, second]
            const double* Tp = trans ? dT + s0 * ldt + f0 : dT + f0 * ldt + s0;
            e = launch_dgemm_tiles(w, s1 - s0, f1 - f0, -1.0, X + f0, ld, Tp, ldt, r.scale, X + s0, ld, st, 0, nullptr, 0, trans ? 1 : 0);
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
    debug_jitter(t_dbg, st);
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

// HCLOOC_FACTOR_TIMING: where the time of one pipeline call went (from the context's trace records)
void trace_summary(hclooc_ctx* ctx, const char* what) {
    static const char* names[] = {"H2D_A", "H2D_B", "H2D_C", "GEMM", "D2H_C"};
    for (int kind = 0; kind < 5; ++kind) {
        double first = 1e30, last = 0, busy = 0, cur_s = -1, cur_e = -1;
        size_t n = 0;
        uint64_t bytes = 0;
        std::vector<std::pair<double, double>> iv;
        for (const hclooc_trace_rec& r : ctx->trace_recs) if (r.kind == kind) { iv.emplace_back(r.t_start_ms, r.t_end_ms); bytes += r.bytes; ++n; }
        if (!n) continue;
        std::sort(iv.begin(), iv.end());
        for (auto& p : iv) {
            first = std::min(first, p.first); last = std::max(last, p.second);
            if (p.first > cur_e) { if (cur_e >= 0) busy += cur_e - cur_s; cur_s = p.first; cur_e = p.second; } else cur_e = std::max(cur_e, p.second);
        }
        busy += cur_e - cur_s;
        std::fprintf(stderr, "    %s %s: %zu ops, first start %.2f ms, last end %.2f ms, busy %.2f ms, %.3f GB\n", what, names[kind], n, first, last, busy, bytes / 1e9);
    }
}

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
    // two resident panels (one if a single panel covers the matrix) in at most half the budget
    auto fits = [&](int64_t nb) { return (nb >= N ? 1 : 2) * round_1k((size_t)N * round_even(nb) * 8) <= budget / 2; };
    while (NB > 128 && !fits(NB)) NB -= 128;
    while (NB > 32 && !fits(NB)) NB -= 32;
    if (!fits(NB)) return HCLOOC_ERR_BUDGET;
    if (NB > N) NB = N;
    *nb_out = NB;
    return HCLOOC_OK;
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------------------
// The device phases on their own: in-core DTRSM and DPOTRF on DEVICE pointers, asynchronous on the caller's stream -- what
// hclDgemmAsync is to hclooc_dgemm (the paper's runtime has the in-core kernel as a call of its own).
extern "C" int hclDtrsmAsync(int side, int uplo, int trans, int diag, int64_t M, int64_t N, double alpha, const double* dA, int64_t lda,
                             double* dB, int64_t ldb, hclStream s, hclEvent* ev) {
    if (side != HCL_SIDE_LEFT && side != HCL_SIDE_RIGHT) return -1;
    if (uplo != HCL_UPLO_LOWER && uplo != HCL_UPLO_UPPER) return -2;
    if (trans != HCL_OP_N && trans != HCL_OP_T) return -3;
    if (diag != HCL_DIAG_NONUNIT && diag != HCL_DIAG_UNIT) return -4;
    if (M < 0) return -5;
    if (N < 0) return -6;
    const int64_t n = side == HCL_SIDE_LEFT ? M : N;
    if (M > 0 && N > 0) {
        if (!dA) return -8;
        if (lda < n) return -9;
        if (!dB) return -10;
        if (ldb < N) return -11;
        if (((uintptr_t)dA & 15u) || ((uintptr_t)dB & 15u) || (lda & 1) || (ldb & 1)) return HCLOOC_ERR_ALIGN;
        uint64_t nk = 0;
        const int lower_op = (uplo == HCL_UPLO_LOWER) != (trans == HCL_OP_T);
        int rc = dev_trsm(side == HCL_SIDE_RIGHT, dA, lda, lower_op, trans, diag, dB, ldb, side == HCL_SIDE_LEFT ? N : M, n, alpha, (cudaStream_t)s, &nk);
        if (rc) return rc;
    }
    if (ev) {
        if (!*ev) { cudaEvent_t e; HCL_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming)); *ev = (hclEvent)e; }
        HCL_CUDA(cudaEventRecord((cudaEvent_t)*ev, (cudaStream_t)s));
    }
    return HCLOOC_OK;
}

extern "C" int hclDpotrfAsync(int uplo, int64_t N, double* dA, int64_t lda, long long* d_info, hclStream s, hclEvent* ev) {
    if (uplo != HCL_UPLO_LOWER && uplo != HCL_UPLO_UPPER) return -1;
    if (N < 0) return -2;
    if (!d_info) return -5;
    if (N > 0) {
        if (!dA) return -3;
        if (lda < N) return -4;
        if (((uintptr_t)dA & 15u) || (lda & 1)) return HCLOOC_ERR_ALIGN;
        uint64_t nk = 0;
        HCL_CUDA(cudaMemsetAsync(d_info, 0, sizeof(long long), (cudaStream_t)s));
        int rc = dev_potrf(dA, lda, N, uplo == HCL_UPLO_LOWER ? 1 : 0, d_info, 0, (cudaStream_t)s, &nk);
        if (rc) return rc;
    }
    if (ev) {
        if (!*ev) { cudaEvent_t e; HCL_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming)); *ev = (hclEvent)e; }
        HCL_CUDA(cudaEventRecord((cudaEvent_t)*ev, (cudaStream_t)s));
    }
    return HCLOOC_OK;
}

extern "C" int hclooc_dpotrf_plan(int64_t N, size_t device_budget_bytes, int64_t* NB, uint64_t* panel_bytes) {
    if (N < 1) return -1;
    if (!NB || !panel_bytes) return -3;
    int rc = potrf_nb(N, device_budget_bytes, NB);
    if (rc) return rc;
    *panel_bytes = (*NB >= N ? 1 : 2) * round_1k((size_t)N * round_even(*NB) * 8) + 1024;
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
    if ((rc = ensure_aux(ctx))) return rc;
    const bool lower = uplo == HCL_UPLO_LOWER;
    const int64_t nblk = (N + NB - 1) / NB;
    // TWO resident panels (one when the matrix is a single panel): panel j is factored in one while panel j+1 is uploaded into the
    // other and receives its out-of-core update.  Lower: (N - c0) x nbj, a block column; upper: nbj x (N - c0), a block row.
    const int npan = nblk > 1 ? 2 : 1;
    const size_t panel_bytes = lower ? round_1k((size_t)N * round_even(NB) * 8) : round_1k((size_t)NB * round_even(N) * 8);
    const size_t reserved = npan * panel_bytes + 1024;            // + the info word
    if (own) { if ((rc = ensure_workspace(ctx, budget))) return rc; }
    uint8_t* base = (uint8_t*)ctx->workspace;
    const uintptr_t mis = (uintptr_t)base & 1023u;
    const size_t shift = mis ? 1024 - mis : 0;
    if (reserved + shift > ctx->workspace_bytes) return HCLOOC_ERR_BUDGET;
    double* dPan[2] = {(double*)(base + shift), (double*)(base + shift + (npan - 1) * panel_bytes)};
    long long* d_info = (long long*)(base + shift + npan * panel_bytes);
    Reserve guard(ctx, reserved + shift);
    DbgScope dbg(ctx);
    // streams of this routine's own device work (the DGEMM pipeline keeps its own): diagonal phases, panel uploads, panel downloads
    cudaStream_t s_diag = ctx->s_aux[0], s_up = ctx->s_aux[1], s_down = ctx->s_aux[2], s_pot = ctx->s_aux[3];
    cudaEvent_t ev_up[2] = {ctx->ev_aux[0], ctx->ev_aux[1]}, ev_down[2] = {ctx->ev_aux[2], ctx->ev_aux[3]};
    cudaEvent_t ev_diag = ctx->ev_aux[4], ev_upd2 = ctx->ev_aux[5], ev_2a = ctx->ev_aux[6], ev_pot = ctx->ev_aux[7];
    struct Drain {      // whatever happens, nothing of this call is left running when it returns
        hclooc_ctx* c;
        ~Drain() { for (cudaStream_t st : c->s_aux) if (st) cudaStreamSynchronize(st); }
    } drain{ctx};
    static const bool timing = std::getenv("HCLOOC_FACTOR_TIMING") != nullptr;
    HCL_CUDA(cudaMemsetAsync(d_info, 0, sizeof(long long), s_diag));
    *ctx->h_word = 0;
    hclooc_stats acc;
    std::memset(&acc, 0, sizeof(acc));
    double t_enq = 0.0;
    size_t ws_max = reserved;
    auto geom = [&](int64_t bj, int64_t* c0, int64_t* nbj, int64_t* prow, int64_t* pcol, int64_t* ldp) {
        *c0 = bj * NB; *nbj = std::min(NB, N - *c0);
        const int64_t rest = N - *c0;
        *prow = lower ? rest : *nbj; *pcol = lower ? *nbj : rest; *ldp = round_even(*pcol);
    };
    auto upload = [&](int64_t bj, int buf) -> int {
        int64_t c0, nbj, prow, pcol, ldp;
        geom(bj, &c0, &nbj, &prow, &pcol, &ldp);
        int e = copy2d(dPan[buf], (size_t)ldp * 8, A + c0 * lda + c0, (size_t)lda * 8, (size_t)pcol * 8, (size_t)prow, s_up);
        if (e) return e;
        acc.bytes_h2d += (uint64_t)prow * pcol * 8; ++acc.n_copies_h2d;
        HCL_CUDA(cudaEventRecord(ev_up[buf], s_up));
        return HCLOOC_OK;
    };
    if ((rc = upload(0, 0))) return rc;
    long long h_info = 0;
    for (int64_t bj = 0; bj < nblk; ++bj) {
        const int cur = (int)(bj % npan), alt = npan - 1 - cur;
        int64_t c0, nbj, prow, pcol, ldp;
        geom(bj, &c0, &nbj, &prow, &pcol, &ldp);
        const int64_t rest = N - c0;
        double* dP = dPan[cur];
        const auto tp0 = std::chrono::steady_clock::now();
        // ---- panel bj: everything before it has been applied (update 1 by the pipeline, host-synchronised; update 2 on s_diag), and
        // its diagonal block has been factored on s_pot beside the second part of update 2 (panel 0: here)
        if (bj == 0) {
            HCL_CUDA(cudaStreamWaitEvent(s_diag, ev_up[cur], 0));
            if ((rc = dev_potrf(dP, ldp, nbj, lower ? 1 : 0, d_info, (long long)c0, s_diag, &acc.n_kernels))) return rc;
        } else {
            HCL_CUDA(cudaStreamWaitEvent(s_diag, ev_pot, 0));
        }
        if (rest > nbj) {       // the rest of the panel against the diagonal block:  lower: P21 <- P21 L_jj^-T;  upper: P12 <- U_jj^-T P12
            if (lower) rc = dev_trsm(1, dP, ldp, 0, 1, 0, dP + nbj * ldp, ldp, rest - nbj, nbj, 1.0, s_diag, &acc.n_kernels);
            else rc = dev_trsm(0, dP, ldp, 1, 1, 0, dP + nbj, ldp, rest - nbj, nbj, 1.0, s_diag, &acc.n_kernels);
            if (rc) return rc;
        }
        HCL_CUDA(cudaMemcpyAsync(ctx->h_word, d_info, sizeof(long long), cudaMemcpyDeviceToHost, s_diag));
        HCL_CUDA(cudaEventRecord(ev_diag, s_diag));
        // ---- panel bj goes down as soon as it is final, beside everything that follows (a panel that failed goes down too: its
        // leading columns are the factor's, LAPACK leaves the rest undefined).  Only what the factorization owns is written: the
        // diagonal block goes down in strips of 128 rows cut at the diagonal tile -- the panel's blocks that lie wholly in the other
        // triangle were never brought up (the pipeline has no step for them), and the host keeps its bits there.
        HCL_CUDA(cudaStreamWaitEvent(s_down, ev_diag, 0));
        debug_jitter(ctx, s_down);
        {
            double* hP = A + c0 * lda + c0;
            for (int64_t r = 0; r < nbj; r += 128) {
                const int64_t rr = std::min<int64_t>(128, nbj - r);
                if (lower) rc = copy2d(hP + r * lda, (size_t)lda * 8, dP + r * ldp, (size_t)ldp * 8, (size_t)(r + rr) * 8, (size_t)rr, s_down);
                else rc = copy2d(hP + r * lda + r, (size_t)lda * 8, dP + r * ldp + r, (size_t)ldp * 8, (size_t)(rest - r) * 8, (size_t)rr, s_down);
                if (rc) return rc;
                acc.bytes_d2h += (uint64_t)rr * (lower ? r + rr : rest - r) * 8; ++acc.n_copies_d2h;
            }
            if (lower && rest > nbj) {
                if ((rc = copy2d(hP + nbj * lda, (size_t)lda * 8, dP + nbj * ldp, (size_t)ldp * 8, (size_t)nbj * 8, (size_t)(rest - nbj), s_down))) return rc;
                acc.bytes_d2h += (uint64_t)(rest - nbj) * nbj * 8; ++acc.n_copies_d2h;
            }
        }
        HCL_CUDA(cudaEventRecord(ev_down[cur], s_down));
        // ---- meanwhile panel bj+1 comes up into the other buffer and receives the contribution of the panels BEFORE bj from the
        // host: ONE out-of-core DGEMM whose C blocks are read from the host matrix and stored into the device panel (the pipeline
        // itself brings the panel up, under its kernels); its first store waits until the buffer's previous tenant, panel bj-1, has
        // been downloaded and read by the update 2 of panel bj
        int64_t c0n = 0, nbn = 0, prown = 0, pcoln = 0, ldpn = 0;
        bool uploaded_whole = false;
        if (bj + 1 < nblk) {
            geom(bj + 1, &c0n, &nbn, &prown, &pcoln, &ldpn);
            if (c0 > 0) {
                //   lower:  P <- P - L[c0n:N, 0:c0] * L[c0n:c0n+nbn, 0:c0]^T        upper:  P <- P - U[0:c0, c0n:c0n+nbn]^T * U[0:c0, c0n:N]
                // (the 128 x 128 tiles on the panel's diagonal come up whole first: the pipeline brings only the blocks of ITS plan
                // that touch the referenced triangle, and the strips that go down later are cut at these tiles)
                HCL_CUDA(cudaEventSynchronize(ev_down[alt]));   // panel bj-1 is on the HOST: the pipeline is about to read it as an operand
                HCL_CUDA(cudaStreamWaitEvent(s_up, ev_upd2, 0));  // (found by the debug shaker: nothing else orders that download before the uploads)
                debug_jitter(ctx, s_up);
                debug_poison(ctx, dPan[alt], ldpn, prown, pcoln, s_up);         // the buffer is free now: nobody may still read panel bj-1
                for (int64_t r = 0; r < nbn; r += 128) {
                    const int64_t rr = std::min<int64_t>(128, nbn - r);
                    if ((rc = copy2d(dPan[alt] + r * ldpn + r, (size_t)ldpn * 8, A + (c0n + r) * lda + c0n + r, (size_t)lda * 8, (size_t)rr * 8, (size_t)rr, s_up))) return rc;
                    acc.bytes_h2d += (uint64_t)rr * rr * 8; ++acc.n_copies_h2d;
                }
                HCL_CUDA(cudaEventRecord(ev_up[alt], s_up));
                hclooc_stats one;
                DgemmExtra ex;
                ex.C_src = A + c0n * lda + c0n; ex.ldc_src = lda;
                ex.wait_before_store[0] = ev_up[alt];
                const bool trace_was = ctx->trace;
                if (timing) ctx->trace = true;
                if (lower) rc = dgemm_core_locked(ctx, 0, 1, N - c0n, nbn, c0, -1.0, A + c0n * lda, lda, A + c0n * lda, lda, 1.0, dPan[alt], ldpn, budget, &one, 1, &ex);
                else rc = dgemm_core_locked(ctx, 1, 0, nbn, N - c0n, c0, -1.0, A + c0n, lda, A + c0n, lda, 1.0, dPan[alt], ldpn, budget, &one, 2, &ex);
                ctx->trace = trace_was;
                if (rc) return rc;
                if (timing) trace_summary(ctx, "update 1");
                add_stats(acc, one, &t_enq);
                ws_max = std::max(ws_max, reserved + (size_t)one.plan.workspace_bytes);
                if (timing) std::fprintf(stderr, "  update %lld x %lld x %lld: %.2f ms (%.1f TFLOP/s), plan %lld x %lld blocks of %lld x %lld, %d C / %d A / %d B buffers, ksplit %d, %.2f GB up\n",
                                         (long long)(lower ? N - c0n : nbn), (long long)(lower ? nbn : N - c0n), (long long)c0, 1e3 * one.t_total_s,
                                         2e-12 * (double)(N - c0n) * nbn * c0 / one.t_total_s, (long long)one.plan.h, (long long)one.plan.w, (long long)one.plan.mb,
                                         (long long)one.plan.nb, one.plan.n_sets, one.plan.n_abuf, one.plan.n_bbuf, one.plan.ksplit, one.bytes_h2d / 1e9);
            } else {            // panel 1: nothing before panel 0, it just comes up whole (the buffer has had no tenant yet)
                if ((rc = upload(bj + 1, alt))) return rc;
                uploaded_whole = true;
            }
        }
        const auto tp1 = std::chrono::steady_clock::now();
        HCL_CUDA(cudaEventSynchronize(ev_diag));
        h_info = *ctx->h_word;
        if (timing) {
            const auto tp2 = std::chrono::steady_clock::now();
            std::fprintf(stderr, "dpotrf panel %lld: upload + out-of-core update of the next panel %.2f ms, then %.2f ms more for the diagonal phase\n",
                         (long long)bj, 1e3 * std::chrono::duration<double>(tp1 - tp0).count(), 1e3 * std::chrono::duration<double>(tp2 - tp1).count());
        }
        if (h_info != 0) break;                                     // not positive definite
        // ---- panel bj+1 receives panel bj's contribution straight from device memory (update 2): first its diagonal block, which
        // is then factored on a stream of its own WHILE the rest of the panel is updated (the factorization of a 4096-block is a chain
        // of small launches that leaves nearly every SM idle)
        if (bj + 1 < nblk) {
            if (uploaded_whole) HCL_CUDA(cudaStreamWaitEvent(s_diag, ev_up[alt], 0));
            debug_jitter(ctx, s_diag);
            const int64_t below = N - c0n - nbn;                  // rows (lower) / columns (upper) of panel bj+1 past its diagonal block
            //   lower:  P' <- P' - L[c0n:N, c0:c0n] * L[c0n:c0n+nbn, c0:c0n]^T, both operands = rows nbj.. of the panel just factored
            if (lower) rc = launch_dgemm_tiles(nbn, nbn, nbj, -1.0, dP + nbj * ldp, ldp, dP + nbj * ldp, ldp, 1.0, dPan[alt], ldpn, s_diag, 0, nullptr, 0, 1, 1, 0);
            else rc = launch_dgemm_tiles(nbn, nbn, nbj, -1.0, dP + nbj, ldp, dP + nbj, ldp, 1.0, dPan[alt], ldpn, s_diag, 0, nullptr, 1, 0, 2, 0);
            if (rc) return rc;
            ++acc.n_kernels;
            HCL_CUDA(cudaEventRecord(ev_2a, s_diag));
            HCL_CUDA(cudaStreamWaitEvent(s_pot, ev_2a, 0));
            debug_jitter(ctx, s_pot);
            if ((rc = dev_potrf(dPan[alt], ldpn, nbn, lower ? 1 : 0, d_info, (long long)c0n, s_pot, &acc.n_kernels))) return rc;
            HCL_CUDA(cudaEventRecord(ev_pot, s_pot));
            if (below > 0) {
                if (lower) rc = launch_dgemm_tiles(below, nbn, nbj, -1.0, dP + (nbj + nbn) * ldp, ldp, dP + nbj * ldp, ldp, 1.0, dPan[alt] + nbn * ldpn, ldpn, s_diag, 0, nullptr, 0, 1);
                else rc = launch_dgemm_tiles(nbn, below, nbj, -1.0, dP + nbj, ldp, dP + nbj + nbn, ldp, 1.0, dPan[alt] + nbn, ldpn, s_diag, 0, nullptr, 1, 0);
                if (rc) return rc;
                ++acc.n_kernels;
            }
            HCL_CUDA(cudaEventRecord(ev_upd2, s_diag));
        }
    }
    for (cudaStream_t st : {s_diag, s_up, s_down, s_pot}) HCL_CUDA(cudaStreamSynchronize(st));
    *info = (int64_t)h_info;
    if (stats) {
        *stats = acc;
        stats->plan.M = N; stats->plan.N = N; stats->plan.K = N;
        stats->plan.mb = lower ? N : NB; stats->plan.nb = lower ? NB : N; stats->plan.kb = 128;
        stats->plan.h = lower ? 1 : nblk; stats->plan.w = lower ? nblk : 1; stats->plan.kpanels = 1; stats->plan.n_steps = nblk;
        stats->plan.workspace_bytes = ws_max;
        stats->plan.n_sets = npan;
        stats->plan.bytes_h2d = acc.bytes_h2d; stats->plan.bytes_d2h = acc.bytes_d2h;
        stats->plan.n_copies_h2d = acc.n_copies_h2d; stats->plan.n_copies_d2h = acc.n_copies_d2h;
        stats->plan.flops = (double)N * (double)N * (double)N / 3.0;
        stats->t_enqueue_s = t_enq;
        stats->t_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
    }
    return HCLOOC_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// DTRSM, side = Right, with a LOOK-AHEAD of one block column: the mirror image of dtrsm_left_lookahead below.  Block column j
// (M x NB) is solved in device memory -- T_jj uploaded, row chunks on two streams, each chunk downloaded as soon as it is solved --
// WHILE block column j+1 is brought up by the DGEMM pipeline and receives
//     B_{j+1} <- alpha*B_{j+1} - X[:, solved before j] op(T)[solved before j, j+1]
// (C blocks read from the host matrix, stored into the other resident buffer); the contribution of block column j,
// -X_j op(T)[j, j+1], then comes straight from device memory.  ctx->mu is held by the caller.
static int dtrsm_right_lookahead(hclooc_ctx* ctx, int uplo, int trans, int diag, int64_t M, int64_t N, double alpha, const double* A, int64_t lda,
                                 double* B, int64_t ldb, size_t budget, bool own, int64_t NB, hclooc_stats* stats) {
    const auto t_begin = std::chrono::steady_clock::now();
    int rc;
    if ((rc = ensure_aux(ctx))) return rc;
    const bool lower_op = (uplo == HCL_UPLO_LOWER) != (trans == HCL_OP_T);    // op(T) is lower triangular
    const int64_t nblk = (N + NB - 1) / NB, ldp = round_even(NB), ldt = round_even(NB);
    const size_t pbytes = round_1k((size_t)M * ldp * 8), tbytes = round_1k((size_t)NB * ldt * 8);
    const size_t reserved0 = 2 * pbytes + 2 * tbytes;
    if (own) { if ((rc = ensure_workspace(ctx, budget))) return rc; }
    uint8_t* base = (uint8_t*)ctx->workspace;
    const uintptr_t mis = (uintptr_t)base & 1023u;
    const size_t shift = mis ? 1024 - mis : 0;
    if (reserved0 + shift > ctx->workspace_bytes) return HCLOOC_ERR_BUDGET;
    double* dP[2] = {(double*)(base + shift), (double*)(base + shift + pbytes)};
    double* dT = (double*)(base + shift + 2 * pbytes);               // T_jj of the block column being solved
    double* dT2 = (double*)(base + shift + 2 * pbytes + tbytes);     // op(T)[current, next] as stored
    Reserve guard(ctx, reserved0 + shift);
    DbgScope dbg(ctx);
    cudaStream_t s_sol[2] = {ctx->s_aux[0], ctx->s_aux[3]}, s_up = ctx->s_aux[1], s_down = ctx->s_aux[2];
    cudaEvent_t ev_T = ctx->ev_aux[0], ev_T2 = ctx->ev_aux[1], ev_down[2] = {ctx->ev_aux[2], ctx->ev_aux[3]};
    cudaEvent_t ev_sol[2] = {ctx->ev_aux[4], ctx->ev_aux[5]}, ev_ready = ctx->ev_aux[6], ev_chunk = ctx->ev_aux[7];
    struct Drain {
        hclooc_ctx* c;
        ~Drain() { for (cudaStream_t st : c->s_aux) if (st) cudaStreamSynchronize(st); }
    } drain{ctx};
    static const int nchunk = [] { const char* e = std::getenv("HCLOOC_TRSM_CHUNKS"); const int v = e ? std::atoi(e) : 0; return v > 0 ? v : 4; }();
    hclooc_stats acc;
    std::memset(&acc, 0, sizeof(acc));
    double t_enq = 0.0;
    size_t ws_max = reserved0;
    // x_j depends on the block columns BEFORE j when op(T) is upper, on the ones after it when op(T) is lower
    auto cols_of = [&](int64_t bj, int64_t* c0, int64_t* nbj) {
        const int64_t j = lower_op ? nblk - 1 - bj : bj;
        *c0 = j * NB; *nbj = std::min(NB, N - *c0);
    };
    {   // block column 0 comes up whole
        int64_t c0, nb0;
        cols_of(0, &c0, &nb0);
        if ((rc = copy2d(dP[0], (size_t)ldp * 8, B + c0, (size_t)ldb * 8, (size_t)nb0 * 8, (size_t)M, s_up))) return rc;
        acc.bytes_h2d += (uint64_t)M * nb0 * 8; ++acc.n_copies_h2d;
        HCL_CUDA(cudaEventRecord(ev_ready, s_up));
    }
    int64_t hr = ((M + nchunk - 1) / nchunk + 63) / 64 * 64;        // rows per chunk
    if (hr < 1024) hr = 1024;
    bool scaled = false;                                            // has alpha reached the block column in dP[cur]?
    for (int64_t bj = 0; bj < nblk; ++bj) {
        const int cur = (int)(bj & 1), alt = 1 - cur;
        int64_t c0, nbj;
        cols_of(bj, &c0, &nbj);
        // ---- T_jj up, then the row chunks of block column bj on two streams; every chunk goes down as soon as it is solved
        if ((rc = copy2d(dT, (size_t)ldt * 8, A + c0 * lda + c0, (size_t)lda * 8, (size_t)nbj * 8, (size_t)nbj, s_up))) return rc;
        acc.bytes_h2d += (uint64_t)nbj * nbj * 8; ++acc.n_copies_h2d;
        HCL_CUDA(cudaEventRecord(ev_T, s_up));
        int64_t c = 0;
        for (int64_t r0 = 0; r0 < M; r0 += hr, ++c) {
            const int64_t hrows = std::min(hr, M - r0);
            cudaStream_t st = s_sol[c & 1];
            if (c < 2) { HCL_CUDA(cudaStreamWaitEvent(st, ev_T, 0)); HCL_CUDA(cudaStreamWaitEvent(st, ev_ready, 0)); }
            if ((rc = dev_trsm(1, dT, ldt, lower_op ? 1 : 0, trans, diag, dP[cur] + r0 * ldp, ldp, hrows, nbj, scaled ? 1.0 : alpha, st, &acc.n_kernels))) return rc;
            HCL_CUDA(cudaEventRecord(ev_chunk, st));
            HCL_CUDA(cudaStreamWaitEvent(s_down, ev_chunk, 0));
            debug_jitter(ctx, s_down);
            if ((rc = copy2d(B + r0 * ldb + c0, (size_t)ldb * 8, dP[cur] + r0 * ldp, (size_t)ldp * 8, (size_t)nbj * 8, (size_t)hrows, s_down))) return rc;
            acc.bytes_d2h += (uint64_t)hrows * nbj * 8; ++acc.n_copies_d2h;
        }
        HCL_CUDA(cudaEventRecord(ev_down[cur], s_down));
        for (int s = 0; s < 2; ++s) HCL_CUDA(cudaEventRecord(ev_sol[s], s_sol[s]));
        if (bj + 1 == nblk) break;
        // ---- meanwhile: block column bj+1
        int64_t q0, nb2;
        cols_of(bj + 1, &q0, &nb2);
        // op(T)[current, next] as stored: T[c0.., q0..] (nbj x nb2), or, transposed, T[q0.., c0..] (nb2 x nbj); dT2's previous reader
        // is the update 2 of this block column, issued at the end of the last round and possibly still running
        HCL_CUDA(cudaStreamWaitEvent(s_up, ev_ready, 0));
        if (trans) rc = copy2d(dT2, (size_t)ldt * 8, A + q0 * lda + c0, (size_t)lda * 8, (size_t)nbj * 8, (size_t)nb2, s_up);
        else rc = copy2d(dT2, (size_t)ldt * 8, A + c0 * lda + q0, (size_t)lda * 8, (size_t)nb2 * 8, (size_t)nbj, s_up);
        if (rc) return rc;
        acc.bytes_h2d += (uint64_t)nbj * nb2 * 8; ++acc.n_copies_h2d;
        HCL_CUDA(cudaEventRecord(ev_T2, s_up));
        // columns solved BEFORE the current block column: [0, c0) when op(T) is upper, [c0 + nbj, N) when it is lower
        const int64_t k0 = lower_op ? c0 + nbj : 0, kk = lower_op ? N - (c0 + nbj) : c0;
        bool next_scaled = false;
        if (kk > 0) {
            HCL_CUDA(cudaEventSynchronize(ev_down[alt]));                       // X of block column bj-1 is on the host (the pipeline reads it)
            const double* Tp = trans ? A + q0 * lda + k0 : A + k0 * lda + q0;   // op(T)[solved, next], as stored
            hclooc_stats one;
            DgemmExtra ex;
            ex.C_src = B + q0; ex.ldc_src = ldb;
            ex.wait_before_store[0] = ev_ready;                                 // update 2 of block column bj read X_{bj-1} from dP[alt]
            if (ctx->dbg_poison) {                                              // debug: the buffer is free now, nobody may still read X_{bj-1}
                debug_poison(ctx, dP[alt], ldp, M, nb2, s_up);
                HCL_CUDA(cudaEventRecord(ev_T2, s_up));
                ex.wait_before_store[1] = ev_T2;
            }
            rc = dgemm_core_locked(ctx, 0, trans ? 1 : 0, M, nb2, kk, -1.0, B + k0, ldb, Tp, lda, alpha, dP[alt], ldp, budget, &one, 0, &ex);
            if (rc) return rc;
            add_stats(acc, one, &t_enq);
            ws_max = std::max(ws_max, reserved0 + (size_t)one.plan.workspace_bytes);
            next_scaled = true;
        } else {                                                                // the second block column: nothing before the first one
            if ((rc = copy2d(dP[alt], (size_t)ldp * 8, B + q0, (size_t)ldb * 8, (size_t)nb2 * 8, (size_t)M, s_up))) return rc;
            acc.bytes_h2d += (uint64_t)M * nb2 * 8; ++acc.n_copies_h2d;
            HCL_CUDA(cudaEventRecord(ev_T2, s_up));                             // (covers the block of T and the block column)
        }
        for (int s = 0; s < 2; ++s) HCL_CUDA(cudaEventSynchronize(ev_sol[s]));  // block column bj is solved
        // ---- update 2: B_next <- beta' * B_next - X_current op(T)[current, next], all in device memory
        HCL_CUDA(cudaStreamWaitEvent(s_sol[0], ev_T2, 0));
        debug_jitter(ctx, s_sol[0]);
        rc = launch_dgemm_tiles(M, nb2, nbj, -1.0, dP[cur], ldp, dT2, ldt, next_scaled ? 1.0 : alpha, dP[alt], ldp, s_sol[0], -1, nullptr, 0, trans ? 1 : 0);
        if (rc) return rc;
        ++acc.n_kernels;
        HCL_CUDA(cudaEventRecord(ev_ready, s_sol[0]));
        scaled = true;
    }
    for (cudaStream_t st : ctx->s_aux) if (st) HCL_CUDA(cudaStreamSynchronize(st));
    if (stats) {
        *stats = acc;
        stats->plan.M = M; stats->plan.N = N; stats->plan.K = N;
        stats->plan.mb = std::min(M, hr); stats->plan.nb = NB; stats->plan.kb = 128;
        stats->plan.h = (M + hr - 1) / hr; stats->plan.w = nblk; stats->plan.kpanels = 1; stats->plan.n_steps = nblk;
        stats->plan.workspace_bytes = ws_max;
        stats->plan.n_sets = 2;
        stats->plan.ldc_dev = ldp;
        stats->plan.bytes_h2d = acc.bytes_h2d; stats->plan.bytes_d2h = acc.bytes_d2h;
        stats->plan.n_copies_h2d = acc.n_copies_h2d; stats->plan.n_copies_d2h = acc.n_copies_d2h;
        stats->plan.flops = (double)M * (double)N * (double)N;
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
    // two whole block columns (M x NB) and two NB x NB blocks of T beside a quarter of the budget for the pipeline: the look-ahead
    // form above (HCLOOC_TRSM_LOOKAHEAD=0: never); the widest NB of 4096, 2048, 1024 that fits
    {
        const char* e = std::getenv("HCLOOC_TRSM_LOOKAHEAD");
        if (!(e && std::atoi(e) == 0) && N > 1024) {
            for (int64_t nb = 4096; nb >= 1024; nb /= 2) {
                const int64_t nbe = std::min(nb, N);
                const size_t pb = round_1k((size_t)M * round_even(nbe) * 8), tb = round_1k((size_t)nbe * round_even(nbe) * 8);
                if (2 * pb + 2 * tb + budget / 4 <= budget) {
                    rc = dtrsm_right_lookahead(ctx, uplo, trans, diag, M, N, alpha, A, lda, B, ldb, budget, own, nbe, stats);
                    if (!rc && stats) stats->t_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
                    return rc;
                }
            }
        }
    }
    // staged form.  Block-column width NB: the triangle buffer (NB x NB) takes at most a quarter of the budget; band height Mb: a band of one
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
    DbgScope dbg(ctx);
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

// ---------------------------------------------------------------------------------------------------------------------
// hclooc_dtrsm (side = Left) with a LOOK-AHEAD of one block row, the resident mode of executor.cu's hclooc_dtrsm when two block
// rows and two NB x NB blocks of T fit beside the pipeline.  Block row i (NB x N) is solved in device memory -- T_ii uploaded,
// column chunks on two streams, each chunk downloaded as soon as it is solved -- WHILE block row i+1 is brought up and receives
//     B_{i+1} <- alpha*B_{i+1} - op(T)[i+1, solved before i] X[solved before i]
// as one out-of-core DGEMM whose C blocks are read from the host matrix and stored into the other resident buffer (the pipeline
// itself brings the block row up).  The contribution of block row i, -op(T)[i+1, i] X_i, then comes straight from device memory
// (one GPU-filling launch; only the NB x NB block of T crosses the link).  ctx->mu is held by the caller for the whole solve.
namespace hclooc {

// the device triangular solve for the other routines built on it (lu.cu); dbg: the context whose debug shaker applies (nullable)
int dev_trsm_ctx(hclooc_ctx* dbg, int right, const double* dT, int64_t ldt, int lower, int trans, int unit, double* X, int64_t ld, int64_t w,
                 int64_t n, double scale, cudaStream_t st, uint64_t* n_kernels) {
    DbgScope scope(dbg);
    return dev_trsm(right, dT, ldt, lower, trans, unit, X, ld, w, n, scale, st, n_kernels);
}

int dtrsm_left_lookahead(hclooc_ctx* ctx, int uplo, int trans, int diag, int64_t M, int64_t N, double alpha, const double* A, int64_t lda,
                         double* B, int64_t ldb, size_t budget, bool own, int64_t NB, hclooc_stats* stats) {
    const auto t_begin = std::chrono::steady_clock::now();
    int rc;
    HCL_CUDA(cudaSetDevice(ctx->device));
    if ((rc = ensure_aux(ctx))) return rc;
    const bool lower = (uplo == HCL_UPLO_LOWER) != (trans == HCL_OP_T);       // op(T) is lower triangular
    const int64_t nblk = (M + NB - 1) / NB, ldx = round_even(N), ldt = round_even(NB);
    const size_t rbytes = round_1k((size_t)NB * ldx * 8), tbytes = round_1k((size_t)NB * ldt * 8);
    const size_t reserved0 = 2 * rbytes + 2 * tbytes;
    if (own) { if ((rc = ensure_workspace(ctx, budget))) return rc; }
    uint8_t* base = (uint8_t*)ctx->workspace;
    const uintptr_t mis = (uintptr_t)base & 1023u;
    const size_t shift = mis ? 1024 - mis : 0;
    if (reserved0 + shift > ctx->workspace_bytes) return HCLOOC_ERR_BUDGET;
    double* dR[2] = {(double*)(base + shift), (double*)(base + shift + rbytes)};
    double* dT = (double*)(base + shift + 2 * rbytes);              // T_ii of the block row being solved
    double* dT2 = (double*)(base + shift + 2 * rbytes + tbytes);    // op(T)[next, current] as stored
    Reserve guard(ctx, reserved0 + shift);
    DbgScope dbg(ctx);
    cudaStream_t s_sol[2] = {ctx->s_aux[0], ctx->s_aux[3]}, s_up = ctx->s_aux[1], s_down = ctx->s_aux[2];
    cudaEvent_t ev_T = ctx->ev_aux[0], ev_T2 = ctx->ev_aux[1], ev_down[2] = {ctx->ev_aux[2], ctx->ev_aux[3]};
    cudaEvent_t ev_sol[2] = {ctx->ev_aux[4], ctx->ev_aux[5]}, ev_ready = ctx->ev_aux[6], ev_chunk = ctx->ev_aux[7];
    struct Drain {
        hclooc_ctx* c;
        ~Drain() { for (cudaStream_t st : c->s_aux) if (st) cudaStreamSynchronize(st); }
    } drain{ctx};
    static const bool timing = std::getenv("HCLOOC_FACTOR_TIMING") != nullptr;
    static const int nchunk = [] { const char* e = std::getenv("HCLOOC_TRSM_CHUNKS"); const int v = e ? std::atoi(e) : 0; return v > 0 ? v : 4; }();
    hclooc_stats acc;
    std::memset(&acc, 0, sizeof(acc));
    double t_enq = 0.0;
    size_t ws_max = reserved0;
    auto rows_of = [&](int64_t bi, int64_t* r0, int64_t* nbi) {
        const int64_t i = lower ? bi : nblk - 1 - bi;
        *r0 = i * NB; *nbi = std::min(NB, M - *r0);
    };
    // block row 0 comes up whole
    {
        int64_t r0, nb0;
        rows_of(0, &r0, &nb0);
        if ((rc = copy2d(dR[0], (size_t)ldx * 8, B + r0 * ldb, (size_t)ldb * 8, (size_t)N * 8, (size_t)nb0, s_up))) return rc;
        acc.bytes_h2d += (uint64_t)nb0 * N * 8; ++acc.n_copies_h2d;
        HCL_CUDA(cudaEventRecord(ev_ready, s_up));
    }
    bool scaled = false;                                                        // has alpha reached the block row in dR[cur]?
    for (int64_t bi = 0; bi < nblk; ++bi) {
        const int cur = (int)(bi & 1), alt = 1 - cur;
        int64_t r0, nbi;
        rows_of(bi, &r0, &nbi);
        const auto tp0 = std::chrono::steady_clock::now();
        // ---- T_ii up, then the column chunks of block row bi on two streams; every chunk goes down as soon as it is solved
        if ((rc = copy2d(dT, (size_t)ldt * 8, A + r0 * lda + r0, (size_t)lda * 8, (size_t)nbi * 8, (size_t)nbi, s_up))) return rc;
        acc.bytes_h2d += (uint64_t)nbi * nbi * 8; ++acc.n_copies_h2d;
        HCL_CUDA(cudaEventRecord(ev_T, s_up));
        int64_t wr = ((N + nchunk - 1) / nchunk + 63) / 64 * 64;
        if (wr < 1024) wr = 1024;
        int64_t c = 0;
        for (int64_t c0 = 0; c0 < N; c0 += wr, ++c) {
            const int64_t w = std::min(wr, N - c0);
            cudaStream_t st = s_sol[c & 1];
            if (c < 2) { HCL_CUDA(cudaStreamWaitEvent(st, ev_T, 0)); HCL_CUDA(cudaStreamWaitEvent(st, ev_ready, 0)); }
            if ((rc = dev_trsm(0, dT, ldt, lower ? 1 : 0, trans, diag, dR[cur] + c0, ldx, w, nbi, scaled ? 1.0 : alpha, st, &acc.n_kernels))) return rc;
            HCL_CUDA(cudaEventRecord(ev_chunk, st));
            HCL_CUDA(cudaStreamWaitEvent(s_down, ev_chunk, 0));
            debug_jitter(ctx, s_down);
            if ((rc = copy2d(B + r0 * ldb + c0, (size_t)ldb * 8, dR[cur] + c0, (size_t)ldx * 8, (size_t)w * 8, (size_t)nbi, s_down))) return rc;
            acc.bytes_d2h += (uint64_t)nbi * w * 8; ++acc.n_copies_d2h;
        }
        HCL_CUDA(cudaEventRecord(ev_down[cur], s_down));
        for (int s = 0; s < 2; ++s) HCL_CUDA(cudaEventRecord(ev_sol[s], s_sol[s]));
        if (bi + 1 == nblk) break;
        // ---- meanwhile: block row bi+1
        int64_t q0, nb2;
        rows_of(bi + 1, &q0, &nb2);
        // op(T)[next, current] as stored: T[q0.., r0..] (nb2 x nbi), or, transposed, T[r0.., q0..] (nbi x nb2); dT2's previous
        // reader is the update 2 of this block row, issued at the end of the last round and possibly still running
        HCL_CUDA(cudaStreamWaitEvent(s_up, ev_ready, 0));                      // ... on the device: after that update 2
        if (trans) rc = copy2d(dT2, (size_t)ldt * 8, A + r0 * lda + q0, (size_t)lda * 8, (size_t)nb2 * 8, (size_t)nbi, s_up);
        else rc = copy2d(dT2, (size_t)ldt * 8, A + q0 * lda + r0, (size_t)lda * 8, (size_t)nbi * 8, (size_t)nb2, s_up);
        if (rc) return rc;
        acc.bytes_h2d += (uint64_t)nbi * nb2 * 8; ++acc.n_copies_h2d;
        HCL_CUDA(cudaEventRecord(ev_T2, s_up));
        // rows solved BEFORE the current block row: [0, r0) when op(T) is lower, [r0 + nbi, M) when it is upper
        const int64_t k0 = lower ? 0 : r0 + nbi, kk = lower ? r0 : M - (r0 + nbi);
        bool next_scaled = false;
        if (kk > 0) {
            HCL_CUDA(cudaEventSynchronize(ev_down[alt]));                       // X of block row bi-1 is on the host (the pipeline reads it)
            const double* Ap = trans ? A + k0 * lda + q0 : A + q0 * lda + k0;   // op(T)[next, solved], as stored
            hclooc_stats one;
            DgemmExtra ex;
            ex.C_src = B + q0 * ldb; ex.ldc_src = ldb;
            ex.wait_before_store[0] = ev_ready;                                 // update 2 of block row bi read X_{bi-1} from dR[alt]
            if (ctx->dbg_poison) {                                              // debug: the buffer is free now, nobody may still read X_{bi-1}
                debug_poison(ctx, dR[alt], ldx, nb2, N, s_up);                  // (s_up has waited for ev_ready above; the download was host-synchronised)
                HCL_CUDA(cudaEventRecord(ev_T2, s_up));
                ex.wait_before_store[1] = ev_T2;
            }
            rc = dgemm_core_locked(ctx, trans ? 1 : 0, 0, nb2, N, kk, -1.0, Ap, lda, B + k0 * ldb, ldb, alpha, dR[alt], ldx, budget, &one, 0, &ex);
            if (rc) return rc;
            add_stats(acc, one, &t_enq);
            ws_max = std::max(ws_max, reserved0 + (size_t)one.plan.workspace_bytes);
            next_scaled = true;
            if (timing) std::fprintf(stderr, "  dtrsm update %lld x %lld x %lld: %.2f ms (%.1f TFLOP/s), %lld x %lld blocks of %lld x %lld, %.2f GB up\n", (long long)nb2, (long long)N,
                                     (long long)kk, 1e3 * one.t_total_s, 2e-12 * (double)nb2 * N * kk / one.t_total_s, (long long)one.plan.h, (long long)one.plan.w,
                                     (long long)one.plan.mb, (long long)one.plan.nb, one.bytes_h2d / 1e9);
        } else {                                                                // the second block row: nothing before the first one
            if ((rc = copy2d(dR[alt], (size_t)ldx * 8, B + q0 * ldb, (size_t)ldb * 8, (size_t)N * 8, (size_t)nb2, s_up))) return rc;
            acc.bytes_h2d += (uint64_t)nb2 * N * 8; ++acc.n_copies_h2d;
            HCL_CUDA(cudaEventRecord(ev_T2, s_up));                             // (covers the block of T and the block row)
        }
        const auto tp1 = std::chrono::steady_clock::now();
        for (int s = 0; s < 2; ++s) HCL_CUDA(cudaEventSynchronize(ev_sol[s]));  // block row bi is solved
        if (timing) std::fprintf(stderr, "dtrsm block row %lld: next block row's upload + out-of-core update %.2f ms, then %.2f ms more for the solve\n", (long long)bi,
                                 1e3 * std::chrono::duration<double>(tp1 - tp0).count(), 1e3 * std::chrono::duration<double>(std::chrono::steady_clock::now() - tp1).count());
        // ---- update 2: B_next <- beta' * B_next - op(T)[next, current] X_current, all in device memory
        HCL_CUDA(cudaStreamWaitEvent(s_sol[0], ev_T2, 0));
        debug_jitter(ctx, s_sol[0]);
        rc = launch_dgemm_tiles(nb2, N, nbi, -1.0, dT2, ldt, dR[cur], ldx, next_scaled ? 1.0 : alpha, dR[alt], ldx, s_sol[0], -1, nullptr, trans ? 1 : 0, 0);
        if (rc) return rc;
        ++acc.n_kernels;
        HCL_CUDA(cudaEventRecord(ev_ready, s_sol[0]));
        scaled = true;
    }
    for (cudaStream_t st : ctx->s_aux) if (st) HCL_CUDA(cudaStreamSynchronize(st));
    if (stats) {
        *stats = acc;
        stats->plan.M = M; stats->plan.N = N; stats->plan.K = M;
        stats->plan.mb = NB; stats->plan.nb = std::min<int64_t>(N, std::max<int64_t>(1024, ((N + nchunk - 1) / nchunk + 63) / 64 * 64)); stats->plan.kb = 128;
        stats->plan.h = nblk; stats->plan.w = (N + stats->plan.nb - 1) / stats->plan.nb; stats->plan.kpanels = 1; stats->plan.n_steps = nblk;
        stats->plan.workspace_bytes = ws_max;
        stats->plan.n_sets = 2;
        stats->plan.ldc_dev = ldx;
        stats->plan.bytes_h2d = acc.bytes_h2d; stats->plan.bytes_d2h = acc.bytes_d2h;
        stats->plan.n_copies_h2d = acc.n_copies_h2d; stats->plan.n_copies_d2h = acc.n_copies_d2h;
        stats->plan.flops = (double)M * (double)M * (double)N;
        stats->t_enqueue_s = t_enq;
        stats->t_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
    }
    return HCLOOC_OK;
}

}  // namespace hclooc
