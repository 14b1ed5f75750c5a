// lu.cu -- LU factorization with partial pivoting on the out-of-core DGEMM ("out-of-core factorizations (LU, QR,
// Cholesky) that use the out-of-core matrix-matrix multiplication (DGEMM) as a fundamental building block"):
//
//     hclooc_dgetrf   P A = L U of a host-resident M x N matrix under a device budget
//     hclDgetrf       the same on a matrix in device memory (the device phase on its own)
//
// LEFT-LOOKING over block columns of NB columns, like the Cholesky of factor.cu: a panel (all M rows x NB columns) lives in device
// memory from its upload to the download of its final values.  For every block column k factored before it, the panel (1) takes
// that block's row interchanges, (2) has its block row k solved against the unit lower triangle L_kk (device DTRSM, L_kk uploaded
// one step ahead), (3) receives  P[below] -= L[below, k] * P[block row k]  as ONE out-of-core DGEMM through the pipeline of
// executor.cu with A streamed from the host and B, C in device memory; then its rows from the diagonal down are factored in
// device memory by recursive halving (the flops in tile-kernel launches and DTRSM, the pivot search in getrf_sm100.cu's panel
// kernel).  The next panel is uploaded meanwhile.
//
// Row interchanges never touch the host matrix during the factorization: block column k of L is stored in the row order that was
// current when it was factored, and step (1) brings the panel into exactly that order before step (3) multiplies with it -- so
// the operands of every product agree without moving the 8 M N bytes to the left of the panel over the link at every panel.  A
// final pass brings each block column of L into the final order (LAPACK's convention: P A = L U with L fully permuted): up,
// one gather kernel, down, uploads and downloads overlapped.
#include <algorithm>
#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <thread>
#include <unordered_map>
#include <vector>
#include "executor.h"

using namespace hclooc;

namespace {

int64_t round_even(int64_t x) { return (x + 1) & ~(int64_t)1; }
size_t round_1k(size_t x) { return (x + 1023) & ~(size_t)1023; }

struct LuState {
    hclooc_ctx* ctx = nullptr;          // debug shaker of the device solves (nullable)
    cudaStream_t st = nullptr;
    long long* h_ipiv = nullptr;        // pinned: pivot rows (global row indices), written by the panel kernel
    long long* d_info = nullptr;
    void* slots = nullptr;
    int gcap = 1;                       // CTAs the slots were sized for (the panel kernel's launch on all M rows)
    unsigned long long bar_base = 0;
    double* tmp = nullptr;              // scratch of the row permutations
    size_t tmp_elems = 0;
    int* arena = nullptr;               // pinned: (source, destination) lists the permutation kernels read; reset at every stream sync
    size_t arena_ints = 0, arena_used = 0;
    int bw = 32;                        // width of the panel kernel's panels
    bool pivots_pending = false;        // a panel kernel has been enqueued since the last synchronisation
    uint64_t n_kernels = 0;
};

int lu_sync(LuState& L) {
    HCL_CUDA(cudaStreamSynchronize(L.st));
    L.arena_used = 0;
    L.pivots_pending = false;
    return HCLOOC_OK;
}

// The interchanges k0 <= k < k1 (row k <-> row h_ipiv[k], global indices) applied, in that order, to the ncols columns at X, whose
// row 0 is global row `row_off`.
int lu_permute(LuState& L, double* X, int64_t ld, int64_t ncols, int64_t k0, int64_t k1, int64_t row_off) {
    if (ncols <= 0 || k1 <= k0) return HCLOOC_OK;
    int rc;
    if (L.pivots_pending && (rc = lu_sync(L))) return rc;
    std::unordered_map<int64_t, int64_t> cur;                // position -> the original row sitting there now
    cur.reserve((size_t)(k1 - k0) * 2);
    for (int64_t k = k0; k < k1; ++k) {
        const int64_t a = k - row_off, b = (int64_t)L.h_ipiv[k] - row_off;
        if (a == b) continue;
        auto ia = cur.find(a), ib = cur.find(b);
        const int64_t ca = ia == cur.end() ? a : ia->second, cb = ib == cur.end() ? b : ib->second;
        cur[a] = cb; cur[b] = ca;
    }
    std::vector<std::pair<int, int>> moves;                  // (destination, source)
    moves.reserve(cur.size());
    for (auto& kv : cur) if (kv.first != kv.second) moves.emplace_back((int)kv.first, (int)kv.second);
    if (moves.empty()) return HCLOOC_OK;
    std::sort(moves.begin(), moves.end());
    const size_t nt = moves.size();
    if (2 * nt > L.arena_ints) return HCLOOC_ERR_INTERNAL;
    if (L.arena_used + 2 * nt > L.arena_ints && (rc = lu_sync(L))) return rc;
    int* src = L.arena + L.arena_used;
    int* dst = src + nt;
    L.arena_used += 2 * nt;
    for (size_t i = 0; i < nt; ++i) { dst[i] = moves[i].first; src[i] = moves[i].second; }
    debug_jitter(L.ctx, L.st);
    return launch_row_permute(X, ld, ncols, (int)nt, src, dst, L.tmp, L.tmp_elems, L.st, &L.n_kernels);
}

int64_t lu_split(int64_t n, int bw) {
    const int64_t unit = n > 256 ? 128 : bw;
    return (n / unit + 1) / 2 * unit;
}

// P A = L U of the m x n block at P (device, ld even) by recursive halving over the columns; P's row 0 is global row `row0`, its
// pivots are number piv0, piv0 + 1, ... (h_ipiv[piv0 + k] = global row exchanged with row row0 + k).
int dev_getrf(LuState& L, double* P, int64_t ld, int64_t m, int64_t n, int64_t row0, int64_t piv0) {
    if (m <= 0 || n <= 0) return HCLOOC_OK;
    int rc;
    if (n <= L.bw) {
        debug_jitter(L.ctx, L.st);
        rc = launch_getrf_panel(P, ld, m, (int)n, L.h_ipiv + piv0, (long long)row0, L.d_info, (long long)piv0, L.slots, L.gcap, &L.bar_base, L.st);
        ++L.n_kernels;
        L.pivots_pending = true;
        return rc;
    }
    const int64_t n1 = lu_split(n, L.bw), n2 = n - n1;
    if ((rc = dev_getrf(L, P, ld, m, n1, row0, piv0))) return rc;
    const int64_t np1 = std::min(m, n1);
    if ((rc = lu_permute(L, P + n1, ld, n2, piv0, piv0 + np1, row0))) return rc;
    //   A12 <- L11^-1 A12
    if ((rc = dev_trsm_ctx(L.ctx, 0, P, ld, /*lower*/ 1, /*trans*/ 0, /*unit*/ 1, P + n1, ld, n2, np1, 1.0, L.st, &L.n_kernels))) return rc;
    if (m > n1) {
        //   A22 <- A22 - A21 A12
        debug_jitter(L.ctx, L.st);
        if ((rc = launch_dgemm_tiles(m - n1, n2, n1, -1.0, P + n1 * ld, ld, P + n1, ld, 1.0, P + n1 * ld + n1, ld, L.st, 0))) return rc;
        ++L.n_kernels;
        if ((rc = dev_getrf(L, P + n1 * ld + n1, ld, m - n1, n2, row0 + n1, piv0 + n1))) return rc;
        const int64_t np2 = std::min(m - n1, n2);
        if ((rc = lu_permute(L, P + n1 * ld, ld, n1, piv0 + n1, piv0 + n1 + np2, row0 + n1))) return rc;
    }
    return HCLOOC_OK;
}

struct PinnedBuf {
    void* p = nullptr;
    ~PinnedBuf() { if (p) cudaFreeHost(p); }
    int alloc(size_t bytes) { HCL_CUDA(cudaHostAlloc(&p, bytes ? bytes : 8, cudaHostAllocDefault)); return HCLOOC_OK; }
};
struct DevBuf {
    void* p = nullptr;
    ~DevBuf() { if (p) cudaFree(p); }
};
struct EventSet {
    std::vector<cudaEvent_t> ev;
    ~EventSet() { for (cudaEvent_t e : ev) if (e) cudaEventDestroy(e); }
    int make(int n) {
        for (int i = 0; i < n; ++i) { cudaEvent_t e; HCL_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming)); ev.push_back(e); }
        return HCLOOC_OK;
    }
};

constexpr size_t LU_ARENA_INTS = (size_t)1 << 18;          // 1 MiB of pinned memory for the permutation lists
constexpr size_t LU_TMP_MAX = (size_t)64 << 20;

// Panel width of hclooc_dgetrf under `budget`: two resident panels (one if a single panel covers the matrix), two L_kk blocks, the
// scratch of the row permutations and the panel kernel's slots in at most 5/8 of the budget; 4096 where that fits.
struct LuShape { int64_t NB, ldp, ldt; int npan; size_t panel_bytes, t_bytes, tmp_bytes, slot_bytes, reserved; };
int lu_shape(int64_t M, int64_t N, size_t budget, LuShape* out) {
    const int gcap = (int)std::min<int64_t>((M + 127) / 128, 192);            // at most one CTA per 128 rows (getrf_panel_shape)
    static const int64_t nb_env = [] { const char* e = std::getenv("HCLOOC_GETRF_NB"); const long v = e ? std::atol(e) : 0; return v >= 32 ? (int64_t)(v / 32 * 32) : (int64_t)0; }();
    const int npan_env = [] { const char* e = std::getenv("HCLOOC_GETRF_PANELS"); const int v = e ? std::atoi(e) : 0; return v == 2 || v == 3 ? v : 0; }();   // knob, read at every call
    // three resident panels where they fit 7/8 of the budget (the pipeline works in what is left: its buffers for K = NB are a few
    // hundred MiB at most): the panel after next is then uploaded a whole iteration ahead; else two in 5/8 (its upload follows the
    // freshest update range by range); one if a single panel covers the matrix
    auto shape = [&](int64_t nb, LuShape* s) {
        s->NB = std::min(nb, N);
        s->ldp = round_even(s->NB); s->ldt = s->ldp;
        s->panel_bytes = round_1k((size_t)M * s->ldp * 8);
        s->tmp_bytes = round_1k(std::min(LU_TMP_MAX, (size_t)2 * s->NB * std::max<int64_t>(s->NB, 32) * 8));
        s->slot_bytes = round_1k(getrf_slot_bytes(gcap));
        const int64_t npanels = (N + s->NB - 1) / s->NB;
        for (int np = npanels >= 3 ? 3 : (int)npanels; np >= (npanels >= 2 ? 2 : 1); --np) {
            if (npan_env && np > npan_env) continue;
            s->npan = np;
            s->t_bytes = np == 1 ? 0 : round_1k((size_t)s->NB * s->ldt * 8);
            s->reserved = np * s->panel_bytes + 2 * s->t_bytes + 2 * s->tmp_bytes + s->slot_bytes + 1024;
            if (s->reserved <= budget / 8 * (np == 3 ? 7 : 5)) return true;
        }
        return false;
    };
    int64_t NB = nb_env ? nb_env : 4096;
    LuShape s;
    while (NB > 128 && !shape(NB, &s)) NB -= 128;
    while (NB > 32 && !shape(NB, &s)) NB -= 32;
    if (!shape(NB, &s)) return HCLOOC_ERR_BUDGET;
    *out = s;
    return HCLOOC_OK;
}

double lu_flops(int64_t M, int64_t N) {
    const double m = (double)M, n = (double)N;
    return M >= N ? m * n * n - n * n * n / 3.0 : n * m * m - m * m * m / 3.0;
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------------------
extern "C" int hclDgetrf(int64_t M, int64_t N, double* dA, int64_t lda, int64_t* ipiv, int64_t* info, hclStream s) {
    if (M < 0) return -1;
    if (N < 0) return -2;
    if (!info) return -6;
    *info = 0;
    if (M == 0 || N == 0) return HCLOOC_OK;
    if (!dA) return -3;
    if (lda < N) return -4;
    if (!ipiv) return -5;
    if (((uintptr_t)dA & 15u) || (lda & 1)) return HCLOOC_ERR_ALIGN;
    if (M > 0x7fffffffLL || N > 0x7fffffffLL) return -1;
    const int64_t n = std::min(M, N);
    int rc, G, rpc;
    LuState L;
    L.st = (cudaStream_t)s;
    L.bw = getrf_panel_shape(M, &G, &rpc);
    if (L.bw < 8) return HCLOOC_ERR_BUDGET;
    PinnedBuf hp, ha;
    if ((rc = hp.alloc((size_t)n * 8 + 64)) || (rc = ha.alloc(LU_ARENA_INTS * 4))) return rc;
    L.h_ipiv = (long long*)hp.p;
    L.arena = (int*)ha.p; L.arena_ints = LU_ARENA_INTS;
    // scratch: the row permutations never touch more than 2 * (half the columns) rows of at most half the columns
    L.gcap = G;
    const size_t slot_bytes = round_1k(getrf_slot_bytes(G));
    const size_t tmp_bytes = round_1k(std::min(LU_TMP_MAX, std::max<size_t>((size_t)N * std::max<int64_t>(N / 2, 32) * 8, (size_t)1 << 16)));
    DevBuf scratch;
    {
        cudaError_t e = cudaMalloc(&scratch.p, slot_bytes + tmp_bytes + 1024);
        if (e != cudaSuccess) { set_last_cuda_error((int)e); cudaGetLastError(); return HCLOOC_ERR_NOMEM; }
    }
    L.slots = scratch.p;
    L.tmp = (double*)((uint8_t*)scratch.p + slot_bytes);
    L.tmp_elems = tmp_bytes / 8;
    L.d_info = (long long*)((uint8_t*)scratch.p + slot_bytes + tmp_bytes);
    HCL_CUDA(cudaMemsetAsync(L.slots, 0, 64, L.st));
    HCL_CUDA(cudaMemsetAsync(L.d_info, 0, 8, L.st));
    rc = dev_getrf(L, dA, lda, M, N, 0, 0);
    long long h_info = 0;
    if (!rc) {
        cudaError_t e = cudaMemcpyAsync(&h_info, L.d_info, 8, cudaMemcpyDeviceToHost, L.st);
        if (e != cudaSuccess) rc = cuda_fail(e);
    }
    { cudaError_t e = cudaStreamSynchronize(L.st); if (e != cudaSuccess && !rc) rc = cuda_fail(e); }
    if (rc) return rc;
    for (int64_t k = 0; k < n; ++k) ipiv[k] = (int64_t)L.h_ipiv[k];
    *info = (int64_t)h_info;
    return HCLOOC_OK;
}

extern "C" int hclooc_dgetrf_plan(int64_t M, int64_t N, size_t device_budget_bytes, int64_t* NB, uint64_t* reserved_bytes) {
    if (M < 1) return -1;
    if (N < 1) return -2;
    if (!NB || !reserved_bytes) return -4;
    LuShape s;
    int rc = lu_shape(M, N, device_budget_bytes, &s);
    if (rc) return rc;
    *NB = s.NB; *reserved_bytes = s.reserved;
    return HCLOOC_OK;
}

extern "C" int hclooc_dgetrf(hclooc_ctx* ctx, int64_t M, int64_t N, double* A, int64_t lda, int64_t* ipiv, size_t device_budget_bytes,
                             int64_t* info, hclooc_stats* stats) {
    const auto t_begin = std::chrono::steady_clock::now();
    if (M < 0) return -2;
    if (N < 0) return -3;
    if (!info) return -8;
    *info = 0;
    if (stats) std::memset(stats, 0, sizeof(*stats));
    if (M == 0 || N == 0) return HCLOOC_OK;
    if (!A) return -4;
    if (lda < N) return -5;
    if (!ipiv) return -6;
    if (M > 0x7fffffffLL || N > 0x7fffffffLL) return -2;
    int rc;
    if (!ctx && (rc = default_ctx(&ctx))) return rc;
    std::lock_guard<std::mutex> lk(ctx->mu);
    HCL_CUDA(cudaSetDevice(ctx->device));
    bool dummy = true;
    if ((rc = check_resident(A, &dummy))) return rc;
    size_t budget = 0;
    bool own = false;
    if ((rc = resolve_budget(ctx, device_budget_bytes, &budget, &own))) return rc;
    LuShape S;
    if ((rc = lu_shape(M, N, budget, &S))) return rc;
    if ((rc = ensure_aux(ctx))) return rc;
    const int64_t n = std::min(M, N), NB = S.NB, ldp = S.ldp, ldt = S.ldt;
    const int64_t npanels = (N + NB - 1) / NB, npiv = (n + NB - 1) / NB;      // block columns; those that hold pivots
    if (own) { if ((rc = ensure_workspace(ctx, budget))) return rc; }
    uint8_t* base = (uint8_t*)ctx->workspace;
    const uintptr_t mis = (uintptr_t)base & 1023u;
    const size_t shift = mis ? 1024 - mis : 0;
    if (S.reserved + shift > ctx->workspace_bytes) return HCLOOC_ERR_BUDGET;
    uint8_t* q = base + shift;
    double* dPan[3];
    for (int i = 0; i < 3; ++i) { dPan[i] = i < S.npan ? (double*)q : dPan[0]; if (i < S.npan) q += S.panel_bytes; }
    double* dT[2];
    dT[0] = (double*)q; q += S.t_bytes;
    dT[1] = (double*)q; q += S.t_bytes;
    // L: the state of this thread's stream (interchanges, DTRSMs, the update from the freshest block); W: the worker's, which
    // factors a panel on a stream of its own while this thread drives the next panel's out-of-core updates through the pipeline
    LuState L, W;
    L.ctx = ctx;
    L.tmp = (double*)q; L.tmp_elems = S.tmp_bytes / 8; q += S.tmp_bytes;
    W.tmp = (double*)q; W.tmp_elems = S.tmp_bytes / 8; q += S.tmp_bytes;
    W.slots = q; q += S.slot_bytes;
    L.d_info = W.d_info = (long long*)q;
    struct Reserve {
        hclooc_ctx* c;
        Reserve(hclooc_ctx* cc, size_t bytes) : c(cc) { c->reserved_bytes = bytes; }
        ~Reserve() { c->reserved_bytes = 0; }
    } guard(ctx, S.reserved + shift);
    int G, rpc;
    W.bw = L.bw = getrf_panel_shape(M, &G, &rpc);
    if (L.bw < 8) return HCLOOC_ERR_BUDGET;
    W.gcap = (int)std::min<int64_t>((M + 127) / 128, 192);
    if (G > W.gcap) return HCLOOC_ERR_INTERNAL;
    PinnedBuf hp, ha, hperm;
    if ((rc = hp.alloc((size_t)n * 8 + 64)) || (rc = ha.alloc(2 * LU_ARENA_INTS * 4)) || (rc = hperm.alloc((size_t)M * 4 * 2))) return rc;
    L.h_ipiv = W.h_ipiv = (long long*)hp.p;
    L.arena = (int*)ha.p; L.arena_ints = LU_ARENA_INTS;
    W.arena = (int*)ha.p + LU_ARENA_INTS; W.arena_ints = LU_ARENA_INTS;
    // streams of this call: four for this thread's device work (interchanges, DTRSMs in column chunks, the freshest update) at a
    // priority between the pipeline's (highest) and the worker's factorization (lowest), so that the latency-bound solves on the
    // critical path are scheduled ahead of the factorization that runs beside them; copies go on the context's streams
    cudaStream_t s_up = ctx->s_aux[1], s_down = ctx->s_aux[2], s_T = ctx->s_aux[3];
    struct OwnStreams {
        cudaStream_t s[5] = {};
        ~OwnStreams() { for (cudaStream_t x : s) if (x) { cudaStreamSynchronize(x); cudaStreamDestroy(x); } }
    } streams;
    {
        int prio_lo = 0, prio_hi = 0;
        HCL_CUDA(cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
        static const int wp = [] { const char* e = std::getenv("HCLOOC_GETRF_WORKER_PRIO"); return e ? std::atoi(e) : 2; }();   // experiment knob: 0 lowest, 1 middle, 2 highest (measured best: 1.24 s against 1.27-1.28 s)
        static const int mp = [] { const char* e = std::getenv("HCLOOC_GETRF_MAIN_PRIO"); return e ? std::atoi(e) : 1; }();
        const int pr[3] = {prio_lo, (prio_lo + prio_hi) / 2, prio_hi};
        for (int i = 0; i < 5; ++i) HCL_CUDA(cudaStreamCreateWithPriority(&streams.s[i], cudaStreamNonBlocking, i < 4 ? pr[mp] : pr[wp]));
    }
    cudaStream_t st = streams.s[0], s_fact = streams.s[4];
    L.st = st;
    W.st = s_fact;
    // the worker's share of the debug shaker: a context of its own for the random delays (the generator is not thread-safe)
    hclooc_ctx shadow;
    shadow.dbg_rng = ctx->dbg_rng ? ctx->dbg_rng * 0x9E3779B97F4A7C15ull + 1 : 0;
    shadow.dbg_poison = ctx->dbg_poison;
    W.ctx = &shadow;
    cudaEvent_t ev_T[2] = {ctx->ev_aux[4], ctx->ev_aux[5]}, ev_Tfree[2] = {ctx->ev_aux[6], ctx->ev_aux[7]};
    EventSet extra;
    if ((rc = extra.make(22))) return rc;
    cudaEvent_t ev_up[3] = {extra.ev[16], extra.ev[17], extra.ev[18]}, ev_down[3] = {extra.ev[19], extra.ev[20], extra.ev[21]};
    cudaEvent_t ev_fresh = extra.ev[0], ev_g = extra.ev[1], ev_u = extra.ev[2], ev_d = extra.ev[3], ev_fact = extra.ev[4];
    cudaEvent_t ev_s0 = extra.ev[5], ev_sol[3] = {extra.ev[6], extra.ev[7], extra.ev[8]}, ev_ftrsm = extra.ev[9];
    cudaEvent_t ev_fchunk[6] = {extra.ev[10], extra.ev[11], extra.ev[12], extra.ev[13], extra.ev[14], extra.ev[15]};
    static const bool timing = std::getenv("HCLOOC_FACTOR_TIMING") != nullptr;
    static const bool lookahead = [] { const char* e = std::getenv("HCLOOC_GETRF_LOOKAHEAD"); return !e || std::atoi(e) != 0; }();
    HCL_CUDA(cudaMemsetAsync(W.slots, 0, 64, st));
    HCL_CUDA(cudaMemsetAsync(L.d_info, 0, 8, st));
    hclooc_stats acc, wacc;                                   // wacc: what the worker counts (merged after it has been joined)
    std::memset(&acc, 0, sizeof(acc));
    std::memset(&wacc, 0, sizeof(wacc));
    double t_enq = 0.0;
    size_t ws_max = S.reserved;
    bool down_pending[3] = {false, false, false}, tfree_recorded[2] = {false, false};
    auto width = [&](int64_t bj) { return std::min(NB, N - bj * NB); };
    // rows [r_lo, r_hi) of panel bj come up into dPan[buf] on s_up, after `after` (nullable: nothing more to wait for)
    auto upload_rows = [&](int64_t bj, int buf, int64_t r_lo, int64_t r_hi, cudaEvent_t after) -> int {
        if (r_hi <= r_lo) return HCLOOC_OK;
        const int64_t c0 = bj * NB, nbj = width(bj);
        if (after) HCL_CUDA(cudaStreamWaitEvent(s_up, after, 0));
        debug_jitter(ctx, s_up);
        debug_poison(ctx, dPan[buf] + r_lo * ldp, ldp, r_hi - r_lo, nbj, s_up);
        int e = copy2d(dPan[buf] + r_lo * ldp, (size_t)ldp * 8, A + r_lo * lda + c0, (size_t)lda * 8, (size_t)nbj * 8, (size_t)(r_hi - r_lo), s_up);
        if (e) return e;
        acc.bytes_h2d += (uint64_t)(r_hi - r_lo) * nbj * 8; ++acc.n_copies_h2d;
        return HCLOOC_OK;
    };
    auto upload = [&](int64_t bj, int buf) -> int {
        if (down_pending[buf]) HCL_CUDA(cudaStreamWaitEvent(s_up, ev_down[buf], 0));      // the buffer's previous tenant has gone down
        int e = upload_rows(bj, buf, 0, M, nullptr);
        if (e) return e;
        HCL_CUDA(cudaEventRecord(ev_up[buf], s_up));
        return HCLOOC_OK;
    };
    // X (pk x ncols, leading dimension ldp) <- T^-1 X, T unit lower: the columns in up to four chunks on as many streams (one
    // chunk's recursion is a chain of small launches that leaves most SMs idle); everything is ordered after and before `st`
    auto solve_chunks = [&](const double* T, int64_t ldT, double* X, int64_t ncols, int64_t pk) -> int {
        const int nch = ncols >= 2048 ? 4 : (ncols >= 1024 ? 2 : 1);
        if (nch == 1) return dev_trsm_ctx(ctx, 0, T, ldT, 1, 0, 1, X, ldp, ncols, pk, 1.0, st, &L.n_kernels);
        const int64_t wc = ((ncols + nch - 1) / nch + 127) / 128 * 128;
        HCL_CUDA(cudaEventRecord(ev_s0, st));
        int c = 0;
        for (int64_t x0 = 0; x0 < ncols; x0 += wc, ++c) {
            cudaStream_t sc = streams.s[c];
            if (c) HCL_CUDA(cudaStreamWaitEvent(sc, ev_s0, 0));
            int e = dev_trsm_ctx(ctx, 0, T, ldT, 1, 0, 1, X + x0, ldp, std::min(wc, ncols - x0), pk, 1.0, sc, &L.n_kernels);
            if (e) return e;
            if (c) HCL_CUDA(cudaEventRecord(ev_sol[c - 1], sc));
        }
        for (int i = 1; i < c; ++i) HCL_CUDA(cudaStreamWaitEvent(st, ev_sol[i - 1], 0));
        return HCLOOC_OK;
    };
    // L_kk (pk x pk, unit lower) of pivot block k comes up from the host into dT[k & 1]
    auto upload_T = [&](int64_t k) -> int {
        const int64_t c0k = k * NB, pk = std::min(NB, n - c0k);
        const int b = (int)(k & 1);
        if (tfree_recorded[b]) HCL_CUDA(cudaStreamWaitEvent(s_T, ev_Tfree[b], 0));
        debug_jitter(ctx, s_T);
        int e = copy2d(dT[b], (size_t)ldt * 8, A + c0k * lda + c0k, (size_t)lda * 8, (size_t)pk * 8, (size_t)pk, s_T);
        if (e) return e;
        acc.bytes_h2d += (uint64_t)pk * pk * 8; ++acc.n_copies_h2d;
        HCL_CUDA(cudaEventRecord(ev_T[b], s_T));
        return HCLOOC_OK;
    };
    // the worker's job: the rows of panel bj from its diagonal down are factored on s_fact (which has been told to wait for the
    // panel's last update), and the finished panel goes down at once
    std::chrono::steady_clock::time_point w_t0, w_t1;
    auto factor_panel = [&](int64_t bj, int buf) -> int {
        w_t0 = std::chrono::steady_clock::now();
        if (cudaSetDevice(ctx->device) != cudaSuccess) return HCLOOC_ERR_CUDA;
        const int64_t c0 = bj * NB, nbj = width(bj);
        int e = HCLOOC_OK;
        if (c0 < n) {
            int g2, r2;
            W.bw = getrf_panel_shape(M - c0, &g2, &r2);           // shorter panels take wider leaves
            e = dev_getrf(W, dPan[buf] + c0 * ldp, ldp, M - c0, nbj, c0, c0);
        }
        if (e) return e;
        HCL_CUDA(cudaEventRecord(ev_fact, s_fact));
        HCL_CUDA(cudaStreamWaitEvent(s_down, ev_fact, 0));
        debug_jitter(W.ctx, s_down);
        if ((e = copy2d(A + c0, (size_t)lda * 8, dPan[buf], (size_t)ldp * 8, (size_t)nbj * 8, (size_t)M, s_down))) return e;
        wacc.bytes_d2h += (uint64_t)M * nbj * 8; ++wacc.n_copies_d2h;
        HCL_CUDA(cudaEventRecord(ev_down[buf], s_down));
        e = lu_sync(W);                                          // the interchanges of the panel are on the host
        w_t1 = std::chrono::steady_clock::now();
        return e;
    };
    struct Worker {
        std::thread th;
        int rc = HCLOOC_OK;
        bool active = false;
        int join() { if (active) { th.join(); active = false; } return rc; }
        ~Worker() { join(); }
    } worker;
    struct Drain {      // whatever happens, nothing of this call is left running when it returns (declared after the worker: runs first... the
        hclooc_ctx* c;  // worker's destructor joins before the streams are drained because it is destroyed later -- so join explicitly)
        Worker* w;
        ~Drain() { w->join(); for (cudaStream_t s : c->s_aux) if (s) cudaStreamSynchronize(s); }
    } drain{ctx, &worker};
    for (int64_t b0 = 0; b0 < std::min<int64_t>(std::max(S.npan - 1, 1), npanels); ++b0)
        if ((rc = upload(b0, (int)b0))) return rc;
    for (int64_t bj = 0; bj < npanels; ++bj) {
        // panel bj sits in buffer cur, panel bj-1 in alt, panel bj+1 goes to (or is in) nxt; `take` is the panel that takes over alt
        const int cur = (int)(bj % S.npan), alt = (int)((bj + S.npan - 1) % S.npan), nxt = (int)((bj + 1) % S.npan);
        const int64_t take = bj + std::max(S.npan - 1, 1);
        const int64_t nbj = width(bj);
        double* dP = dPan[cur];
        const auto tp0 = std::chrono::steady_clock::now();
        // ---- panel bj-1 is factored, its interchanges are known and its download has been enqueued
        if ((rc = worker.join())) return rc;
        if (bj >= 1) down_pending[alt] = true;
        if (timing && bj >= 1) std::fprintf(stderr, "dgetrf panel %lld: factorization %.2f ms (worker)\n", (long long)(bj - 1), 1e3 * std::chrono::duration<double>(w_t1 - w_t0).count());
        HCL_CUDA(cudaStreamWaitEvent(st, ev_up[cur], 0));
        // ---- the update from the FRESHEST block (k = bj-1) comes straight from device memory: panel bj-1 still sits in the other
        // buffer, so neither its download nor the link is waited for
        // (the next panel comes up into that buffer range by range, each as soon as this update has read it: its top rows -- the U
        // part of panel bj-1 -- at once, the diagonal block after the DTRSM, the rest behind the row chunks of the product)
        const bool next = S.npan >= 2 && take < npanels;
        bool next_up = false;
        if (bj >= 1 && bj - 1 < npiv) {
            const int64_t k = bj - 1, c0k = k * NB, pk = std::min(NB, n - c0k), r1 = c0k + pk;
            const double* Lk = dPan[alt] + c0k * ldp;                                // rows c0k.. of panel k: L_kk, then L[r1:M, block k]
            if (next) {
                if (down_pending[alt]) HCL_CUDA(cudaStreamWaitEvent(s_up, ev_down[alt], 0));
                if ((rc = upload_rows(take, alt, 0, c0k, nullptr))) return rc;
            }
            if ((rc = lu_permute(L, dP, ldp, nbj, c0k, c0k + pk, 0))) return rc;
            if ((rc = solve_chunks(Lk, ldp, dP + c0k * ldp, nbj, pk))) return rc;
            HCL_CUDA(cudaEventRecord(ev_ftrsm, st));
            if (next && (rc = upload_rows(take, alt, c0k, r1, ev_ftrsm))) return rc;
            if (M > r1) {
                // (the GPU is these launches': the worker has been joined, the pipeline is idle)
                const int64_t rows = M - r1;
                const int nch = rows >= 16384 ? 6 : (rows >= 4096 ? 4 : 1);
                const int64_t hc = ((rows + nch - 1) / nch + 127) / 128 * 128;
                int c = 0;
                for (int64_t x0 = 0; x0 < rows; x0 += hc, ++c) {
                    const int64_t hh = std::min(hc, rows - x0);
                    debug_jitter(ctx, st);
                    if ((rc = launch_dgemm_tiles(hh, nbj, pk, -1.0, Lk + (pk + x0) * ldp, ldp, dP + c0k * ldp, ldp, 1.0, dP + (r1 + x0) * ldp, ldp, st, -1))) return rc;
                    ++L.n_kernels;
                    if (next) {
                        HCL_CUDA(cudaEventRecord(ev_fchunk[c], st));
                        if ((rc = upload_rows(take, alt, r1 + x0, r1 + x0 + hh, ev_fchunk[c]))) return rc;
                    }
                }
            }
            if (next) { HCL_CUDA(cudaEventRecord(ev_up[alt], s_up)); next_up = true; }
        }
        HCL_CUDA(cudaEventRecord(ev_fresh, st));
        const auto tp1 = std::chrono::steady_clock::now();
        // ---- panel bj is factored by the worker ...
        HCL_CUDA(cudaStreamWaitEvent(s_fact, ev_fresh, 0));
        worker.rc = HCLOOC_OK;
        bool spawned = false;
        if (lookahead) {
            try {                                                // nothing throws across this ABI: no thread to be had -> factor in line
                worker.th = std::thread([&worker, &factor_panel, bj, cur] { worker.rc = factor_panel(bj, cur); });
                worker.active = spawned = true;
            } catch (...) { spawned = false; }
        }
        if (!spawned && (rc = factor_panel(bj, cur))) return rc;
        // ---- ... while panel bj+1 comes up and receives the updates of the blocks BEFORE bj through the pipeline (L from the host)
        if (next && !next_up) {
            HCL_CUDA(cudaStreamWaitEvent(s_up, ev_fresh, 0));                        // nothing of this call still reads the buffer's previous tenant
            if ((rc = upload(take, alt))) return rc;
        }
        if (bj + 1 < npanels) {
            HCL_CUDA(cudaStreamWaitEvent(st, ev_up[nxt], 0));
            if (timing) {
                HCL_CUDA(cudaEventSynchronize(ev_up[nxt]));
                std::fprintf(stderr, "  dgetrf panel %lld is up %.2f ms after the freshest update of panel %lld was enqueued\n", (long long)(bj + 1),
                             1e3 * std::chrono::duration<double>(std::chrono::steady_clock::now() - tp1).count(), (long long)bj);
            }
            double* dQ = dPan[nxt];
            const int64_t nbn = width(bj + 1);
            const int64_t nk = std::min(bj, npiv);
            // block bj-1 must be on the HOST before the pipeline (and the upload of its diagonal block) reads L there: its download
            // was enqueued when its factorization ended, moments ago -- waited for as late as possible
            auto host_has = [&](int64_t k) -> int {
                if (k == bj - 1 && down_pending[alt]) HCL_CUDA(cudaEventSynchronize(ev_down[alt]));
                return HCLOOC_OK;
            };
            if (nk > 0 && ((rc = host_has(0)) || (rc = upload_T(0)))) return rc;
            for (int64_t k = 0; k < nk; ++k) {
                const int64_t c0k = k * NB, pk = std::min(NB, n - c0k), r1 = c0k + pk;
                const int b = (int)(k & 1);
                const auto ts0 = std::chrono::steady_clock::now();
                // (1) the interchanges of block k, over all rows from c0k down
                if ((rc = lu_permute(L, dQ, ldp, nbn, c0k, c0k + pk, 0))) return rc;
                // (2) block row k of the panel:  U_kj <- L_kk^-1 P_k
                HCL_CUDA(cudaStreamWaitEvent(st, ev_T[b], 0));
                if ((rc = solve_chunks(dT[b], ldt, dQ + c0k * ldp, nbn, pk))) return rc;
                HCL_CUDA(cudaEventRecord(ev_Tfree[b], st));
                tfree_recorded[b] = true;
                if (k + 1 < nk && ((rc = host_has(k + 1)) || (rc = upload_T(k + 1)))) return rc;
                // (3) the rows below:  P[r1:M] <- P[r1:M] - L[r1:M, block k] U_kj, L streamed from the host by the pipeline
                if (M > r1) {
                    if ((rc = lu_sync(L))) return rc;
                    if (timing) std::fprintf(stderr, "  dgetrf panel %lld, block %lld: interchanges + DTRSM %.2f ms\n", (long long)(bj + 1), (long long)k,
                                             1e3 * std::chrono::duration<double>(std::chrono::steady_clock::now() - ts0).count());
                    hclooc_stats one;
                    rc = dgemm_core_locked(ctx, 0, 0, M - r1, nbn, pk, -1.0, A + r1 * lda + c0k, lda, dQ + c0k * ldp, ldp, 1.0, dQ + r1 * ldp, ldp, budget, &one);
                    if (rc) return rc;
                    acc.bytes_h2d += one.bytes_h2d; acc.bytes_d2h += one.bytes_d2h; acc.n_kernels += one.n_kernels;
                    acc.n_copies_h2d += one.n_copies_h2d; acc.n_copies_d2h += one.n_copies_d2h; t_enq += one.t_enqueue_s;
                    ws_max = std::max(ws_max, S.reserved + (size_t)one.plan.workspace_bytes);
                    if (timing) std::fprintf(stderr, "  dgetrf panel %lld, block %lld: update %lld x %lld x %lld %.2f ms (%.1f TFLOP/s), %lld x %lld blocks of %lld x %lld\n",
                                             (long long)(bj + 1), (long long)k, (long long)(M - r1), (long long)nbn, (long long)pk, 1e3 * one.t_total_s,
                                             2e-12 * (double)(M - r1) * nbn * pk / one.t_total_s, (long long)one.plan.h, (long long)one.plan.w, (long long)one.plan.mb, (long long)one.plan.nb);
                }
            }
        }
        if (timing) std::fprintf(stderr, "dgetrf iteration %lld: freshest update enqueued in %.2f ms, look-ahead updates of panel %lld %.2f ms\n", (long long)bj,
                                 1e3 * std::chrono::duration<double>(tp1 - tp0).count(), (long long)(bj + 1),
                                 1e3 * std::chrono::duration<double>(std::chrono::steady_clock::now() - tp1).count());
    }
    if ((rc = worker.join())) return rc;
    if ((rc = lu_sync(L))) return rc;
    HCL_CUDA(cudaStreamSynchronize(s_down));
    acc.bytes_d2h += wacc.bytes_d2h; acc.n_copies_d2h += wacc.n_copies_d2h;
    L.n_kernels += W.n_kernels;
    // ---- final pass: block column k of L, rows below its diagonal block, into the final row order (the interchanges of the
    // blocks after it); X = dPan[0], Y = dPan[1]; upload k+1 runs beside download k
    const auto tf0 = std::chrono::steady_clock::now();
    if (S.npan >= 2) {
        int* perm[2] = {(int*)hperm.p, (int*)hperm.p + M};
        bool first = true;
        int which = 0;
        for (int64_t k = 0; k < npiv; ++k) {
            const int64_t c0k = k * NB, pk = std::min(NB, n - c0k), r1 = c0k + pk, rows = M - r1;
            if (rows <= 0 || r1 >= n) break;
            int* pm = perm[which];
            if (!first) HCL_CUDA(cudaEventSynchronize(ev_g));          // (the gather two blocks back has long read its list; this orders k-1's)
            for (int64_t i = 0; i < rows; ++i) pm[i] = (int)i;
            bool moved = false;
            for (int64_t s2 = r1; s2 < n; ++s2) {
                const int64_t p = (int64_t)L.h_ipiv[s2] - r1;
                if (p != s2 - r1) { std::swap(pm[s2 - r1], pm[p]); moved = true; }
            }
            if (!moved) continue;
            if (!first) HCL_CUDA(cudaStreamWaitEvent(s_up, ev_g, 0));                     // X is free once the previous gather has read it
            debug_jitter(ctx, s_up);
            if ((rc = copy2d(dPan[0], (size_t)ldp * 8, A + r1 * lda + c0k, (size_t)lda * 8, (size_t)pk * 8, (size_t)rows, s_up))) return rc;
            acc.bytes_h2d += (uint64_t)rows * pk * 8; ++acc.n_copies_h2d;
            HCL_CUDA(cudaEventRecord(ev_u, s_up));
            HCL_CUDA(cudaStreamWaitEvent(st, ev_u, 0));
            if (!first) HCL_CUDA(cudaStreamWaitEvent(st, ev_d, 0));                       // Y is free once the previous download has read it
            debug_jitter(ctx, st);
            if ((rc = launch_row_gather_all(dPan[0], ldp, pk, rows, pm, dPan[1], ldp, st))) return rc;
            ++L.n_kernels;
            HCL_CUDA(cudaEventRecord(ev_g, st));
            HCL_CUDA(cudaStreamWaitEvent(s_down, ev_g, 0));
            debug_jitter(ctx, s_down);
            if ((rc = copy2d(A + r1 * lda + c0k, (size_t)lda * 8, dPan[1], (size_t)ldp * 8, (size_t)pk * 8, (size_t)rows, s_down))) return rc;
            acc.bytes_d2h += (uint64_t)rows * pk * 8; ++acc.n_copies_d2h;
            HCL_CUDA(cudaEventRecord(ev_d, s_down));
            first = false;
            which ^= 1;
        }
    }
    long long h_info = 0;
    HCL_CUDA(cudaMemcpyAsync(&h_info, L.d_info, 8, cudaMemcpyDeviceToHost, st));
    for (cudaStream_t s : {st, s_up, s_down, s_T}) HCL_CUDA(cudaStreamSynchronize(s));
    if (timing) std::fprintf(stderr, "dgetrf final pass (L into the final row order): %.2f ms\n", 1e3 * std::chrono::duration<double>(std::chrono::steady_clock::now() - tf0).count());
    for (int64_t k = 0; k < n; ++k) ipiv[k] = (int64_t)L.h_ipiv[k];
    *info = (int64_t)h_info;
    if (stats) {
        acc.n_kernels += L.n_kernels;
        *stats = acc;
        stats->plan.M = M; stats->plan.N = N; stats->plan.K = n;
        stats->plan.mb = M; stats->plan.nb = NB; stats->plan.kb = L.bw;
        stats->plan.h = 1; stats->plan.w = npanels; stats->plan.kpanels = 1; stats->plan.n_steps = npanels;
        stats->plan.workspace_bytes = ws_max;
        stats->plan.n_sets = S.npan;
        stats->plan.bytes_h2d = acc.bytes_h2d; stats->plan.bytes_d2h = acc.bytes_d2h;
        stats->plan.n_copies_h2d = acc.n_copies_h2d; stats->plan.n_copies_d2h = acc.n_copies_d2h;
        stats->plan.flops = lu_flops(M, N);
        stats->t_enqueue_s = t_enq;
        stats->t_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
    }
    return HCLOOC_OK;
}
