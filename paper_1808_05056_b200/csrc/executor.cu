// executor.cu -- S0 (validate), S2-S4/S6 (copies), S7 (events) of the hot path, and the context.
//
// The pipeline of PAPER.md:303-313 (five stages S(b_j), S(a_i), S(c_ij), DGEMM, R(c_ij)) on three
// role streams -- one host-to-device copy stream, one device-to-host copy stream, several compute
// streams -- ordered by CUDA events.  The paper's Figure 2 (:182-271) uses two round-robin streams,
// double-buffered A/C and a single B buffer; here a schedule is generated from the plan as an
// explicit operation list (hclooc_schedule) and then issued verbatim, so the hazard rule of :311
// ("data stored in device buffers is not overwritten until kernel executions that operate on the
// data have completed") can be checked on the list itself without a GPU.
#include <algorithm>
#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>
#include "internal.h"
#include "executor.h"

namespace hclooc {

static thread_local int g_last_cuda_error = 0;
void set_last_cuda_error(int e) { g_last_cuda_error = e; }

namespace {

constexpr int DEFAULT_COMPUTE_STREAMS = 8;

// event ids inside a schedule
struct EventIds {
    int n_sets, n_bbuf, n_abuf;
    int up_ready(int c) const { return c; }                  // rA/rC: the uploads of the step using C buffer c have arrived
    int kernel_done(int c) const { return n_sets + c; }      // eA: the kernel writing C buffer c finished
    int c_stored(int c) const { return 2 * n_sets + c; }     // eC: C buffer c is back on the host
    int b_ready(int b) const { return 3 * n_sets + b; }      // rB: B slice buffer b received
    int b_free(int b) const { return 3 * n_sets + n_bbuf + b; }  // every kernel of the column that read B buffer b finished
    // readers of A buffer a record alternately into two events; reader r waits for reader r-2 (same event) first,
    // so the latest record of each event covers every earlier reader of its parity
    int a_free(int a, int parity) const { return 3 * n_sets + 2 * n_bbuf + 2 * a + parity; }
    int count() const { return 3 * n_sets + 2 * n_bbuf + 2 * n_abuf; }
};

// Expand the plan into the operation list.  This is the single source of truth for the executor.
//
// Order of the steps: columns of blocks one after the other (:189-190), rows in SERPENTINE order (down
// the even columns, up the odd ones) so that the A slices still resident when a column ends are the
// first ones the next column needs.  A slices live in an LRU cache of n_abuf device buffers keyed by
// (row slice, K panel); C blocks use n_sets buffers round-robin by step.
void build_schedule(const hclooc_plan_t& P, int ncs, std::vector<hclooc_op_t>& ops) {
    ops.clear();
    if (P.n_steps == 0) return;
    if (P.ksplit < 0) ncs = std::max(1, std::min(ncs, (int)P.n_scratch));   // stream-K steps: one scratch buffer per compute stream
    const int n_sets = P.n_sets, n_abuf = std::max(1, (int)P.n_abuf);
    const EventIds ev{n_sets, P.n_bbuf, n_abuf};
    const bool scale_only = P.scale_only != 0;
    std::vector<char> set_used(n_sets, 0), set_stored(n_sets, 0);
    // K panels p > 0 re-read from the HOST the block that panel p-1 stored there, possibly through another C buffer:
    // per (i, j) block the C buffer whose R(c_ij) wrote it last (-1: not yet stored in this call)
    std::vector<int> stored_through(P.kpanels > 1 ? (size_t)(P.h * P.w) : 0, -1);
    // A-slice cache
    struct ABuf { int64_t row = -1, panel = -1; int64_t last_use = -1; int ready_ev = -1; int64_t readers = 0; };
    std::vector<ABuf> acache(n_abuf);
    auto push = [&](int kind, int stream, int event) -> hclooc_op_t& {
        hclooc_op_t o;
        std::memset(&o, 0, sizeof(o));
        o.kind = kind; o.stream = stream; o.event = event; o.buf = o.buf2 = o.buf3 = -1; o.step = -1;
        ops.push_back(o);
        return ops.back();
    };
    auto cbuf_id = [&](int c) { return n_abuf + c; };
    auto bbuf_id = [&](int b) { return n_abuf + n_sets + b; };
    // wait until every kernel issued so far has finished (the latest kernel of a C buffer finishes after
    // all earlier kernels of that buffer: each waited for the download of its predecessor)
    auto wait_all_kernels = [&](int stream) {
        for (int c = 0; c < n_sets; ++c)
            if (set_used[c]) push(HCLOOC_OP_WAIT, stream, ev.kernel_done(c));
    };
    auto load_b = [&](int64_t p, int64_t j, int b, int64_t kr0, int64_t krows) {
        hclooc_op_t& o = push(HCLOOC_OP_H2D_B, 0, -1);
        o.buf = bbuf_id(b);
        o.r0 = p * P.kb + kr0; o.nr = krows;
        o.c0 = j * P.nb; o.nc = std::min(P.nb, P.N - j * P.nb);
        o.dev_r0 = kr0;
    };
    struct Step { int64_t sl, p, j, i, t, seq; int abuf; bool a_hit; bool uploaded; };
    const int64_t slabs = P.w * P.kpanels;
    auto make_step = [&](int64_t sl, int64_t t, int64_t seq) {
        Step s{};
        s.sl = sl; s.p = sl / P.w; s.j = sl % P.w; s.t = t; s.seq = seq;
        s.i = (sl & 1) ? P.h - 1 - t : t;
        s.abuf = -1; s.a_hit = false; s.uploaded = false;
        return s;
    };
    // ---- the uploads of one step on the H2D stream: S(a_i) unless the slice is cached, S(c_ij) if C is read
    auto issue_uploads = [&](Step& s) {
        const int c = (int)(s.seq % n_sets);
        const int64_t k0 = s.p * P.kb, kk = scale_only ? 0 : std::min(P.kb, P.K - k0);
        const int64_t i0 = s.i * P.mb, mi = std::min(P.mb, P.M - i0);
        const int64_t j0 = s.j * P.nb, nj = std::min(P.nb, P.N - j0);
        const bool cload = P.beta_nonzero || s.p > 0;
        const int64_t idx = s.i + P.h * (s.j + P.w * s.p);
        bool any = false;
        if (!scale_only) {
            int hit = -1, victim = 0;
            for (int a = 0; a < n_abuf; ++a) {
                if (acache[a].row == s.i && acache[a].panel == s.p) hit = a;
                if (acache[a].last_use < acache[victim].last_use) victim = a;
            }
            if (hit >= 0) { s.abuf = hit; s.a_hit = true; }
            else {
                ABuf& ab = acache[victim];
                for (int par = 0; par < 2 && par < ab.readers; ++par)
                    push(HCLOOC_OP_WAIT, 0, ev.a_free(victim, par));                      // Wait(eA): buffer free (:311)
                ab.readers = 0;
                hclooc_op_t& o = push(HCLOOC_OP_H2D_A, 0, -1);                            // S(a_i)
                o.buf = victim; o.r0 = i0; o.nr = mi; o.c0 = k0; o.nc = kk; o.step = idx;
                ab.row = s.i; ab.panel = s.p; ab.ready_ev = ev.up_ready(c);
                s.abuf = victim;
                any = true;
            }
            acache[s.abuf].last_use = s.seq;
        }
        if (cload) {
            if (set_stored[c]) push(HCLOOC_OP_WAIT, 0, ev.c_stored(c));                  // Wait(eC): block is back on the host
            if (s.p > 0) {
                // the host block itself: S(c_ij) of panel p reads what R(c_ij) of panel p-1 wrote.  That download was issued
                // earlier (a whole slab of steps ago) on the in-order D2H stream, so the newest record of its buffer's
                // c_stored event -- that download's own or a later one's -- covers it.
                const int prev = stored_through[(size_t)(s.i + P.h * s.j)];
                if (prev >= 0 && prev != c) push(HCLOOC_OP_WAIT, 0, ev.c_stored(prev));
            }
            hclooc_op_t& o = push(HCLOOC_OP_H2D_C, 0, -1);                                // S(c_ij)
            o.buf = cbuf_id(c); o.r0 = i0; o.nr = mi; o.c0 = j0; o.nc = nj; o.step = idx;
            any = true;
        }
        if (any) push(HCLOOC_OP_RECORD, 0, ev.up_ready(c));                               // Rec(rA), Rec(rC)
        s.uploaded = any;
        return any;
    };
    // ---- DGEMM on a compute stream, then R(c_ij) on the D2H stream
    auto issue_compute = [&](Step& s, bool any_upload, int b, bool last_of_slab) {
        const int c = (int)(s.seq % n_sets);
        const int cs = 2 + (int)(s.seq % ncs);
        const int64_t k0 = s.p * P.kb, kk = scale_only ? 0 : std::min(P.kb, P.K - k0);
        const int64_t i0 = s.i * P.mb, mi = std::min(P.mb, P.M - i0);
        const int64_t j0 = s.j * P.nb, nj = std::min(P.nb, P.N - j0);
        const bool cload = P.beta_nonzero || s.p > 0;
        const int64_t idx = s.i + P.h * (s.j + P.w * s.p);
        if (any_upload) push(HCLOOC_OP_WAIT, cs, ev.up_ready(c));                         // Wait(rA), Wait(rC)
        if (!scale_only && s.a_hit) {
            // cached slice: its upload arrived; and this kernel is ordered after the reader before the previous
            // one (at least a column of steps ago), whose event it is about to record over
            if (acache[s.abuf].ready_ev != ev.up_ready(c)) push(HCLOOC_OP_WAIT, cs, acache[s.abuf].ready_ev);
            if (acache[s.abuf].readers >= 2) push(HCLOOC_OP_WAIT, cs, ev.a_free(s.abuf, (int)(acache[s.abuf].readers & 1)));
        }
        if (!scale_only) push(HCLOOC_OP_WAIT, cs, ev.b_ready(b));                         // Wait(rB)
        if (!cload && set_stored[c]) push(HCLOOC_OP_WAIT, cs, ev.c_stored(c));            // C buffer still draining
        {
            hclooc_op_t& o = push(HCLOOC_OP_GEMM, cs, -1);
            o.buf = scale_only ? -1 : s.abuf; o.buf2 = scale_only ? -1 : bbuf_id(b); o.buf3 = cbuf_id(c);
            o.r0 = i0; o.nr = mi; o.c0 = j0; o.nc = nj; o.k0 = k0; o.kk = kk; o.step = idx;
            o.beta = (s.p > 0) ? 1.0 : -1.0;             // -1: "use the caller's beta" (resolved by the executor)
        }
        push(HCLOOC_OP_RECORD, cs, ev.kernel_done(c));                                    // Rec(eA)
        set_used[c] = 1;
        if (!scale_only) { push(HCLOOC_OP_RECORD, cs, ev.a_free(s.abuf, (int)(acache[s.abuf].readers & 1))); ++acache[s.abuf].readers; }
        push(HCLOOC_OP_WAIT, 1, ev.kernel_done(c));
        if (last_of_slab && P.n_bbuf == 2 && !scale_only) push(HCLOOC_OP_RECORD, 1, ev.b_free(b));  // the column's kernels are done
        {
            hclooc_op_t& o = push(HCLOOC_OP_D2H_C, 1, -1);                                // R(c_ij)
            o.buf = cbuf_id(c); o.r0 = i0; o.nr = mi; o.c0 = j0; o.nc = nj; o.step = idx;
        }
        push(HCLOOC_OP_RECORD, 1, ev.c_stored(c));                                        // Rec(eC)
        set_stored[c] = 1;
        if (!stored_through.empty()) stored_through[(size_t)(s.i + P.h * s.j)] = c;
    };

    // With one B buffer the uploads of the first steps of a column go out BEFORE the B reload, so the link
    // has work while the kernels of the previous column drain (the paper leaves that reload exposed, :236-242).
    // plan.tri (hclooc_dsyrk): blocks that lie wholly in the triangle of C that is not referenced are not steps at all --
    // no upload, no kernel, no download.  A column's steps are its LIVE blocks, in serpentine order.
    auto in_triangle = [&](int64_t i, int64_t j) {
        if (P.tri == 0) return true;
        const int64_t r0 = i * P.mb, r1 = std::min(P.M, r0 + P.mb), c0 = j * P.nb, c1 = std::min(P.N, c0 + P.nb);
        return P.tri == 1 ? c0 <= r1 - 1 : c1 - 1 >= r0;
    };
    std::vector<Step> early;
    std::vector<int64_t> live;
    int64_t seq = 0;
    for (int64_t sl = 0; sl < slabs; ++sl) {
        const int64_t p = sl / P.w, j = sl % P.w;
        const int64_t kk = scale_only ? 0 : std::min(P.kb, P.K - p * P.kb);
        const int b = (int)(sl % P.n_bbuf);
        live.clear();
        for (int64_t t = 0; t < P.h; ++t)
            if (in_triangle((sl & 1) ? P.h - 1 - t : t, j)) live.push_back(t);
        if (live.empty()) live.push_back(0);              // keeps the B slice chain intact; the kernel skips its tiles
        const int64_t hl = (int64_t)live.size();
        // With one B buffer the uploads of the first steps of a column go out BEFORE the B reload, so the link
        // has work while the kernels of the previous column drain (the paper leaves that reload exposed, :236-242).
        const int64_t pre = (P.n_bbuf == 1 && !scale_only) ? early_uploads(hl, n_sets, n_abuf) : 0;
        early.clear();
        if (!scale_only && (P.n_bbuf == 1 || sl == 0)) {
            if (sl > 0) {
                for (int64_t q = 0; q < pre; ++q) {
                    early.push_back(make_step(sl, live[q], seq + q));
                    issue_uploads(early.back());
                }
                wait_all_kernels(0);             // S(b_j) overwrites the single buffer: every kernel of the previous column is done
            }
            load_b(p, j, b, 0, kk);
            push(HCLOOC_OP_RECORD, 0, ev.b_ready(b));
        }
        // next slice, prefetched in chunks during this column when there are two B buffers
        const bool prefetch = !scale_only && P.n_bbuf == 2 && sl + 1 < slabs;
        const int64_t np = (sl + 1) / P.w, nj_idx = (sl + 1) % P.w;
        const int64_t nkk = prefetch ? std::min(P.kb, P.K - np * P.kb) : 0;
        int64_t pf_i0 = 0, nchunks = 0;
        if (prefetch) prefetch_layout(hl, nkk, n_sets, &pf_i0, &nchunks);
        const int nb_buf = (int)((sl + 1) % P.n_bbuf);
        for (int64_t q = 0; q < hl; ++q, ++seq) {
            Step s = (q < (int64_t)early.size()) ? early[q] : make_step(sl, live[q], seq);
            const bool any = (q < (int64_t)early.size()) ? s.uploaded : issue_uploads(s);
            if (prefetch && q >= pf_i0 && q < pf_i0 + nchunks) {
                const int64_t ci = q - pf_i0;
                if (ci == 0 && sl >= 1) push(HCLOOC_OP_WAIT, 0, ev.b_free(nb_buf));   // last read by the column before this one
                const int64_t r_lo = nkk * ci / nchunks, r_hi = nkk * (ci + 1) / nchunks;
                load_b(np, nj_idx, nb_buf, r_lo, r_hi - r_lo);
                if (ci == nchunks - 1) push(HCLOOC_OP_RECORD, 0, ev.b_ready(nb_buf));
            }
            issue_compute(s, any, b, q == hl - 1);
        }
    }
}

}  // namespace
}  // namespace hclooc

using namespace hclooc;


extern "C" int hclooc_schedule(const hclooc_plan_t* plan, int n_compute, hclooc_op_t* ops, size_t max_ops, size_t* n_ops) {
    if (!plan) return -1;
    if (n_compute < 1 || n_compute > MAX_COMPUTE_STREAMS) return -2;
    if (!n_ops) return -5;
    std::vector<hclooc_op_t> v;
    build_schedule(*plan, n_compute, v);
    *n_ops = v.size();
    if (ops) std::memcpy(ops, v.data(), std::min(max_ops, v.size()) * sizeof(hclooc_op_t));
    return HCLOOC_OK;
}

extern "C" int hclooc_ctx_create(hclooc_ctx** out, int device, void* d_workspace, size_t workspace_bytes,
                                 hclStream stream_h2d, hclStream stream_d2h, hclStream* compute_streams, int n_compute) {
    if (!out) return -1;
    if (device < 0) return -2;
    if ((d_workspace == nullptr) != (workspace_bytes == 0)) return -4;
    if (n_compute < 0 || n_compute > MAX_COMPUTE_STREAMS || ((compute_streams == nullptr) != (n_compute == 0))) return -8;
    HCL_CUDA(cudaSetDevice(device));
    hclooc_ctx* c = new (std::nothrow) hclooc_ctx();
    if (!c) return HCLOOC_ERR_NOMEM;
    c->device = device;
    c->workspace = d_workspace;
    c->workspace_bytes = workspace_bytes;
    c->owns_workspace = false;
    // library-owned streams get the HIGHEST priority: the pipeline is latency sensitive (a kernel that waits for an SM holds its C
    // buffer and with it the uploads behind), while the device phases that run beside it in hclooc_dpotrf / hclooc_dtrsm (big
    // recursive-solve launches on the auxiliary streams, default priority) have slack of a whole pipeline call
    int prio_lo = 0, prio_hi = 0;
    cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);
    auto mk = [prio_hi](cudaStream_t* s) { return cudaStreamCreateWithPriority(s, cudaStreamNonBlocking, prio_hi); };
    cudaError_t e = cudaSuccess;
    if (stream_h2d) c->s_h2d = (cudaStream_t)stream_h2d; else { e = mk(&c->s_h2d); c->owns_h2d = true; }
    if (e == cudaSuccess) { if (stream_d2h) c->s_d2h = (cudaStream_t)stream_d2h; else { e = mk(&c->s_d2h); c->owns_d2h = true; } }
    if (e == cudaSuccess) {
        if (compute_streams) {
            c->n_compute = n_compute;
            for (int i = 0; i < n_compute; ++i) c->s_compute[i] = (cudaStream_t)compute_streams[i];
        } else {
            c->n_compute = DEFAULT_COMPUTE_STREAMS;
            c->owns_compute = true;
            for (int i = 0; i < c->n_compute && e == cudaSuccess; ++i) e = mk(&c->s_compute[i]);
        }
    }
    if (e != cudaSuccess) { hclooc_ctx_destroy(c); return cuda_fail(e); }
    if (const char* j = std::getenv("HCLOOC_DEBUG_JITTER")) { c->dbg_rng = (uint64_t)std::strtoull(j, nullptr, 10); c->dbg_poison = c->dbg_rng != 0; }
    *out = c;
    return HCLOOC_OK;
}

extern "C" int hclooc_ctx_destroy(hclooc_ctx* c) {
    if (!c) return HCLOOC_OK;
    cudaSetDevice(c->device);
    cudaDeviceSynchronize();
    for (cudaEvent_t e : c->events) cudaEventDestroy(e);
    for (cudaEvent_t e : c->trace_events) cudaEventDestroy(e);
    for (cudaEvent_t e : c->join_events) cudaEventDestroy(e);
    if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
    if (c->owns_h2d && c->s_h2d) cudaStreamDestroy(c->s_h2d);
    if (c->owns_d2h && c->s_d2h) cudaStreamDestroy(c->s_d2h);
    if (c->owns_compute) for (int i = 0; i < c->n_compute; ++i) if (c->s_compute[i]) cudaStreamDestroy(c->s_compute[i]);
    if (c->owns_workspace && c->workspace) cudaFree(c->workspace);
    if (c->res_c) cudaFree(c->res_c);
    for (cudaStream_t st : c->s_aux) if (st) cudaStreamDestroy(st);
    for (cudaEvent_t e : c->ev_aux) if (e) cudaEventDestroy(e);
    if (c->h_word) cudaFreeHost(c->h_word);
    delete c;
    return HCLOOC_OK;
}

namespace {
hclooc_ctx* g_default_ctx = nullptr;
std::mutex g_default_mu;
}  // namespace

namespace hclooc {

int default_ctx(hclooc_ctx** out) {
    std::lock_guard<std::mutex> lk(g_default_mu);
    if (!g_default_ctx) {
        int dev = 0;
        HCL_CUDA(cudaGetDevice(&dev));
        int rc = hclooc_ctx_create(&g_default_ctx, dev, nullptr, 0, nullptr, nullptr, nullptr, 0);
        if (rc) return rc;
    }
    *out = g_default_ctx;
    return HCLOOC_OK;
}

// 0 = ok, HCLOOC_ERR_NOT_PINNED if pageable host memory; *on_device is cleared unless p is device memory;
// *dev_alias (nullable) = the address under which kernels on the device reach p (NULL if they cannot)
int check_resident(const void* p, bool* on_device, const void** dev_alias) {
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, p);
    if (e != cudaSuccess) { cudaGetLastError(); return HCLOOC_ERR_NOT_PINNED; }
    if (at.type == cudaMemoryTypeUnregistered) return HCLOOC_ERR_NOT_PINNED;
    if (at.type != cudaMemoryTypeDevice) *on_device = false;
    if (dev_alias) *dev_alias = at.devicePointer;
    return HCLOOC_OK;
}

bool overlaps(const double* a, int64_t rows_a, int64_t cols_a, int64_t lda, const double* b, int64_t rows_b, int64_t cols_b, int64_t ldb) {
    if (rows_a == 0 || cols_a == 0 || rows_b == 0 || cols_b == 0) return false;
    const uintptr_t a0 = (uintptr_t)a, a1 = a0 + 8 * (uintptr_t)((rows_a - 1) * lda + cols_a);
    const uintptr_t b0 = (uintptr_t)b, b1 = b0 + 8 * (uintptr_t)((rows_b - 1) * ldb + cols_b);
    return a0 < b1 && b0 < a1;
}

int copy2d(void* dst, size_t dpitch, const void* src, size_t spitch, size_t width, size_t rows, cudaStream_t s) {
    if (width == 0 || rows == 0) return HCLOOC_OK;
    if (dpitch == width && spitch == width) HCL_CUDA(cudaMemcpyAsync(dst, src, width * rows, cudaMemcpyDefault, s));
    else HCL_CUDA(cudaMemcpy2DAsync(dst, dpitch, src, spitch, width, rows, cudaMemcpyDefault, s));
    return HCLOOC_OK;
}

// tri != 0 (hclooc_dsyrk): only the lower (1) / upper (2) triangle of this call's C, whose element (0, 0) lies on the diagonal,
// is referenced.  The kernels skip the other triangle; its elements still ride along in the C blocks that cross the
// diagonal, which is why such a call uploads its C blocks even when beta == 0 (they come back unchanged).
int dgemm_core(hclooc_ctx* ctx, int transa, int transb, int64_t M, int64_t N, int64_t K, double alpha, const double* A,
               int64_t lda, const double* B, int64_t ldb, double beta, double* C, int64_t ldc,
               size_t device_budget_bytes, hclooc_stats* stats, int tri) {
    // argument errors and the quick returns need no context (and must not create one: validation touches no device)
    int rc = dgemm_core_locked(nullptr, transa, transb, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, device_budget_bytes, stats, tri);
    if (rc != HCLOOC_ERR_INTERNAL + 1000) return rc;
    if (!ctx && (rc = default_ctx(&ctx))) return rc;
    std::lock_guard<std::mutex> lk(ctx->mu);
    return dgemm_core_locked(ctx, transa, transb, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, device_budget_bytes, stats, tri);
}

// the same with ctx->mu already held by the caller (a routine that keeps one lock over all its DGEMM calls and its own
// device work between them: hclooc_dtrsm, hclooc_dpotrf); ctx must not be NULL
int dgemm_core_locked(hclooc_ctx* ctx, int transa, int transb, int64_t M, int64_t N, int64_t K, double alpha, const double* A,
                      int64_t lda, const double* B, int64_t ldb, double beta, double* C, int64_t ldc,
                      size_t device_budget_bytes, hclooc_stats* stats, int tri, const DgemmExtra* extra) {
    const auto t_begin = std::chrono::steady_clock::now();
    // ---------------------------------------------------------------- S0 validate (argument numbers of hclooc_dgemm)
    if (M < 0) return -1;
    if (N < 0) return -2;
    if (K < 0) return -3;
    if (stats) std::memset(stats, 0, sizeof(*stats));
    if (M == 0 || N == 0) return HCLOOC_OK;
    const bool scale_only = (alpha == 0.0 || K == 0);
    // stored shapes: op(A) is M x K, so A is K x M when transposed; op(B) is K x N, so B is N x K when transposed
    const int64_t a_rows = transa ? K : M, a_cols = transa ? M : K, b_rows = transb ? N : K, b_cols = transb ? K : N;
    if (!scale_only) {
        if (!A) return -5;
        if (lda < a_cols) return -6;
        if (!B) return -7;
        if (ldb < b_cols) return -8;
    }
    if (!C) return -10;
    if (ldc < N) return -11;
    if (!scale_only && !(extra && extra->in_place) &&
        (overlaps(C, M, N, ldc, A, a_rows, a_cols, lda) || overlaps(C, M, N, ldc, B, b_rows, b_cols, ldb))) return -10;
    if (scale_only && beta == 1.0) return HCLOOC_OK;            // C = 1*C
    if (scale_only) transa = transb = 0;                        // A and B are not referenced
    if (!ctx) return HCLOOC_ERR_INTERNAL + 1000;                // validation-only pass of dgemm_core: the arguments are fine
    int rc;
    HCL_CUDA(cudaSetDevice(ctx->device));
    bool on_device = true, c_dev = true, a_dev = true, b_dev = true;
    const void *A_alias = nullptr, *B_alias = nullptr, *C_alias = nullptr;
    if ((rc = check_resident(C, &c_dev, &C_alias))) return rc;
    if (!scale_only && ((rc = check_resident(A, &a_dev, &A_alias)) || (rc = check_resident(B, &b_dev, &B_alias)))) return rc;
    const bool ab_dev = a_dev && b_dev;
    on_device = c_dev && ab_dev;

    // ---------------------------------------------------------------- S1 plan
    size_t budget = device_budget_bytes;
    if (!ctx->owns_workspace && ctx->workspace) {
        budget = (budget == 0) ? ctx->workspace_bytes : std::min(budget, ctx->workspace_bytes);
    } else if (budget == 0) {
        size_t fr = 0, tot = 0;
        HCL_CUDA(cudaMemGetInfo(&fr, &tot));
        fr += ctx->workspace_bytes;                                // what we already hold counts as free
        const size_t margin = (size_t)1 << 30;
        budget = fr > 2 * margin ? fr - margin : fr / 2;
    }
    const size_t reserved = ctx->reserved_bytes;
    if (reserved) {
        if (budget <= reserved) return HCLOOC_ERR_BUDGET;
        budget -= reserved;
    }
    hclooc_plan_t P;
    // in-core case: every operand already in device memory and addressable by the tile kernel as it is
    const bool aligned = (((uintptr_t)C & 15u) == 0) && (ldc % 2 == 0) &&
                         (scale_only || ((((uintptr_t)A | (uintptr_t)B) & 15u) == 0 && lda % 2 == 0 && ldb % 2 == 0));
    const bool masked = extra && (extra->amask || extra->bmask || extra->in_place);     // triangular operands: the staged pipeline only
    const bool in_core = on_device && aligned && !masked && M <= 0x7fffffffLL && N <= 0x7fffffffLL && K <= 0x7fffffffLL;
    // direct mode needs host matrices the kernel can address as they are: mapped, TMA-legal, host/device address
    // arithmetic interchangeable (the alias of the first element is what the tensor maps are built on)
    static const int direct_env = [] { const char* e = std::getenv("HCLOOC_DIRECT"); return e ? std::atoi(e) : -1; }();
    const int direct_mode = ctx->direct_mode >= 0 ? ctx->direct_mode : direct_env;
    if (direct_mode != 0) {
        static std::once_flag once;
        std::call_once(once, [] { set_planner_max_cluster(direct_max_cluster()); });
    }
    const bool direct_ok = !in_core && !c_dev && aligned && !masked && direct_mode != 0 && M <= 0x7fffffffLL && N <= 0x7fffffffLL && K <= 0x7fffffffLL &&
                           C_alias && (((uintptr_t)C_alias & 15u) == 0) &&
                           (scale_only || (A_alias && B_alias && ((((uintptr_t)A_alias | (uintptr_t)B_alias) & 15u) == 0)));
    {
        const bool c_in_host = extra && extra->C_src;
        if (c_in_host && (!c_dev || in_core || beta == 0.0 || scale_only)) return HCLOOC_ERR_INTERNAL;
        const int where = in_core ? 1 : (c_dev ? (c_in_host ? 5 : 2) : (direct_ok ? (direct_mode == 1 ? 4 : 3) : 0));
        const hclooc_ctx::PlanKey key{M, N, K, beta != 0.0 || tri != 0, alpha == 0.0, where + (transa ? 8 : 0) + (transb ? 16 : 0) + 32 * tri, budget};
        bool hit = false;
        for (const auto& kv : ctx->plan_cache) {
            const hclooc_ctx::PlanKey& k = kv.first;
            if (k.M == key.M && k.N == key.N && k.K == key.K && k.beta_nz == key.beta_nz && k.alpha_zero == key.alpha_zero &&
                k.where == key.where && k.budget == key.budget) { P = kv.second; hit = true; break; }
        }
        if (!hit) {
            rc = plan_impl(M, N, K, key.beta_nz, key.alpha_zero, budget, where, transa, transb, &P);
            if (rc) return rc;
            P.tri = tri;
            if (ctx->plan_cache.size() >= 16) ctx->plan_cache.erase(ctx->plan_cache.begin());
            ctx->plan_cache.emplace_back(key, P);
        }
    }
    if (extra && extra->in_place && P.kpanels > 1) return HCLOOC_ERR_BUDGET;
    // host matrices that fit the budget: the resident schedule (resident.cu) where its model beats the slice plan's
    if (!in_core && !P.direct && !scale_only && !c_dev && !a_dev && !b_dev && !transa && !transb && tri == 0 && !extra && !reserved) {
        ResidentShape RS;
        if (resident_applies(M, N, K, beta != 0.0, budget, P.t_model_s, &RS)) {
            ctx->graph_key.clear(); ctx->graph_valid = false;
            return dgemm_resident(ctx, RS, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, stats, t_begin);
        }
    }
    if (in_core || P.direct) {
        const auto t0 = std::chrono::steady_clock::now();
        if (P.direct) { A = (const double*)A_alias; B = (const double*)B_alias; C = (double*)C_alias; }
        // direct: one CTA per tile (every tile is bound by its own reads over the link; the persistent kernel's
        // device scratch would also break the promise that the call uses no device memory)
        if (P.direct && P.direct_cm * P.direct_cn > 1 && tri == 0)     // (a masked call always has a transposed operand: no clusters)
            rc = launch_dgemm_direct(M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, ctx->s_compute[0], P.direct_cm, P.direct_cn);
        else
            rc = launch_dgemm_tiles(M, N, scale_only ? 0 : K, scale_only ? 0.0 : alpha, A, lda, B, ldb, beta, C, ldc, ctx->s_compute[0], P.direct ? 1 : -1,
                                    nullptr, transa, transb, tri, 0);
        const auto t1 = std::chrono::steady_clock::now();
        cudaError_t e = cudaStreamSynchronize(ctx->s_compute[0]);
        if (rc) return rc;
        if (e != cudaSuccess) return cuda_fail(e);
        ctx->trace_recs.clear();
        if (stats) {
            stats->plan = P;
            stats->n_kernels = 1;
            stats->bytes_h2d = P.bytes_h2d; stats->bytes_d2h = P.bytes_d2h;      // direct mode: the tiles' own reads and writes
            stats->t_enqueue_s = std::chrono::duration<double>(t1 - t0).count();
            stats->t_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
        }
        return HCLOOC_OK;
    }
    if (reserved && P.workspace_bytes + reserved > ctx->workspace_bytes) return HCLOOC_ERR_BUDGET;   // the caller sized the workspace
    if (!reserved && P.workspace_bytes > ctx->workspace_bytes) {
        if (ctx->workspace && !ctx->owns_workspace) return HCLOOC_ERR_BUDGET;
        if (ctx->workspace) { HCL_CUDA(cudaDeviceSynchronize()); cudaFree(ctx->workspace); ctx->workspace = nullptr; ctx->workspace_bytes = 0; }
        void* p = nullptr;
        cudaError_t e = cudaMalloc(&p, P.workspace_bytes);
        if (e != cudaSuccess) { set_last_cuda_error((int)e); cudaGetLastError(); return HCLOOC_ERR_NOMEM; }
        ctx->workspace = p; ctx->workspace_bytes = P.workspace_bytes; ctx->owns_workspace = true;
    }
    // ---------------------------------------------------------------- buffers carved from the workspace
    uint8_t* base = (uint8_t*)ctx->workspace + reserved;
    const uintptr_t mis = (uintptr_t)base & 1023u;
    if (mis) {   // caller workspace not 1 KiB aligned: shift (costs < 1 KiB, checked against the size)
        base += 1024 - mis;
        if (P.workspace_bytes + reserved + 1024 - mis > ctx->workspace_bytes) return HCLOOC_ERR_BUDGET;
    }
    std::vector<double*> bufs(P.n_abuf + P.n_sets + P.n_bbuf);
    uint8_t* scratch[MAX_COMPUTE_STREAMS] = {};
    if (P.n_scratch > MAX_COMPUTE_STREAMS) return HCLOOC_ERR_INTERNAL;
    {
        uint8_t* q = base;
        for (int b = 0; b < P.n_bbuf; ++b) { bufs[P.n_abuf + P.n_sets + b] = (double*)q; q += P.bytes_b_buf; }
        for (int a = 0; a < P.n_abuf; ++a) { bufs[a] = (double*)q; q += P.bytes_a_buf; }
        for (int c = 0; c < P.n_sets; ++c) { bufs[P.n_abuf + c] = (double*)q; q += P.bytes_c_buf; }
        for (int i = 0; i < P.n_scratch; ++i) { scratch[i] = q; q += P.bytes_scratch; }
        if ((size_t)(q - base) != P.workspace_bytes) return HCLOOC_ERR_INTERNAL;
    }
    // ---------------------------------------------------------------- events
    const size_t n_events = (size_t)EventIds{P.n_sets, P.n_bbuf, std::max(1, (int)P.n_abuf)}.count();
    while (ctx->events.size() < n_events) {
        cudaEvent_t e;
        HCL_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        ctx->events.push_back(e);
    }
    // ---------------------------------------------------------------- S2-S7: issue the schedule
    build_schedule(P, ctx->n_compute, ctx->ops);
    if (P.tri != 0) {
        // blocks outside the referenced triangle are not steps: the traffic of this plan is what its schedule says
        uint64_t up = 0, down = 0, nup = 0, ndown = 0;
        for (const hclooc_op_t& o : ctx->ops) {
            const uint64_t bytes = (uint64_t)o.nr * (uint64_t)o.nc * 8;
            if (o.kind == HCLOOC_OP_H2D_A || o.kind == HCLOOC_OP_H2D_B) { up += bytes; ++nup; }
            else if (o.kind == HCLOOC_OP_H2D_C) { if (!c_dev || (extra && extra->C_src && o.step < P.h * P.w)) up += bytes; ++nup; }
            else if (o.kind == HCLOOC_OP_D2H_C) { if (!c_dev) down += bytes; ++ndown; }
        }
        P.bytes_h2d = up; P.bytes_d2h = down; P.n_copies_h2d = nup; P.n_copies_d2h = ndown;
    }
    for (int i = 0; i < P.n_scratch && i < ctx->n_compute; ++i)   // stream-K tile counters start at zero
        HCL_CUDA(cudaMemsetAsync(scratch[i] + streamk_counter_offset(), 0, streamk_counter_bytes(), ctx->s_compute[i]));
    auto stream_of = [&](int s) { return s == 0 ? ctx->s_h2d : (s == 1 ? ctx->s_d2h : ctx->s_compute[s - 2]); };
    if (extra)       // every store into C goes through the in-order D2H stream: its first one waits for the buffer's previous tenant
        for (cudaEvent_t e : extra->wait_before_store) if (e) HCL_CUDA(cudaStreamWaitEvent(ctx->s_d2h, e, 0));
    uint64_t bytes_h2d = 0, bytes_d2h = 0, n_h2d = 0, n_d2h = 0, n_kernels = 0;
    const auto t_enq0 = std::chrono::steady_clock::now();
    rc = HCLOOC_OK;
    const bool trace = ctx->trace;
    // Latency-bound schedules (many small operations: config 1) are captured once as a CUDA graph and replayed when
    // the very same call comes again; long schedules gain nothing (their enqueue time hides behind the transfers).
    static const int graph_mode = [] { const char* e = std::getenv("HCLOOC_GRAPH"); return e ? std::atoi(e) : -1; }();
    bool use_graph = !trace && !extra && !scale_only && P.n_scratch == 0 && !ctx->dbg_rng && !ctx->dbg_poison &&
                     (graph_mode == 1 || (graph_mode < 0 && P.n_steps <= 512 && P.t_model_s < 5e-3));
    std::vector<int64_t> key;
    if (!use_graph) { ctx->graph_key.clear(); ctx->graph_valid = false; }
    if (use_graph) {
        union { double d; int64_t i; } ua{alpha}, ub{beta};
        key = {M, N, K, ua.i, ub.i, (int64_t)(uintptr_t)A, lda, (int64_t)(uintptr_t)B, ldb, (int64_t)(uintptr_t)C, ldc,
               (int64_t)(uintptr_t)base, (int64_t)P.workspace_bytes, P.mb, P.nb, P.kb, P.n_sets, P.n_abuf, P.n_bbuf, P.ksplit, transa, transb, tri};
        if (key != ctx->graph_key) {
            // first time this call is seen: run it the ordinary way, capture it if it comes again
            ctx->graph_key = key;
            ctx->graph_valid = false;
            use_graph = false;
        } else if (ctx->graph_valid && ctx->graph_exec) {
            HCL_CUDA(cudaGraphLaunch(ctx->graph_exec, ctx->s_h2d));
            const auto t_enq1g = std::chrono::steady_clock::now();
            HCL_CUDA(cudaStreamSynchronize(ctx->s_h2d));
            if (stats) {
                stats->plan = P;
                stats->bytes_h2d = P.bytes_h2d; stats->bytes_d2h = P.bytes_d2h;
                stats->n_kernels = (uint64_t)P.n_steps; stats->n_copies_h2d = P.n_copies_h2d; stats->n_copies_d2h = P.n_copies_d2h;
                stats->t_enqueue_s = std::chrono::duration<double>(t_enq1g - t_enq0).count();
                stats->t_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
            }
            return HCLOOC_OK;
        }
        if (use_graph) HCL_CUDA(cudaStreamBeginCapture(ctx->s_h2d, cudaStreamCaptureModeRelaxed));
    }
    size_t n_traced = 0;
    if (trace) {
        size_t need = 1;
        for (const hclooc_op_t& o : ctx->ops) if (o.kind != HCLOOC_OP_WAIT && o.kind != HCLOOC_OP_RECORD) need += 2;
        while (ctx->trace_events.size() < need) {
            cudaEvent_t e;
            HCL_CUDA(cudaEventCreate(&e));
            ctx->trace_events.push_back(e);
        }
        ctx->trace_recs.clear();
        HCL_CUDA(cudaEventRecord(ctx->trace_events[0], ctx->s_h2d));
    }
    for (const hclooc_op_t& o : ctx->ops) {
        cudaStream_t st = stream_of(o.stream);
        const bool traced = trace && o.kind != HCLOOC_OP_WAIT && o.kind != HCLOOC_OP_RECORD;
        if (traced) {
            cudaEventRecord(ctx->trace_events[1 + 2 * n_traced], st);
            hclooc_trace_rec r;
            std::memset(&r, 0, sizeof(r));
            r.kind = o.kind; r.stream = o.stream; r.step = o.step;
            if (o.kind == HCLOOC_OP_GEMM) r.flops = 2.0 * (double)o.nr * (double)o.nc * (double)o.kk;
            else r.bytes = (uint64_t)o.nr * (uint64_t)o.nc * 8;
            ctx->trace_recs.push_back(r);
        }
        if (ctx->dbg_rng && o.kind != HCLOOC_OP_WAIT && o.kind != HCLOOC_OP_RECORD && !use_graph) debug_jitter(ctx, st);
        if (ctx->dbg_poison && !use_graph) {       // the op list has put every wait this overwrite needs in front of it
            if (o.kind == HCLOOC_OP_H2D_A) debug_poison(ctx, bufs[o.buf], P.lda_dev, transa ? o.nc : o.nr, transa ? o.nr : o.nc, st);
            else if (o.kind == HCLOOC_OP_H2D_B && !transb) debug_poison(ctx, bufs[o.buf] + o.dev_r0 * P.ldb_dev, P.ldb_dev, o.nr, o.nc, st);
            else if (o.kind == HCLOOC_OP_H2D_C) debug_poison(ctx, bufs[o.buf], P.ldc_dev, o.nr, o.nc, st);
        }
        switch (o.kind) {
            case HCLOOC_OP_WAIT: {
                if (ctx->dbg_poison == 2 && o.stream == 0) break;     // sabotage (tests): the upload stream ignores its waits
                cudaError_t e = cudaStreamWaitEvent(st, ctx->events[o.event], 0);
                if (e != cudaSuccess) rc = cuda_fail(e);
                break;
            }
            case HCLOOC_OP_RECORD: {
                cudaError_t e = cudaEventRecord(ctx->events[o.event], st);
                if (e != cudaSuccess) rc = cuda_fail(e);
                break;
            }
            case HCLOOC_OP_H2D_A:
                // A^T: the slice op(A)[r0.., c0..] is the stored block A[c0.., r0..] (k rows x m columns) and stays that way
                if (transa) rc = copy2d(bufs[o.buf], (size_t)P.lda_dev * 8, A + o.c0 * lda + o.r0, (size_t)lda * 8, (size_t)o.nr * 8, (size_t)o.nc, st);
                else rc = copy2d(bufs[o.buf], (size_t)P.lda_dev * 8, A + o.r0 * lda + o.c0, (size_t)lda * 8, (size_t)o.nc * 8, (size_t)o.nr, st);
                bytes_h2d += (uint64_t)o.nr * o.nc * 8; ++n_h2d;
                break;
            case HCLOOC_OP_H2D_B:
                if (transb) {
                    // B^T: the slice is the stored block B[c0.., k0..] (n rows x k columns).  The schedule cuts a prefetched
                    // slice into chunks of k rows [dev_r0, dev_r0 + nr) of kk; for the stored layout those would be narrow
                    // column strips, so the same chunk takes the matching share of the n rows instead (whole k rows of B^T:
                    // contiguous runs); the chunks of a slice still tile it exactly, and b_ready follows the last one.
                    const int64_t k0 = o.r0 - o.dev_r0, kk = std::min(P.kb, K - k0);
                    const int64_t n_lo = o.nc * o.dev_r0 / kk, n_hi = o.nc * (o.dev_r0 + o.nr) / kk;
                    rc = copy2d(bufs[o.buf] + n_lo * P.ldb_dev, (size_t)P.ldb_dev * 8, B + (o.c0 + n_lo) * ldb + k0, (size_t)ldb * 8, (size_t)kk * 8, (size_t)(n_hi - n_lo), st);
                    bytes_h2d += (uint64_t)(n_hi - n_lo) * kk * 8; ++n_h2d;
                    break;
                }
                rc = copy2d(bufs[o.buf] + o.dev_r0 * P.ldb_dev, (size_t)P.ldb_dev * 8, B + o.r0 * ldb + o.c0, (size_t)ldb * 8, (size_t)o.nc * 8, (size_t)o.nr, st);
                bytes_h2d += (uint64_t)o.nr * o.nc * 8; ++n_h2d;
                break;
            case HCLOOC_OP_H2D_C:
                if (extra && extra->C_src && o.step < P.h * P.w) {        // K panel 0: the initial C comes from the host matrix
                    rc = copy2d(bufs[o.buf], (size_t)P.ldc_dev * 8, extra->C_src + o.r0 * extra->ldc_src + o.c0, (size_t)extra->ldc_src * 8, (size_t)o.nc * 8, (size_t)o.nr, st);
                    bytes_h2d += (uint64_t)o.nr * o.nc * 8; ++n_h2d;
                    break;
                }
                rc = copy2d(bufs[o.buf], (size_t)P.ldc_dev * 8, C + o.r0 * ldc + o.c0, (size_t)ldc * 8, (size_t)o.nc * 8, (size_t)o.nr, st);
                if (!c_dev) bytes_h2d += (uint64_t)o.nr * o.nc * 8;   // device-resident C: not link traffic
                ++n_h2d;
                break;
            case HCLOOC_OP_D2H_C:
                rc = copy2d(C + o.r0 * ldc + o.c0, (size_t)ldc * 8, bufs[o.buf], (size_t)P.ldc_dev * 8, (size_t)o.nc * 8, (size_t)o.nr, st);
                if (!c_dev) bytes_d2h += (uint64_t)o.nr * o.nc * 8;
                ++n_d2h;
                if (ctx->dbg_poison && !use_graph) debug_poison(ctx, bufs[o.buf], P.ldc_dev, o.nr, o.nc, st);   // stored: nobody may still want it
                break;
            case HCLOOC_OP_GEMM: {
                const double b_eff = (o.beta < 0.0) ? beta : o.beta;
                rc = launch_dgemm_tiles(o.nr, o.nc, o.kk, scale_only ? 0.0 : alpha, o.buf >= 0 ? bufs[o.buf] : nullptr, P.lda_dev,
                                        o.buf2 >= 0 ? bufs[o.buf2] : nullptr, P.ldb_dev, b_eff, bufs[o.buf3], P.ldc_dev, st,
                                        P.ksplit != 0 ? P.ksplit : 1, P.ksplit < 0 ? scratch[o.stream - 2] : nullptr, transa, transb,
                                        tri, (int)(o.r0 - o.c0), extra ? (extra->amask | (extra->bmask << 2)) : 0,
                                        extra ? (int)(o.r0 - o.k0) + extra->adiag : 0, extra ? (int)(o.k0 - o.c0) + extra->bdiag : 0);
                ++n_kernels;
                break;
            }
            default: rc = HCLOOC_ERR_INTERNAL;
        }
        if (traced) { cudaEventRecord(ctx->trace_events[2 + 2 * n_traced], st); ++n_traced; }
        if (rc) break;
    }
    if (use_graph) {
        // join every stream the capture forked into, end the capture, instantiate and launch
        const int n_other = 1 + ctx->n_compute;
        while ((int)ctx->join_events.size() < n_other) {
            cudaEvent_t e;
            if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) { rc = HCLOOC_ERR_CUDA; break; }
            ctx->join_events.push_back(e);
        }
        for (int i = 0; i < n_other && !rc; ++i) {
            cudaStream_t st = (i == 0) ? ctx->s_d2h : ctx->s_compute[i - 1];
            cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
            if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { rc = HCLOOC_ERR_CUDA; break; }
            if (cs != cudaStreamCaptureStatusActive) continue;
            if (cudaEventRecord(ctx->join_events[i], st) != cudaSuccess || cudaStreamWaitEvent(ctx->s_h2d, ctx->join_events[i], 0) != cudaSuccess) rc = HCLOOC_ERR_CUDA;
        }
        cudaGraph_t graph = nullptr;
        cudaError_t ge = cudaStreamEndCapture(ctx->s_h2d, &graph);
        if (ge != cudaSuccess && !rc) rc = cuda_fail(ge);
        if (!rc) {
            if (ctx->graph_exec) { cudaGraphExecDestroy(ctx->graph_exec); ctx->graph_exec = nullptr; }
            ge = cudaGraphInstantiate(&ctx->graph_exec, graph, 0);
            if (ge != cudaSuccess) rc = cuda_fail(ge);
        }
        if (graph) cudaGraphDestroy(graph);
        if (!rc) {
            ctx->graph_valid = true;
            ge = cudaGraphLaunch(ctx->graph_exec, ctx->s_h2d);
            if (ge != cudaSuccess) rc = cuda_fail(ge);
        } else {
            ctx->graph_key.clear();
            ctx->graph_valid = false;
            cudaGetLastError();
        }
    }
    const auto t_enq1 = std::chrono::steady_clock::now();
    // ---------------------------------------------------------------- final synchronisation (:268-269)
    cudaError_t e1 = cudaStreamSynchronize(ctx->s_d2h);
    cudaError_t e2 = cudaStreamSynchronize(ctx->s_h2d);
    cudaError_t e3 = cudaSuccess;
    for (int i = 0; i < ctx->n_compute && e3 == cudaSuccess; ++i) e3 = cudaStreamSynchronize(ctx->s_compute[i]);
    if (rc) return rc;
    if (e1 != cudaSuccess) return cuda_fail(e1);
    if (e2 != cudaSuccess) return cuda_fail(e2);
    if (e3 != cudaSuccess) return cuda_fail(e3);
    if (trace) {
        for (size_t i = 0; i < n_traced && i < ctx->trace_recs.size(); ++i) {
            float a = 0, b = 0;
            cudaEventElapsedTime(&a, ctx->trace_events[0], ctx->trace_events[1 + 2 * i]);
            cudaEventElapsedTime(&b, ctx->trace_events[0], ctx->trace_events[2 + 2 * i]);
            ctx->trace_recs[i].t_start_ms = a;
            ctx->trace_recs[i].t_end_ms = b;
        }
    }
    if (bytes_h2d != P.bytes_h2d || bytes_d2h != P.bytes_d2h || n_h2d != P.n_copies_h2d || n_d2h != P.n_copies_d2h) return HCLOOC_ERR_INTERNAL;
    if (stats) {
        stats->plan = P;
        stats->bytes_h2d = bytes_h2d; stats->bytes_d2h = bytes_d2h;
        stats->n_kernels = n_kernels; stats->n_copies_h2d = n_h2d; stats->n_copies_d2h = n_d2h;
        stats->t_enqueue_s = std::chrono::duration<double>(t_enq1 - t_enq0).count();
        stats->t_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
    }
    return HCLOOC_OK;
}

}  // namespace

extern "C" int hclooc_dgemm_ex(hclooc_ctx* ctx, int64_t M, int64_t N, int64_t K, double alpha, const double* A,
                               int64_t lda, const double* B, int64_t ldb, double beta, double* C, int64_t ldc,
                               size_t device_budget_bytes, hclooc_stats* stats) {
    return dgemm_core(ctx, 0, 0, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, device_budget_bytes, stats);
}

extern "C" int hclooc_dgemm_t(hclooc_ctx* ctx, int transa, int transb, int64_t M, int64_t N, int64_t K, double alpha,
                              const double* A, int64_t lda, const double* B, int64_t ldb, double beta, double* C, int64_t ldc,
                              size_t device_budget_bytes, hclooc_stats* stats) {
    if (transa != HCL_OP_N && transa != HCL_OP_T) return -15;
    if (transb != HCL_OP_N && transb != HCL_OP_T) return -16;
    return dgemm_core(ctx, transa, transb, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, device_budget_bytes, stats);
}

// Out-of-core DSYRK on top of the DGEMM path: one pass of the pipeline with the triangle mask (plan.tri).
extern "C" int hclooc_dsyrk(hclooc_ctx* ctx, int uplo, int trans, int64_t N, int64_t K, double alpha, const double* A, int64_t lda,
                            double beta, double* C, int64_t ldc, size_t device_budget_bytes, hclooc_stats* stats) {
    const auto t_begin = std::chrono::steady_clock::now();
    if (uplo != HCL_UPLO_LOWER && uplo != HCL_UPLO_UPPER) return -2;
    if (trans != HCL_OP_N && trans != HCL_OP_T) return -3;
    if (N < 0) return -4;
    if (K < 0) return -5;
    if (stats) std::memset(stats, 0, sizeof(*stats));
    if (N == 0) return HCLOOC_OK;
    const bool scale_only = (alpha == 0.0 || K == 0);
    if (!scale_only) {
        if (!A) return -7;
        if (lda < (trans ? N : K)) return -8;
    }
    if (!C) return -10;
    if (ldc < N) return -11;
    if (scale_only && beta == 1.0) return HCLOOC_OK;
    // One pass of the pipeline over the whole N x N problem with the triangle mask: the schedule leaves out the blocks that lie
    // wholly in the other triangle (no upload, kernel or download), the kernels skip such tiles inside the blocks that cross the
    // diagonal and store only referenced elements.  trans == N: A is N x K, the right operand is A read transposed (transb);
    // trans == T: A is K x N, the left operand is A read transposed (transa).
    hclooc_stats acc;
    std::memset(&acc, 0, sizeof(acc));
    int rc = dgemm_core(ctx, trans ? 1 : 0, trans ? 0 : 1, N, N, K, alpha, A, lda, A, lda, beta, C, ldc, device_budget_bytes, &acc,
                        uplo == HCL_UPLO_LOWER ? 1 : 2);
    if (rc) return rc;
    if (stats) {
        *stats = acc;
        stats->t_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
    }
    return HCLOOC_OK;
}

// Out-of-core DSYR2K: two masked passes of the pipeline over the same triangle, the second one accumulating (beta' = 1).
extern "C" int hclooc_dsyr2k(hclooc_ctx* ctx, int uplo, int trans, int64_t N, int64_t K, double alpha, const double* A, int64_t lda,
                             const double* B, int64_t ldb, double beta, double* C, int64_t ldc, size_t device_budget_bytes,
                             hclooc_stats* stats) {
    const auto t_begin = std::chrono::steady_clock::now();
    if (uplo != HCL_UPLO_LOWER && uplo != HCL_UPLO_UPPER) return -2;
    if (trans != HCL_OP_N && trans != HCL_OP_T) return -3;
    if (N < 0) return -4;
    if (K < 0) return -5;
    if (stats) std::memset(stats, 0, sizeof(*stats));
    if (N == 0) return HCLOOC_OK;
    const bool scale_only = (alpha == 0.0 || K == 0);
    if (!scale_only) {
        if (!A) return -7;
        if (lda < (trans ? N : K)) return -8;
        if (!B) return -9;
        if (ldb < (trans ? N : K)) return -10;
    }
    if (!C) return -12;
    if (ldc < N) return -13;
    if (scale_only && beta == 1.0) return HCLOOC_OK;
    const int tri = uplo == HCL_UPLO_LOWER ? 1 : 2, ta = trans ? 1 : 0, tb = trans ? 0 : 1;
    hclooc_stats one, two;
    std::memset(&one, 0, sizeof(one));
    std::memset(&two, 0, sizeof(two));
    // pass 1: C = alpha * op(A) * op(B)^T + beta * C;  pass 2: C = alpha * op(B) * op(A)^T + C   (each on the triangle only)
    int rc = dgemm_core(ctx, ta, tb, N, N, K, alpha, A, lda, B, ldb, beta, C, ldc, device_budget_bytes, &one, tri);
    if (rc) return rc == -10 ? -12 : rc;                          // C overlapping A or B: argument 12 of this function
    if (!scale_only) {
        rc = dgemm_core(ctx, ta, tb, N, N, K, alpha, B, ldb, A, lda, 1.0, C, ldc, device_budget_bytes, &two, tri);
        if (rc) return rc == -10 ? -12 : rc;
    }
    if (stats) {
        *stats = one;
        stats->bytes_h2d += two.bytes_h2d; stats->bytes_d2h += two.bytes_d2h;
        stats->n_kernels += two.n_kernels; stats->n_copies_h2d += two.n_copies_h2d; stats->n_copies_d2h += two.n_copies_d2h;
        stats->t_enqueue_s += two.t_enqueue_s;
        stats->t_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
    }
    return HCLOOC_OK;
}

extern "C" int hclooc_dgemm(int64_t M, int64_t N, int64_t K, double alpha, const double* A, int64_t lda,
                            const double* B, int64_t ldb, double beta, double* C, int64_t ldc, size_t device_budget_bytes) {
    return hclooc_dgemm_ex(nullptr, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, device_budget_bytes, nullptr);
}

// ---------------------------------------------------------------------------------------------
// Out-of-core DTRSM, side = Left (PAPER.md:412 names the routine as future work):
//     solve op(T) * X = alpha * B,  X overwrites B (M x N, host), T = the `uplo` triangle of the M x M host matrix A.
// Blocked substitution, left-looking at the out-of-core level: the rows of B are cut into block rows of NB rows; block row i
// first receives the contribution of the block rows already solved,
//     B_i <- alpha*B_i - op(T)[i, solved] * X[solved]          one out-of-core DGEMM (dgemm_core: K = rows solved so far)
// then its diagonal block is solved in device memory:  T_ii (NB x NB) is uploaded once, B_i streams through two column
// chunks on two streams (upload, solve, download -- each chunk in stream order, the two chunks overlapping), and inside a
// chunk the solve is right-looking over 128-row blocks: trsm_block_kernel on the 128 x 128 triangle, then one tile-kernel
// launch that updates the rows of the chunk still to be solved.  Left-looking outside keeps the traffic at one read of
// X[solved] per block row (2*NB flops per 8 bytes: NB = 4096 is compute bound on this link); right-looking inside gives
// the tile kernel launches of hundreds of tiles instead of 16.
namespace hclooc {

int resolve_budget(hclooc_ctx* ctx, size_t device_budget_bytes, size_t* budget_out, bool* library_owned) {
    size_t budget = device_budget_bytes;
    if (library_owned) *library_owned = ctx->owns_workspace || !ctx->workspace;
    if (!ctx->owns_workspace && ctx->workspace) {
        budget = (budget == 0) ? ctx->workspace_bytes : std::min(budget, ctx->workspace_bytes);
    } else if (budget == 0) {
        size_t fr = 0, tot = 0;
        HCL_CUDA(cudaMemGetInfo(&fr, &tot));
        fr += ctx->workspace_bytes;                                // what we already hold counts as free
        const size_t margin = (size_t)1 << 30;
        budget = fr > 2 * margin ? fr - margin : fr / 2;
    }
    *budget_out = budget;
    return HCLOOC_OK;
}

int ensure_aux(hclooc_ctx* ctx) {
    for (cudaStream_t& st : ctx->s_aux) if (!st) HCL_CUDA(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));
    for (cudaEvent_t& e : ctx->ev_aux) if (!e) HCL_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    if (!ctx->h_word) HCL_CUDA(cudaHostAlloc((void**)&ctx->h_word, 64, cudaHostAllocDefault));
    return HCLOOC_OK;
}

int ensure_workspace(hclooc_ctx* ctx, size_t bytes) {
    if (bytes <= ctx->workspace_bytes) return HCLOOC_OK;
    if (ctx->workspace && !ctx->owns_workspace) return HCLOOC_ERR_BUDGET;
    if (ctx->workspace) { HCL_CUDA(cudaDeviceSynchronize()); cudaFree(ctx->workspace); ctx->workspace = nullptr; ctx->workspace_bytes = 0; }
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, bytes);
    if (e != cudaSuccess) { set_last_cuda_error((int)e); cudaGetLastError(); return HCLOOC_ERR_NOMEM; }
    ctx->workspace = p; ctx->workspace_bytes = bytes; ctx->owns_workspace = true;
    return HCLOOC_OK;
}

}  // namespace hclooc

namespace {

struct TrsmShape { int64_t NB, ldt, wc; size_t bytes; };

// Block-row height NB, chunk width wc and the device bytes of the diagonal phase under `budget`: the triangle buffer takes
// at most half of it, the two chunk buffers of staged mode share the rest.
int trsm_shape(int64_t M, int64_t N, size_t budget, bool library_owned, TrsmShape* out) {
    static const int64_t nb_env = [] { const char* e = std::getenv("HCLOOC_TRSM_NB_MAX"); const long v = e ? std::atol(e) : 0; return v >= 128 ? (int64_t)(v / 128 * 128) : (int64_t)0; }();
    // Block rows of 4096 rows; of 8192 where two of them (one, if that is the whole problem) can stay resident in device memory
    // beside their 512 MiB triangle with a quarter of the budget left: half the X[solved] traffic and updates twice as tall
    // outweigh the longer diagonal phases (32768^2 under 16 GiB: 1.32 s at 4096, 1.20 s at 8192, 1.29 s at 12288, 1.25 s at 16384).
    int64_t NB = 4096;
    if (library_owned && M > 4096) {
        const int64_t nb8 = M < 8192 ? (M + 127) / 128 * 128 : 8192, ldx = (N + 1) & ~(int64_t)1;
        const size_t tb = (size_t)nb8 * nb8 * 8 + 1024, rb = (size_t)nb8 * ldx * 8 + 1024;
        if (tb <= budget / 2 && (M > nb8 ? 2 : 1) * rb + tb + budget / 4 <= budget) NB = 8192;
    }
    if (nb_env) NB = nb_env;                                        // experiment knob
    while (NB > 128 && (size_t)NB * NB * 8 > budget / 2) NB -= 128;
    while (NB > 32 && (size_t)NB * NB * 8 > budget / 2) NB -= 32;
    if (NB > M) NB = M;
    int64_t ldt = (NB + 1) & ~(int64_t)1;
    size_t tbytes = ((size_t)NB * ldt * 8 + 1023) & ~(size_t)1023;
    while (tbytes + 2 * (size_t)NB * 64 * 8 + 4096 > budget) {       // the two narrowest chunk buffers must fit beside the triangle
        if (NB <= 32) return HCLOOC_ERR_BUDGET;
        NB = NB > 128 ? (NB - 1) / 128 * 128 : (NB - 1) / 32 * 32;
        if (NB < 32) return HCLOOC_ERR_BUDGET;
        ldt = (NB + 1) & ~(int64_t)1;
        tbytes = ((size_t)NB * ldt * 8 + 1023) & ~(size_t)1023;
    }
    int64_t wc = (int64_t)((budget - tbytes - 4096) / (2 * (size_t)NB * 8)) / 64 * 64;
    const int64_t npad = (N + 63) / 64 * 64;
    if (wc > npad) wc = npad;
    // two chunks in flight overlap copies with kernels: do not take the whole width in one chunk when N is large
    if (wc == npad && N >= 4096) wc = (npad / 2 + 63) / 64 * 64;
    out->NB = NB; out->ldt = ldt; out->wc = wc;
    out->bytes = tbytes + 2 * (((size_t)NB * wc * 8 + 1023) & ~(size_t)1023);
    return HCLOOC_OK;
}

// Block rows kept resident in device memory (0 = staged mode) and the bytes of one of them: 2 when two fit beside the
// triangle buffer with a quarter of the budget left for the DGEMM pipeline (and there is more than one block row), else 1
// under the same condition, else 0.  Needs device memory the library may allocate itself.
int trsm_resident(int64_t M, int64_t N, size_t budget, const TrsmShape& S, bool library_owned, size_t* rbytes_out) {
    const int64_t ldx = (N + 1) & ~(int64_t)1;
    const size_t rbytes = ((size_t)S.NB * ldx * 8 + 1023) & ~(size_t)1023;
    const size_t tbytes = ((size_t)S.NB * S.ldt * 8 + 1023) & ~(size_t)1023;
    const int64_t nblk = (M + S.NB - 1) / S.NB;
    if (rbytes_out) *rbytes_out = rbytes;
    if (!library_owned) return 0;
    if (nblk > 1 && 2 * rbytes + tbytes + budget / 4 <= budget) return 2;
    if (rbytes + tbytes + budget / 4 <= budget) return 1;
    return 0;
}

}  // namespace

// The shape hclooc_dtrsm works in under a budget -- pure host arithmetic, needs no GPU (include/hclooc.h).
extern "C" int hclooc_dtrsm_plan(int64_t M, int64_t N, size_t device_budget_bytes, int library_owned, int64_t* NB, int64_t* chunk,
                                 int* resident, uint64_t* device_bytes) {
    if (M < 1) return -1;
    if (N < 1) return -2;
    if (!NB || !chunk || !resident || !device_bytes) return -5;
    TrsmShape S;
    int rc = trsm_shape(M, N, device_budget_bytes, library_owned != 0, &S);
    if (rc) return rc;
    size_t rbytes = 0;
    const int nres = trsm_resident(M, N, device_budget_bytes, S, library_owned != 0, &rbytes);
    const size_t tbytes = ((size_t)S.NB * S.ldt * 8 + 1023) & ~(size_t)1023;
    *NB = S.NB; *chunk = S.wc; *resident = nres;
    *device_bytes = nres ? (uint64_t)(nres * rbytes + tbytes) : (uint64_t)(S.bytes + 1024);
    return HCLOOC_OK;
}

extern "C" int hclooc_dtrsm(hclooc_ctx* ctx, int uplo, int trans, int diag, int64_t M, int64_t N, double alpha,
                            const double* A, int64_t lda, double* B, int64_t ldb, size_t device_budget_bytes, hclooc_stats* stats) {
    const auto t_begin = std::chrono::steady_clock::now();
    if (uplo != HCL_UPLO_LOWER && uplo != HCL_UPLO_UPPER) return -2;
    if (trans != HCL_OP_N && trans != HCL_OP_T) return -3;
    if (diag != HCL_DIAG_NONUNIT && diag != HCL_DIAG_UNIT) return -4;
    if (M < 0) return -5;
    if (N < 0) return -6;
    if (stats) std::memset(stats, 0, sizeof(*stats));
    if (M == 0 || N == 0) return HCLOOC_OK;
    if (alpha != 0.0) {
        if (!A) return -8;
        if (lda < M) return -9;
    }
    if (!B) return -10;
    if (ldb < N) return -11;
    if (alpha != 0.0 && overlaps(B, M, N, ldb, A, M, M, lda)) return -10;
    int rc;
    if (alpha == 0.0) {                                              // X = 0, A not referenced, NaN in B not propagated
        rc = dgemm_core(ctx, 0, 0, M, N, 0, 0.0, nullptr, 1, nullptr, 1, 0.0, B, ldb, device_budget_bytes, stats);
        return rc == -10 ? -10 : rc;
    }
    if (!ctx && (rc = default_ctx(&ctx))) return rc;
    size_t budget = device_budget_bytes;
    bool own = false;                                            // may the library allocate device memory of its own?
    {
        std::lock_guard<std::mutex> lk(ctx->mu);
        HCL_CUDA(cudaSetDevice(ctx->device));
        bool dummy = true;
        if ((rc = check_resident(A, &dummy)) || (rc = check_resident(B, &dummy))) return rc;
        own = ctx->owns_workspace || !ctx->workspace;
        if (!ctx->owns_workspace && ctx->workspace) {
            budget = (budget == 0) ? ctx->workspace_bytes : std::min(budget, ctx->workspace_bytes);
        } else if (budget == 0) {
            size_t fr = 0, tot = 0;
            HCL_CUDA(cudaMemGetInfo(&fr, &tot));
            fr += ctx->workspace_bytes;
            const size_t margin = (size_t)1 << 30;
            budget = fr > 2 * margin ? fr - margin : fr / 2;
        }
    }
    TrsmShape S;
    static const int res_env = [] { const char* e = std::getenv("HCLOOC_TRSM_RESIDENT"); return e ? std::atoi(e) : -1; }();
    if (res_env == 0) own = false;                               // experiment knob: staged mode only
    if ((rc = trsm_shape(M, N, budget, own, &S))) return rc;
    const bool lower = (uplo == HCL_UPLO_LOWER) != (trans == HCL_OP_T);       // op(T) is lower triangular
    const int64_t nblk = (M + S.NB - 1) / S.NB;
    hclooc_stats acc;
    std::memset(&acc, 0, sizeof(acc));
    double t_enq = 0.0;
    size_t ws_max = S.bytes;
    const size_t tbytes = ((size_t)S.NB * S.ldt * 8 + 1023) & ~(size_t)1023, cbytes = ((size_t)S.NB * S.wc * 8 + 1023) & ~(size_t)1023;
    // ---- RESIDENT mode: a whole block row (NB x N) stays in device memory from its upload to the download of its solution --
    // the out-of-core DGEMM updates it there (C on the device: its block copies are device-to-device), the diagonal phase solves
    // it in place, and finished column chunks go down on the D2H stream while the next ones are solved.  With room for two
    // block rows the next one is uploaded during the diagonal phase.  Needs library-owned device memory and a quarter of the
    // budget left for the DGEMM pipeline; otherwise the block row is STAGED through two column-chunk buffers after a DGEMM on
    // host C (one more round trip of B over the link).
    const int64_t ldx = (N + 1) & ~(int64_t)1;
    const size_t rbytes = ((size_t)S.NB * ldx * 8 + 1023) & ~(size_t)1023;
    int nres = 0;
    {
        nres = trsm_resident(M, N, budget, S, own, nullptr);
    }
    // two block rows AND two NB x NB blocks of T beside a quarter of the budget for the pipeline: the look-ahead form (factor.cu)
    static const bool no_lookahead = [] { const char* e = std::getenv("HCLOOC_TRSM_LOOKAHEAD"); return e && std::atoi(e) == 0; }();
    if (nres == 2 && !no_lookahead && 2 * rbytes + 2 * tbytes + budget / 4 <= budget) {
        std::lock_guard<std::mutex> lk(ctx->mu);
        rc = dtrsm_left_lookahead(ctx, uplo, trans, diag, M, N, alpha, A, lda, B, ldb, budget, own, S.NB, stats);
        if (!rc && stats) stats->t_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
        return rc;
    }
    struct DevMem { void* p = nullptr; ~DevMem() { if (p) cudaFree(p); } } resmem;
    double* dres[2] = {nullptr, nullptr};
    double* dTres = nullptr;
    size_t budget_dgemm = budget;
    if (nres > 0) {
        cudaError_t e = cudaMalloc(&resmem.p, nres * rbytes + tbytes);
        if (e != cudaSuccess) { set_last_cuda_error((int)e); cudaGetLastError(); resmem.p = nullptr; nres = 0; }
        else {
            dTres = (double*)resmem.p;
            for (int b = 0; b < nres; ++b) dres[b] = (double*)((uint8_t*)resmem.p + tbytes + b * rbytes);
            budget_dgemm = budget - nres * rbytes - tbytes;
            ws_max = nres * rbytes + tbytes;
        }
    }
    // resident mode: T_ii goes up on a stream of its own WHILE the out-of-core update of its block row runs (the update is compute
    // bound and leaves a third of the link idle; the triangle buffer is free since the previous diagonal phase was drained)
    struct Prefetch {
        cudaStream_t s = nullptr; cudaEvent_t e = nullptr;
        ~Prefetch() { if (e) cudaEventDestroy(e); if (s) cudaStreamDestroy(s); }
    } pref;
    if (nres > 0) {
        HCL_CUDA(cudaStreamCreateWithFlags(&pref.s, cudaStreamNonBlocking));
        HCL_CUDA(cudaEventCreateWithFlags(&pref.e, cudaEventDisableTiming));
    }
    const int ns = ctx->n_compute >= 2 ? 2 : 1;                  // staged mode: one stream per chunk buffer
    // resident mode: the chunks of a block row are independent pieces of one buffer, so more of them can be in flight (the
    // triangle kernel is latency bound and leaves most SMs to the other chunks' tile launches)
    static const int ns_env = [] { const char* e = std::getenv("HCLOOC_TRSM_STREAMS"); const int v = e ? std::atoi(e) : 0; return v > 0 ? v : 2; }();
    const int ns_res = nres ? std::max(1, std::min(ns_env, ctx->n_compute)) : ns;
    {
        std::lock_guard<std::mutex> lk(ctx->mu);
        while (ctx->events.size() < 3) {
            cudaEvent_t e;
            HCL_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            ctx->events.push_back(e);
        }
    }
    // the diagonal phase of one column chunk X (nbi rows, w columns, leading dimension ld) in stream st, by recursive halving
    // over 128-row blocks: solve the half that comes first in the order of substitution, subtract its contribution from the
    // other half with ONE tile-kernel launch (K = the half's height: the flops sit in launches with large K, and every row
    // of the chunk is read and written log2(nbi/128) times instead of nbi/256 times), solve the other half; a 128-row block
    // goes to trsm_block_kernel.  `scale` (alpha, when no out-of-core update applied it) reaches every row exactly once: as
    // beta of the first update that touches it, or in the triangle kernel.  One CTA per tile, so that the order of summation
    // does not depend on the chunk width (resident and staged mode give the same bits).
    struct Range { int64_t lo, hi; double scale; int stage; };
    auto solve_chunk = [&](const double* dT, double* X, int64_t ld, int64_t w, int64_t nbi, double alpha_eff, cudaStream_t st) -> int {
        std::vector<Range> stack;
        stack.push_back({0, nbi, alpha_eff, 0});
        while (!stack.empty()) {
            Range r = stack.back();
            stack.pop_back();
            const int64_t rows = r.hi - r.lo;
            if (rows <= 128) {
                int e = launch_trsm_block(dT + r.lo * S.ldt + r.lo, S.ldt, (int)rows, X + r.lo * ld, ld, w, lower ? 1 : 0, trans, diag, r.scale, st);
                if (e) return e;
                ++acc.n_kernels;
                continue;
            }
            const int64_t mid = r.lo + ((rows + 127) / 128 + 1) / 2 * 128;
            // first = the half solved first, second = the half that then receives first's contribution
            const int64_t f0 = lower ? r.lo : mid, f1 = lower ? mid : r.hi, s0 = lower ? mid : r.lo, s1 = lower ? r.hi : mid;
            if (r.stage == 0) {
                stack.push_back({r.lo, r.hi, r.scale, 1});            // come back for the update and the second half
                stack.push_back({f0, f1, r.scale, 0});
            } else {
                const double* Tp = trans ? dT + f0 * S.ldt + s0 : dT + s0 * S.ldt + f0;     // op(T)[second, first] as stored
                int e = launch_dgemm_tiles(s1 - s0, w, f1 - f0, -1.0, Tp, S.ldt, X + f0 * ld, ld, r.scale, X + s0 * ld, ld, st, 1, nullptr, trans ? 1 : 0, 0);
                if (e) return e;
                ++acc.n_kernels;
                stack.push_back({s0, s1, 1.0, 0});
            }
        }
        return HCLOOC_OK;
    };
    for (int64_t bi = 0; bi < nblk; ++bi) {
        const int64_t i = lower ? bi : nblk - 1 - bi;
        const int64_t r0 = i * S.NB, nbi = std::min(S.NB, M - r0), r1 = r0 + nbi;
        // ---- rows already solved: [0, r0) when op(T) is lower, [r1, M) when it is upper
        const int64_t k0 = lower ? 0 : r1, kk = lower ? r0 : M - r1;
        const double* Ap = trans ? A + k0 * lda + r0 : A + r0 * lda + k0;           // op(T)[rows of i, solved rows], as stored
        double alpha_eff = alpha;
        double* dXr = nres ? dres[bi % nres] : nullptr;
        bool t_prefetched = false;
        if (nres) {
            std::lock_guard<std::mutex> lk(ctx->mu);
            HCL_CUDA(cudaSetDevice(ctx->device));
            if (!(nres == 2 && bi > 0)) {                                           // not prefetched during the previous diagonal phase
                if ((rc = copy2d(dXr, (size_t)ldx * 8, B + r0 * ldb, (size_t)ldb * 8, (size_t)N * 8, (size_t)nbi, ctx->s_h2d))) return rc;
                acc.bytes_h2d += (uint64_t)nbi * N * 8; ++acc.n_copies_h2d;
            }
            HCL_CUDA(cudaStreamSynchronize(ctx->s_h2d));                            // the DGEMM's own streams do not wait for this one
            if (kk > 0) {
                if ((rc = copy2d(dTres, (size_t)S.ldt * 8, A + r0 * lda + r0, (size_t)lda * 8, (size_t)nbi * 8, (size_t)nbi, pref.s))) return rc;
                HCL_CUDA(cudaEventRecord(pref.e, pref.s));
                acc.bytes_h2d += (uint64_t)nbi * nbi * 8; ++acc.n_copies_h2d;
                t_prefetched = true;
            }
        }
        const auto tp0 = std::chrono::steady_clock::now();
        if (kk > 0) {
            hclooc_stats one;
            if (nres) rc = dgemm_core(ctx, trans ? 1 : 0, 0, nbi, N, kk, -1.0, Ap, lda, B + k0 * ldb, ldb, alpha, dXr, ldx, budget_dgemm, &one);
            else rc = dgemm_core(ctx, trans ? 1 : 0, 0, nbi, N, kk, -1.0, Ap, lda, B + k0 * ldb, ldb, alpha, B + r0 * ldb, ldb, budget, &one);
            if (rc) return rc;
            acc.bytes_h2d += one.bytes_h2d; acc.bytes_d2h += one.bytes_d2h; acc.n_kernels += one.n_kernels;
            acc.n_copies_h2d += one.n_copies_h2d; acc.n_copies_d2h += one.n_copies_d2h; t_enq += one.t_enqueue_s;
            ws_max = std::max(ws_max, (size_t)one.plan.workspace_bytes + (nres ? nres * rbytes + tbytes : 0));
            alpha_eff = 1.0;
        }
        // ---- the diagonal block, in device memory
        std::lock_guard<std::mutex> lk(ctx->mu);
        HCL_CUDA(cudaSetDevice(ctx->device));
        const auto te0 = std::chrono::steady_clock::now();
        double* dT = dTres;
        double* dX[2] = {nullptr, nullptr};
        if (!nres) {
            if ((rc = ensure_workspace(ctx, S.bytes + 1024))) return rc;
            uint8_t* base = (uint8_t*)ctx->workspace;
            const uintptr_t mis = (uintptr_t)base & 1023u;
            if (mis) base += 1024 - mis;
            dT = (double*)base;
            dX[0] = (double*)(base + tbytes); dX[1] = (double*)(base + tbytes + cbytes);
        }
        if (!t_prefetched) {
            if ((rc = copy2d(dT, (size_t)S.ldt * 8, A + r0 * lda + r0, (size_t)lda * 8, (size_t)nbi * 8, (size_t)nbi, ctx->s_h2d))) return rc;
            HCL_CUDA(cudaEventRecord(ctx->events[0], ctx->s_h2d));
            acc.bytes_h2d += (uint64_t)nbi * nbi * 8; ++acc.n_copies_h2d;
        }
        for (int s = 0; s < ns_res; ++s) HCL_CUDA(cudaStreamWaitEvent(ctx->s_compute[s], t_prefetched ? pref.e : ctx->events[0], 0));
        if (nres == 2 && bi + 1 < nblk) {                                           // the next block row comes up meanwhile
            const int64_t i2 = lower ? bi + 1 : nblk - 2 - bi, q0 = i2 * S.NB, nb2 = std::min(S.NB, M - q0);
            if ((rc = copy2d(dres[(bi + 1) % 2], (size_t)ldx * 8, B + q0 * ldb, (size_t)ldb * 8, (size_t)N * 8, (size_t)nb2, ctx->s_h2d))) return rc;
            acc.bytes_h2d += (uint64_t)nb2 * N * 8; ++acc.n_copies_h2d;
        }
        if (nres) {
            static const int nchunk = [] { const char* e = std::getenv("HCLOOC_TRSM_CHUNKS"); const int v = e ? std::atoi(e) : 0; return v > 0 ? v : 8; }();
            int64_t wr = ((N + nchunk - 1) / nchunk + 63) / 64 * 64;                // about 8 chunks, at least 1024 columns each
            if (wr < 1024) wr = 1024;
            int64_t c = 0;
            for (int64_t c0 = 0; c0 < N; c0 += wr, ++c) {
                const int64_t w = std::min(wr, N - c0);
                cudaStream_t st = ctx->s_compute[c % ns_res];
                if ((rc = solve_chunk(dT, dXr + c0, ldx, w, nbi, alpha_eff, st))) return rc;
                HCL_CUDA(cudaEventRecord(ctx->events[1 + c % 2], st));
                HCL_CUDA(cudaStreamWaitEvent(ctx->s_d2h, ctx->events[1 + c % 2], 0));
                if ((rc = copy2d(B + r0 * ldb + c0, (size_t)ldb * 8, dXr + c0, (size_t)ldx * 8, (size_t)w * 8, (size_t)nbi, ctx->s_d2h))) return rc;
                acc.bytes_d2h += (uint64_t)nbi * w * 8; ++acc.n_copies_d2h;
            }
        } else {
            int64_t c = 0;
            for (int64_t c0 = 0; c0 < N; c0 += S.wc, ++c) {
                const int64_t w = std::min(S.wc, N - c0);
                cudaStream_t st = ctx->s_compute[c % ns];
                double* X = dX[c % 2];
                double* hB = B + r0 * ldb + c0;
                if ((rc = copy2d(X, (size_t)S.wc * 8, hB, (size_t)ldb * 8, (size_t)w * 8, (size_t)nbi, st))) return rc;
                if ((rc = solve_chunk(dT, X, S.wc, w, nbi, alpha_eff, st))) return rc;
                if ((rc = copy2d(hB, (size_t)ldb * 8, X, (size_t)S.wc * 8, (size_t)w * 8, (size_t)nbi, st))) return rc;
                acc.bytes_h2d += (uint64_t)nbi * w * 8; acc.bytes_d2h += (uint64_t)nbi * w * 8; ++acc.n_copies_h2d; ++acc.n_copies_d2h;
            }
        }
        t_enq += std::chrono::duration<double>(std::chrono::steady_clock::now() - te0).count();
        cudaError_t e = cudaSuccess;
        for (int s = 0; s < ns_res; ++s) { cudaError_t e2 = cudaStreamSynchronize(ctx->s_compute[s]); if (e == cudaSuccess) e = e2; }
        { cudaError_t e2 = cudaStreamSynchronize(ctx->s_d2h); if (e == cudaSuccess) e = e2; }
        if (bi + 1 == nblk) { cudaError_t e2 = cudaStreamSynchronize(ctx->s_h2d); if (e == cudaSuccess) e = e2; }
        if (e != cudaSuccess) return cuda_fail(e);
        static const bool timing = std::getenv("HCLOOC_TRSM_TIMING") != nullptr;       // experiment knob: phase times per block row
        if (timing) {
            const auto tp2 = std::chrono::steady_clock::now();
            std::fprintf(stderr, "dtrsm block row %lld: K = %lld, update %.2f ms, diagonal phase %.2f ms\n", (long long)i, (long long)kk,
                         1e3 * std::chrono::duration<double>(te0 - tp0).count(), 1e3 * std::chrono::duration<double>(tp2 - te0).count());
        }
    }
    if (stats) {
        *stats = acc;
        stats->plan.M = M; stats->plan.N = N; stats->plan.K = M;
        stats->plan.mb = S.NB; stats->plan.nb = S.wc; stats->plan.kb = 128;
        stats->plan.h = nblk; stats->plan.w = (N + S.wc - 1) / S.wc; stats->plan.kpanels = 1; stats->plan.n_steps = nblk;
        stats->plan.workspace_bytes = ws_max;
        stats->plan.n_sets = nres;                                  // block rows resident in device memory (0 = staged)
        stats->plan.ldc_dev = nres ? ldx : S.wc;
        stats->plan.bytes_h2d = acc.bytes_h2d; stats->plan.bytes_d2h = acc.bytes_d2h;
        stats->plan.n_copies_h2d = acc.n_copies_h2d; stats->plan.n_copies_d2h = acc.n_copies_d2h;
        stats->plan.flops = (double)M * (double)M * (double)N;
        stats->t_enqueue_s = t_enq;
        stats->t_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
    }
    return HCLOOC_OK;
}

// ---------------------------------------------------------------------------------------------
// nsteps mode: MMOOC as a subroutine of a blocked algorithm (SUMMA, HSUMMA) that updates the
// same C `nsteps` times.  The paper uploads C only at step 0 and downloads it only at the last step; its listing
// of that logic is garbled (:245, :259-263, G17), so the stated intent is implemented: C lives in device
// memory between the calls of one sequence, and every call streams only its A and B.
extern "C" int hclooc_dgemm_nsteps(hclooc_ctx* ctx, int64_t M, int64_t N, int64_t K, double alpha, const double* A,
                                   int64_t lda, const double* B, int64_t ldb, double beta, double* C, int64_t ldc,
                                   size_t device_budget_bytes, int nsteps, int* step, hclooc_stats* stats) {
    const auto t_begin = std::chrono::steady_clock::now();
    if (M <= 0) return -1;
    if (N <= 0) return -2;
    if (K < 0) return -3;
    if (!C) return -10;
    if (ldc < N) return -11;
    if (nsteps < 1) return -13;
    if (!step || *step < 0 || *step >= nsteps) return -14;
    int rc;
    if (!ctx && (rc = default_ctx(&ctx))) return rc;
    const bool first = (*step == 0), last = (*step == nsteps - 1);
    size_t budget = device_budget_bytes;
    uint64_t up = 0, down = 0;
    {
        std::lock_guard<std::mutex> lk(ctx->mu);
        HCL_CUDA(cudaSetDevice(ctx->device));
        if (budget == 0) {
            if (ctx->workspace && !ctx->owns_workspace) budget = ctx->workspace_bytes + ctx->res_bytes;
            else {
                size_t fr = 0, tot = 0;
                HCL_CUDA(cudaMemGetInfo(&fr, &tot));
                fr += ctx->workspace_bytes + ctx->res_bytes;
                budget = fr > ((size_t)2 << 30) ? fr - ((size_t)1 << 30) : fr / 2;
            }
        }
        if (first) {
            if (ctx->res_c) { cudaFree(ctx->res_c); ctx->res_c = nullptr; ctx->res_bytes = 0; }   // an abandoned sequence
            bool dummy = true;
            if ((rc = check_resident(C, &dummy))) return rc;
            const int64_t ld = (N + 15) / 16 * 16;
            const size_t bytes = (size_t)M * ld * 8;
            if (bytes >= budget) return HCLOOC_ERR_BUDGET;          // C itself does not fit: this mode does not apply
            void* p = nullptr;
            cudaError_t e = cudaMalloc(&p, bytes);
            if (e != cudaSuccess) { set_last_cuda_error((int)e); cudaGetLastError(); return HCLOOC_ERR_NOMEM; }
            ctx->res_c = (double*)p; ctx->res_ld = ld; ctx->res_M = M; ctx->res_N = N; ctx->res_host = C; ctx->res_ldc = ldc;
            ctx->res_bytes = bytes;
            if (beta != 0.0) {                                      // S(C) once, at step 0 (:277)
                rc = copy2d(ctx->res_c, (size_t)ld * 8, C, (size_t)ldc * 8, (size_t)N * 8, (size_t)M, ctx->s_h2d);
                cudaError_t es = cudaStreamSynchronize(ctx->s_h2d);
                if (!rc && es != cudaSuccess) rc = cuda_fail(es);
                if (rc) { cudaFree(ctx->res_c); ctx->res_c = nullptr; ctx->res_bytes = 0; return rc; }
                up = (uint64_t)M * N * 8;
            }
        } else if (!ctx->res_c || ctx->res_M != M || ctx->res_N != N || ctx->res_host != C || ctx->res_ldc != ldc) {
            return -10;                                             // not the C of the running sequence
        }
        if (ctx->res_bytes >= budget) return HCLOOC_ERR_BUDGET;
        budget -= ctx->res_bytes;
    }
    rc = hclooc_dgemm_ex(ctx, M, N, K, alpha, A, lda, B, ldb, beta, ctx->res_c, ctx->res_ld, budget, stats);
    {
        std::lock_guard<std::mutex> lk(ctx->mu);
        if (!rc && last) {                                          // R(C) once, at the last step
            rc = copy2d(C, (size_t)ldc * 8, ctx->res_c, (size_t)ctx->res_ld * 8, (size_t)N * 8, (size_t)M, ctx->s_d2h);
            cudaError_t es = cudaStreamSynchronize(ctx->s_d2h);
            if (!rc && es != cudaSuccess) rc = cuda_fail(es);
            down = (uint64_t)M * N * 8;
        }
        if (rc || last) { cudaFree(ctx->res_c); ctx->res_c = nullptr; ctx->res_bytes = 0; }
    }
    if (rc) return rc;
    ++*step;
    if (stats) {
        stats->bytes_h2d += up; stats->bytes_d2h += down;
        stats->n_copies_h2d += up ? 1 : 0; stats->n_copies_d2h += down ? 1 : 0;
        stats->t_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
    }
    return HCLOOC_OK;
}

extern "C" int hclooc_ctx_set_trace(hclooc_ctx* ctx, int enable) {
    int rc;
    if (!ctx && (rc = default_ctx(&ctx))) return rc;
    std::lock_guard<std::mutex> lk(ctx->mu);
    ctx->trace = enable != 0;
    return HCLOOC_OK;
}

// Measures the host link of the current device -- 256 MiB pinned, 4 copies of 64 MiB per direction alone, then both at once -- and
// hands the rates to the planner's cost model (they stay in force for the process; plans cached by contexts are dropped lazily:
// a context re-plans when its cache misses).  About 60 ms.
extern "C" int hclooc_calibrate_link(hclooc_ctx* ctx, double* h2d_GBps, double* d2h_GBps, double* duplex_GBps) {
    int rc;
    if (!ctx && (rc = default_ctx(&ctx))) return rc;
    std::lock_guard<std::mutex> lk(ctx->mu);
    HCL_CUDA(cudaSetDevice(ctx->device));
    const size_t chunk = (size_t)64 << 20, total = 4 * chunk;
    void *ha = nullptr, *hb = nullptr, *da = nullptr, *db = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    double rate[3] = {0, 0, 0};
    cudaError_t e = cudaHostAlloc(&ha, total, cudaHostAllocDefault);
    if (e == cudaSuccess) e = cudaHostAlloc(&hb, total, cudaHostAllocDefault);
    if (e == cudaSuccess) e = cudaMalloc(&da, total);
    if (e == cudaSuccess) e = cudaMalloc(&db, total);
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    if (e == cudaSuccess) {
        std::memset(ha, 0, total);
        for (int mode = 0; mode < 3 && e == cudaSuccess; ++mode) {          // 0: up, 1: down, 2: both
            for (int rep = 0; rep < 2 && e == cudaSuccess; ++rep) {          // the first round warms up
                cudaStreamSynchronize(ctx->s_h2d); cudaStreamSynchronize(ctx->s_d2h);
                const auto t0 = std::chrono::steady_clock::now();
                for (size_t off = 0; off < total; off += chunk) {
                    if (mode != 1) cudaMemcpyAsync((char*)da + off, (char*)ha + off, chunk, cudaMemcpyHostToDevice, ctx->s_h2d);
                    if (mode != 0) cudaMemcpyAsync((char*)hb + off, (char*)db + off, chunk, cudaMemcpyDeviceToHost, ctx->s_d2h);
                }
                e = cudaStreamSynchronize(ctx->s_h2d);
                if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->s_d2h);
                const double t = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
                if (rep == 1) rate[mode] = (mode == 2 ? 2.0 : 1.0) * (double)total / t;
            }
        }
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (da) cudaFree(da);
    if (db) cudaFree(db);
    if (ha) cudaFreeHost(ha);
    if (hb) cudaFreeHost(hb);
    if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail(e); }
    set_machine_link(rate[0], rate[1], rate[2]);
    ctx->plan_cache.clear();
    if (h2d_GBps) *h2d_GBps = rate[0] / 1e9;
    if (d2h_GBps) *d2h_GBps = rate[1] / 1e9;
    if (duplex_GBps) *duplex_GBps = rate[2] / 1e9;
    return HCLOOC_OK;
}

extern "C" int hclooc_ctx_set_debug(hclooc_ctx* ctx, uint64_t jitter_seed, int poison) {
    int rc;
    if (!ctx && (rc = default_ctx(&ctx))) return rc;
    std::lock_guard<std::mutex> lk(ctx->mu);
    ctx->dbg_rng = jitter_seed;
    ctx->dbg_poison = poison == 2 ? 2 : (poison != 0);
    ctx->graph_key.clear(); ctx->graph_valid = false;       // a captured schedule carries no shaker
    return HCLOOC_OK;
}

extern "C" int hclooc_ctx_set_direct(hclooc_ctx* ctx, int mode) {
    int rc;
    if (mode < -1 || mode > 1) return -2;
    if (!ctx && (rc = default_ctx(&ctx))) return rc;
    std::lock_guard<std::mutex> lk(ctx->mu);
    ctx->direct_mode = mode;
    return HCLOOC_OK;
}

extern "C" int hclooc_ctx_get_trace(hclooc_ctx* ctx, hclooc_trace_rec* recs, size_t max_recs, size_t* n_recs) {
    int rc;
    if (!n_recs) return -4;
    if (!ctx && (rc = default_ctx(&ctx))) return rc;
    std::lock_guard<std::mutex> lk(ctx->mu);
    *n_recs = ctx->trace_recs.size();
    if (recs) std::memcpy(recs, ctx->trace_recs.data(), std::min(max_recs, ctx->trace_recs.size()) * sizeof(hclooc_trace_rec));
    return HCLOOC_OK;
}

extern "C" int hclooc_last_cuda_error(void) { return g_last_cuda_error; }
