// resident.cu -- the RESIDENT schedule of hclooc_dgemm: host matrices that FIT the device budget (the paper's "in-core" side of
// the transition point, PAPER.md:130 / :368: N <= 22528 on its 12 GB cards), where the paper uploads everything, runs one kernel
// and downloads, nothing overlapping -- and where a slice pipeline cannot do much better in the balanced regime (link time ~
// flop time, N ~ 8192 under PCIe-class links): every column of blocks needs all of A, so its first block can finish only after
// a third of the traffic has gone up ("Balanced regime").
//
// Here A, B and C get device copies of their own and K is streamed instead:
//   phase 1  A and B go up in K panels (A[:, p] and B[p, :]; graded: 256 or 512 columns first, doubling up to kb, because a short
//            panel starts the kernels early but a whole-C launch pays a fixed prologue + epilogue per tile); as soon as panel p is
//            there the WHOLE of C gets dC (+)= alpha * A[:, p] * B[p, :];
//   phase 2  starts where the kernels would catch up with the uploads (the panel `p_switch`, from the cost model): C is finished
//            ROW BLOCK by row block -- one launch over the remaining panels (alternating between two compute streams, so that
//            one block's launch fills the last wave of the other's), then dC_r += beta * C0_r from a small ring of staging
//            buffers that the upload stream fills behind the operands (the initial C goes up LAST, it is needed last), then the
//            download of the block, under the kernels of the next ones.
// What is left unhidden: the first panel's upload and the last block's download.  The order of summation differs from the slice
// pipeline's (K in panels, beta * C0 added last), so results agree with it to rounding, not to the bit; integer data stays exact.
#include <algorithm>
#include <chrono>
#include <cstdlib>
#include <cstring>
#include "executor.h"

namespace hclooc {

namespace {

// dC[r][c] += beta * dS[r][c] over rows x cols (cols even, both 16-byte aligned): the initial C joins the finished products
__global__ void __launch_bounds__(256) resident_axpy_kernel(double* __restrict__ dC, long long ldc, const double* __restrict__ dS, long long lds,
                                                            int rows, int cols2, double beta) {
    for (int r = blockIdx.y; r < rows; r += gridDim.y) {
        double2* c = reinterpret_cast<double2*>(dC + (long long)r * ldc);
        const double2* s = reinterpret_cast<const double2*>(dS + (long long)r * lds);
        for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < cols2; j += gridDim.x * blockDim.x) {
            double2 x = c[j];
            const double2 y = s[j];
            x.x += beta * y.x;
            x.y += beta * y.y;
            c[j] = x;
        }
    }
}

inline int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }

}  // namespace

bool resident_applies(int64_t M, int64_t N, int64_t K, bool beta_nonzero, size_t budget, double t_slice_model_s, ResidentShape* out) {
    const char* env = std::getenv("HCLOOC_RESIDENT");        // 0: never, 1: whenever it fits; read per call (tests and bench.py flip it)
    const int mode = env ? std::atoi(env) : -1;
    if (mode == 0) return false;
    if (M < 256 || N < 256 || K < 512) return false;
    if (M > 0x7fffffffLL || N > 0x7fffffffLL || K > 0x7fffffffLL) return false;
    // small problems are latency bound: the pipeline's graph replay and direct mode own them (decided below, after the shape)
    const bool small = (double)M * (double)N * (double)K < 8e9 || M < 1024 || N < 1024 || K < 1024;
    const MachineModel& mm = machine_model();
    ResidentShape S;
    std::memset(&S, 0, sizeof(S));
    S.ldA = round_up(K, 16); S.ldB = round_up(N, 16); S.ldC = round_up(N, 16);
    S.bytesA = (size_t)M * S.ldA * 8; S.bytesB = (size_t)K * S.ldB * 8; S.bytesC = (size_t)M * S.ldC * 8;
    S.mb = std::min<int64_t>(M, std::max<int64_t>(128, round_up((M + 15) / 16, 128)));
    S.h = (M + S.mb - 1) / S.mb;
    // K panels GRADED: the first ones small so that the kernels start early (2 KiB rows of A when the call is compute bound, 4 KiB
    // when the link is the bound: narrower 2-D copies lose 3 % of the link), then doubling up to kb: a whole-C launch pays a fixed
    // prologue + epilogue per tile (measured: rate = peak * kk / (kk + 68) -> 0.80 at kk = 256, 0.93 at 1024, 0.97 at 2048)
    const double flops = 2.0 * (double)M * (double)N * (double)K;
    const double link_total = 8.0 * ((double)M * K + (double)K * N + (beta_nonzero ? 2.0 : 1.0) * (double)M * N);
    const bool compute_bound = flops / mm.fp64_flops > std::max(8.0 * ((double)M * K + (double)K * N + (beta_nonzero ? 1.0 : 0.0) * (double)M * N) / mm.h2d_Bps,
                                                                link_total / mm.duplex_Bps);
    int64_t k_first = compute_bound ? 256 : 512;
    S.kb = std::min<int64_t>(std::max<int64_t>(2 * k_first, round_up((K + 7) / 8, 128)), 2048);
    if (const char* e = std::getenv("HCLOOC_RESIDENT_KB")) {      // experiments: uniform panels of this size
        const int64_t v = std::atoll(e);
        if (v >= 32 && v % 32 == 0) S.kb = k_first = v;
    }
    S.npanels = 0;
    for (int64_t k0 = 0, kk = k_first, rep = 0; k0 < K; ) {
        if (S.npanels >= RESIDENT_MAX_PANELS) return false;
        const int64_t take = std::min(kk, K - k0);
        S.pk0[S.npanels] = k0; S.pkk[S.npanels] = take; ++S.npanels;
        k0 += take;
        if (++rep == 2 && kk < S.kb) { kk = std::min(2 * kk, S.kb); rep = 0; }
    }
    if (S.npanels < 2) return false;
    S.bytes_stage = (size_t)S.mb * S.ldC * 8;
    S.bytes_scratch = streamk_scratch_bytes();
    const size_t fixed = S.bytesA + S.bytesB + S.bytesC + S.bytes_scratch + 4096;
    if (fixed > budget) return false;
    S.ring = 0;
    if (beta_nonzero) {
        const int64_t fit = (int64_t)((budget - fixed) / S.bytes_stage);
        S.ring = (int)std::min<int64_t>(S.h, std::min<int64_t>(fit, 8));
        if (S.ring < std::min<int64_t>(S.h, 2)) return false;
    }
    S.total = fixed + (size_t)S.ring * S.bytes_stage;
    // cost model: where the kernels catch up with the uploads, and what the call should take
    auto rate_of = [&](int64_t kk) { return mm.fp64_flops * (double)kk / ((double)kk + 68.0); };
    const double t_up_ab = 8.0 * ((double)M * K + (double)K * N) / mm.h2d_Bps + 2 * S.npanels * mm.copy_latency_s;
    double t_c = 0.0, t_u = 0.0;                         // when the compute stream becomes free / the upload stream has panel p
    int64_t p_sw = S.npanels;
    for (int64_t p = 0; p < S.npanels; ++p) {
        t_u += 8.0 * (double)(M + N) * (double)S.pkk[p] / mm.h2d_Bps + 2 * mm.copy_latency_s;
        const double start = std::max(t_c, t_u);
        if (p > 0 && start >= t_up_ab) { p_sw = p; break; }
        t_c = start + 2.0 * (double)M * (double)N * (double)S.pkk[p] / rate_of(S.pkk[p]) + mm.launch_latency_s;
    }
    if (p_sw >= S.npanels) p_sw = S.npanels - 1;        // the last panel always belongs to phase 2 (it finishes the row blocks)
    S.p_switch = p_sw;
    const int64_t k_rest_m = K - S.pk0[p_sw];
    const double c_bytes = 8.0 * (double)M * (double)N;
    const double t_c0 = beta_nonzero ? c_bytes / mm.h2d_Bps : 0.0, t_down = c_bytes / mm.d2h_Bps;
    const double t_phase2_link = std::max(std::max(t_c0, t_down), ((beta_nonzero ? c_bytes : 0.0) + c_bytes) / mm.duplex_Bps) +
                                 2.0 * (double)S.h * mm.copy_latency_s;
    const double t_rest = 2.0 * (double)M * (double)N * (double)k_rest_m / (0.975 * rate_of(k_rest_m)) + c_bytes * 3.0 / 6e12;
    const double t_compute_path = std::max(t_c, t_up_ab) + t_rest;
    const double t_link_path = t_up_ab + t_phase2_link * (double)(S.h - 1) / (double)S.h;
    const double t_tail = t_down / (double)S.h + mm.copy_latency_s;
    S.t_flop_s = flops / mm.fp64_flops;
    S.t_link_s = std::max(std::max(t_up_ab + t_c0, t_down), (8.0 * ((double)M * K + (double)K * N) + (beta_nonzero ? 2.0 : 1.0) * c_bytes) / mm.duplex_Bps);
    S.t_model_s = std::max(t_compute_path, t_link_path) + t_tail;
    *out = S;
    if (mode > 0) return true;
    if (small) return false;
    if (!(t_slice_model_s > 0.0)) return true;
    // measured against the slice pipeline on the same calls (profiles/r02_transition_sweep.md): both models are within 2 % of the
    // clock, the resident schedule wins by 25 % at N = 8192, 4 % at 12288, 1.3 % at 16384 and ties at 20480
    return S.t_model_s < 0.985 * t_slice_model_s;
}

// The resident schedule as a list of stream operations in host issue order -- the ONE source of what dgemm_resident enqueues
// (hclooc_resident_schedule exports it; tests/test_resident_plan.py runs a vector-clock hazard check over it without a GPU).
// Streams: 0 = uploads, 1 = downloads, 2.. = compute.  Device buffers: 0 = dA, 1 = dB, 2 = dC, 3 + s = staging slot s.
// Events: panel p uploaded [0, np), C0 block r uploaded [np, np + h), staging slot of block r free again [np + h, np + 2h),
// row block r finished [np + 2h, np + 3h), phase 1 finished np + 3h.
void build_resident_schedule(const ResidentShape& S, int64_t M, int64_t N, int64_t K, bool c0, int n_compute, std::vector<hclooc_op_t>& ops) {
    ops.clear();
    const int64_t h = S.h, np = S.npanels, p_sw = S.p_switch;
    auto blank = [](int kind, int stream) {
        hclooc_op_t o;
        std::memset(&o, 0, sizeof(o));
        o.kind = kind; o.stream = stream; o.event = -1; o.buf = o.buf2 = o.buf3 = -1;
        return o;
    };
    auto wait = [&](int stream, int64_t ev) { hclooc_op_t o = blank(HCLOOC_OP_WAIT, stream); o.event = (int32_t)ev; ops.push_back(o); };
    auto record = [&](int stream, int64_t ev) { hclooc_op_t o = blank(HCLOOC_OP_RECORD, stream); o.event = (int32_t)ev; ops.push_back(o); };
    auto upload_c0 = [&](int64_t r) {
        const int64_t r0 = r * S.mb, mr = std::min(S.mb, M - r0);
        if (r >= S.ring) wait(0, np + h + (r - S.ring));            // the slot's previous tenant has been added to its row block
        hclooc_op_t o = blank(HCLOOC_OP_H2D_C, 0);
        o.buf = 3 + (int32_t)(r % S.ring); o.r0 = r0; o.nr = mr; o.c0 = 0; o.nc = N; o.step = r;
        ops.push_back(o);
        record(0, np + r);
    };
    // ---- phase 1: panels up, whole-C kernels behind them
    for (int64_t p = 0; p < np; ++p) {
        hclooc_op_t a = blank(HCLOOC_OP_H2D_A, 0);
        a.buf = 0; a.r0 = 0; a.nr = M; a.c0 = S.pk0[p]; a.nc = S.pkk[p]; a.k0 = S.pk0[p]; a.kk = S.pkk[p]; a.step = p;
        ops.push_back(a);
        hclooc_op_t b = blank(HCLOOC_OP_H2D_B, 0);
        b.buf = 1; b.r0 = S.pk0[p]; b.nr = S.pkk[p]; b.c0 = 0; b.nc = N; b.k0 = S.pk0[p]; b.kk = S.pkk[p]; b.step = p;
        ops.push_back(b);
        record(0, p);
        if (p < p_sw) {
            wait(2, p);
            hclooc_op_t g = blank(HCLOOC_OP_GEMM, 2);
            g.buf = 0; g.buf2 = 1; g.buf3 = 2; g.r0 = 0; g.nr = M; g.c0 = 0; g.nc = N; g.k0 = S.pk0[p]; g.kk = S.pkk[p];
            g.beta = p == 0 ? 0.0 : 1.0; g.step = p;
            ops.push_back(g);
        }
    }
    // ---- phase 2: row blocks finished, joined with C0, downloaded
    if (c0) for (int64_t r = 0; r < std::min<int64_t>(h, S.ring); ++r) upload_c0(r);
    const int n_k2 = n_compute >= 2 ? 2 : 1;
    const int64_t k_sw = S.pk0[p_sw], k_rest = K - k_sw;
    record(2, np + 3 * h);
    for (int i = 0; i < n_k2; ++i) {
        wait(2 + i, np - 1);                                         // the upload stream is in order: every panel is there
        if (i > 0) wait(2 + i, np + 3 * h);                          // and phase 1 has finished on stream 2
    }
    for (int64_t r = 0; r < h; ++r) {
        const int64_t r0 = r * S.mb, mr = std::min(S.mb, M - r0);
        const int st = 2 + (int)(r % n_k2);
        hclooc_op_t g = blank(HCLOOC_OP_GEMM, st);
        g.buf = 0; g.buf2 = 1; g.buf3 = 2; g.r0 = r0; g.nr = mr; g.c0 = 0; g.nc = N; g.k0 = k_sw; g.kk = k_rest;
        g.beta = p_sw == 0 ? 0.0 : 1.0; g.step = np + r;
        ops.push_back(g);
        if (c0) {
            wait(st, np + r);
            hclooc_op_t x = blank(HCLOOC_OP_AXPY, st);
            x.buf = 3 + (int32_t)(r % S.ring); x.buf3 = 2; x.r0 = r0; x.nr = mr; x.c0 = 0; x.nc = N; x.beta = -1.0; x.step = np + h + r;
            ops.push_back(x);
            record(st, np + h + r);
        }
        record(st, np + 2 * h + r);
        wait(1, np + 2 * h + r);
        hclooc_op_t d = blank(HCLOOC_OP_D2H_C, 1);
        d.buf = 2; d.r0 = r0; d.nr = mr; d.c0 = 0; d.nc = N; d.step = r;
        ops.push_back(d);
        if (c0 && r + S.ring < h) upload_c0(r + S.ring);
    }
}

int dgemm_resident(hclooc_ctx* ctx, const ResidentShape& S, int64_t M, int64_t N, int64_t K, double alpha, const double* A, int64_t lda,
                   const double* B, int64_t ldb, double beta, double* C, int64_t ldc, hclooc_stats* stats,
                   std::chrono::steady_clock::time_point t_begin) {
    int rc;
    if ((rc = ensure_workspace(ctx, S.total))) return rc;
    uint8_t* base = (uint8_t*)ctx->workspace;
    const uintptr_t mis = (uintptr_t)base & 1023u;
    if (mis) base += 1024 - mis;
    if ((size_t)(base - (uint8_t*)ctx->workspace) + S.total - 4096 > ctx->workspace_bytes) return HCLOOC_ERR_BUDGET;   // 4 KiB of slack cover the shift
    double* dA = (double*)base;
    double* dB = (double*)(base + S.bytesA);
    double* dC = (double*)(base + S.bytesA + S.bytesB);
    uint8_t* scratch = base + S.bytesA + S.bytesB + S.bytesC;
    uint8_t* stage0 = scratch + S.bytes_scratch;
    const bool c0 = beta != 0.0;
    const int64_t h = S.h, np = S.npanels, p_sw = S.p_switch;
    const size_t n_events = (size_t)(np + 3 * h + 1);
    while (ctx->events.size() < n_events) {
        cudaEvent_t e;
        HCL_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        ctx->events.push_back(e);
    }
    // phase 2 alternates between two compute streams when the context has them: the launch of row block r + 1 fills the partly
    // empty last wave of row block r (what the slice pipeline's kernels do for each other)
    const int n_k2 = ctx->n_compute >= 2 ? 2 : 1;
    build_resident_schedule(S, M, N, K, c0, ctx->n_compute, ctx->ops);
    auto stream_of = [&](int s) { return s == 0 ? ctx->s_h2d : (s == 1 ? ctx->s_d2h : ctx->s_compute[s - 2]); };
    // tracing: timing events around every copy and kernel, as the pipeline's executor records them
    const bool trace = ctx->trace;
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
    uint64_t bytes_h2d = 0, bytes_d2h = 0, n_h2d = 0, n_d2h = 0, n_kernels = 0;
    const auto t_enq0 = std::chrono::steady_clock::now();
    if (ctx->dbg_poison) {           // nothing of a previous call may stand in for an upload that never came
        debug_poison(ctx, dA, S.ldA, M, S.ldA, ctx->s_h2d);
        debug_poison(ctx, dB, S.ldB, K, S.ldB, ctx->s_h2d);
        debug_poison(ctx, dC, S.ldC, M, S.ldC, ctx->s_h2d);
    }
    HCL_CUDA(cudaMemsetAsync(scratch + streamk_counter_offset(), 0, streamk_counter_bytes(), ctx->s_compute[0]));
    rc = HCLOOC_OK;
    for (const hclooc_op_t& o : ctx->ops) {
        cudaStream_t st = stream_of(o.stream);
        if (o.kind == HCLOOC_OP_WAIT) {
            // sabotage mode of the shaker: the staging ring's waits are dropped on both sides (slots refilled before their tenant
            // was used: event range [np + h, np + 2h) on the upload stream; blocks used before they arrived: [np, np + h))
            if (ctx->dbg_poison == 2 && o.event >= np && o.event < np + 2 * h) continue;
            HCL_CUDA(cudaStreamWaitEvent(st, ctx->events[(size_t)o.event], 0));
            continue;
        }
        if (o.kind == HCLOOC_OP_RECORD) {
            HCL_CUDA(cudaEventRecord(ctx->events[(size_t)o.event], st));
            continue;
        }
        debug_jitter(ctx, st);
        double* stage = o.buf >= 3 ? (double*)(stage0 + (size_t)(o.buf - 3) * S.bytes_stage) : nullptr;
        if (o.kind == HCLOOC_OP_H2D_C && ctx->dbg_poison) debug_poison(ctx, stage, S.ldC, o.nr, N, st);
        if (trace) {
            cudaEventRecord(ctx->trace_events[1 + 2 * n_traced], st);
            hclooc_trace_rec r;
            std::memset(&r, 0, sizeof(r));
            r.kind = o.kind == HCLOOC_OP_AXPY ? HCLOOC_OP_GEMM : o.kind; r.stream = o.stream; r.step = o.step;
            if (o.kind == HCLOOC_OP_GEMM) r.flops = 2.0 * (double)o.nr * (double)o.nc * (double)o.kk;
            else if (o.kind == HCLOOC_OP_AXPY) r.flops = 2.0 * (double)o.nr * (double)o.nc;
            else r.bytes = (uint64_t)o.nr * (uint64_t)o.nc * 8;
            ctx->trace_recs.push_back(r);
        }
        switch (o.kind) {
            case HCLOOC_OP_H2D_A:
                rc = copy2d(dA + o.k0, (size_t)S.ldA * 8, A + o.k0, (size_t)lda * 8, (size_t)o.kk * 8, (size_t)M, st);
                bytes_h2d += (uint64_t)M * o.kk * 8; ++n_h2d;
                break;
            case HCLOOC_OP_H2D_B:
                rc = copy2d(dB + o.k0 * S.ldB, (size_t)S.ldB * 8, B + o.k0 * ldb, (size_t)ldb * 8, (size_t)N * 8, (size_t)o.kk, st);
                bytes_h2d += (uint64_t)o.kk * N * 8; ++n_h2d;
                break;
            case HCLOOC_OP_H2D_C:
                rc = copy2d(stage, (size_t)S.ldC * 8, C + o.r0 * ldc, (size_t)ldc * 8, (size_t)N * 8, (size_t)o.nr, st);
                bytes_h2d += (uint64_t)o.nr * N * 8; ++n_h2d;
                break;
            case HCLOOC_OP_D2H_C:
                rc = copy2d(C + o.r0 * ldc, (size_t)ldc * 8, dC + o.r0 * S.ldC, (size_t)S.ldC * 8, (size_t)N * 8, (size_t)o.nr, st);
                bytes_d2h += (uint64_t)o.nr * N * 8; ++n_d2h;
                break;
            case HCLOOC_OP_GEMM: {
                // a launch that runs alone fills whole waves of 148 tiles well enough by itself or goes out as the persistent
                // stream-K kernel; the phase-2 launches on two streams fill each other's last wave
                const bool alone = o.step < np || n_k2 == 1;
                const int64_t T = ((o.nr + 127) / 128) * ((N + 127) / 128), waves = (T + 147) / 148;
                const bool whole = !alone || (double)T >= 0.988 * (double)(waves * 148);
                rc = launch_dgemm_tiles(o.nr, N, o.kk, alpha, dA + o.r0 * S.ldA + o.k0, S.ldA, dB + o.k0 * S.ldB, S.ldB, o.beta,
                                        dC + o.r0 * S.ldC, S.ldC, st, whole ? 1 : -1, whole ? nullptr : scratch);
                ++n_kernels;
                break;
            }
            case HCLOOC_OP_AXPY: {
                const int cols2 = (int)((N + 1) / 2);
                dim3 grid((unsigned)std::min<int64_t>((cols2 + 255) / 256, 32), (unsigned)std::min<int64_t>(o.nr, 1024));
                resident_axpy_kernel<<<grid, 256, 0, st>>>(dC + o.r0 * S.ldC, (long long)S.ldC, stage, (long long)S.ldC, (int)o.nr, cols2, beta);
                cudaError_t e = cudaGetLastError();
                if (e != cudaSuccess) rc = cuda_fail(e);
                ++n_kernels;
                break;
            }
            default: rc = HCLOOC_ERR_INTERNAL;
        }
        if (trace) { cudaEventRecord(ctx->trace_events[2 + 2 * n_traced], st); ++n_traced; }
        if (rc) break;
    }
    const auto t_enq1 = std::chrono::steady_clock::now();
    cudaError_t e1 = cudaStreamSynchronize(ctx->s_d2h), e2 = cudaStreamSynchronize(ctx->s_h2d), e3 = cudaStreamSynchronize(ctx->s_compute[0]);
    if (e3 == cudaSuccess && n_k2 == 2) e3 = cudaStreamSynchronize(ctx->s_compute[1]);
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
    } else {
        ctx->trace_recs.clear();
    }
    if (stats) {
        hclooc_plan_t& P = stats->plan;
        std::memset(&P, 0, sizeof(P));
        P.M = M; P.N = N; P.K = K;
        P.mb = S.mb; P.nb = N; P.kb = S.kb; P.h = h; P.w = 1; P.kpanels = np;
        P.n_steps = p_sw + h;
        P.n_sets = S.ring; P.n_bbuf = 1; P.n_abuf = 1; P.beta_nonzero = c0 ? 1 : 0; P.ksplit = 1;
        P.lda_dev = S.ldA; P.ldb_dev = S.ldB; P.ldc_dev = S.ldC;
        P.bytes_a_buf = S.bytesA; P.bytes_b_buf = S.bytesB; P.bytes_c_buf = S.bytes_stage;
        P.workspace_bytes = S.total;
        P.bytes_h2d = bytes_h2d; P.bytes_d2h = bytes_d2h; P.n_copies_h2d = n_h2d; P.n_copies_d2h = n_d2h;
        P.flops = 2.0 * (double)M * (double)N * (double)K;
        P.t_flop_s = S.t_flop_s; P.t_link_s = S.t_link_s; P.t_model_s = S.t_model_s;
        P.n_scratch = 1; P.bytes_scratch = S.bytes_scratch;
        P.resident = (int32_t)(1 + p_sw);
        stats->bytes_h2d = bytes_h2d; stats->bytes_d2h = bytes_d2h;
        stats->n_kernels = n_kernels; stats->n_copies_h2d = n_h2d; stats->n_copies_d2h = n_d2h;
        stats->t_enqueue_s = std::chrono::duration<double>(t_enq1 - t_enq0).count();
        stats->t_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
    }
    return HCLOOC_OK;
}

}  // namespace hclooc

extern "C" int hclooc_plan_resident(int64_t M, int64_t N, int64_t K, int beta_nonzero, size_t device_budget_bytes, double t_slice_model_s,
                                    hclooc_resident_plan_t* out) {
    if (M < 1) return -1;
    if (N < 1) return -2;
    if (K < 1) return -3;
    if (!out) return -7;
    std::memset(out, 0, sizeof(*out));
    hclooc::ResidentShape S;
    std::memset(&S, 0, sizeof(S));
    S.total = 0;
    out->applies = hclooc::resident_applies(M, N, K, beta_nonzero != 0, device_budget_bytes, t_slice_model_s, &S) ? 1 : 0;
    if (S.total == 0) return HCLOOC_OK;                 // it does not fit at all: nothing to describe
    out->ring = S.ring;
    out->mb = S.mb; out->h = S.h; out->kb = S.kb; out->npanels = S.npanels; out->p_switch = S.p_switch;
    out->lda_dev = S.ldA; out->ldb_dev = S.ldB; out->ldc_dev = S.ldC;
    out->workspace_bytes = S.total;
    out->t_flop_s = S.t_flop_s; out->t_link_s = S.t_link_s; out->t_model_s = S.t_model_s;
    for (int64_t p = 0; p < S.npanels; ++p) { out->panel_k0[p] = S.pk0[p]; out->panel_kk[p] = S.pkk[p]; }
    return HCLOOC_OK;
}

extern "C" int hclooc_resident_schedule(const hclooc_resident_plan_t* plan, int64_t M, int64_t N, int64_t K, int beta_nonzero, int n_compute,
                                        hclooc_op_t* ops, size_t max_ops, size_t* n_ops) {
    if (!plan) return -1;
    if (M < 1) return -2;
    if (N < 1) return -3;
    if (K < 1) return -4;
    if (n_compute < 1) return -6;
    if (!n_ops) return -9;
    if (plan->npanels < 1 || plan->npanels > HCLOOC_RESIDENT_MAX_PANELS || plan->mb < 1 || plan->h != (M + plan->mb - 1) / plan->mb ||
        plan->p_switch < 0 || plan->p_switch >= plan->npanels || (beta_nonzero && plan->ring < 1)) return -1;
    hclooc::ResidentShape S;
    std::memset(&S, 0, sizeof(S));
    S.mb = plan->mb; S.h = plan->h; S.kb = plan->kb; S.npanels = plan->npanels; S.p_switch = plan->p_switch; S.ring = plan->ring;
    for (int64_t p = 0; p < plan->npanels; ++p) { S.pk0[p] = plan->panel_k0[p]; S.pkk[p] = plan->panel_kk[p]; }
    std::vector<hclooc_op_t> v;
    hclooc::build_resident_schedule(S, M, N, K, beta_nonzero != 0, n_compute, v);
    *n_ops = v.size();
    if (ops) std::memcpy(ops, v.data(), std::min(max_ops, v.size()) * sizeof(hclooc_op_t));
    return HCLOOC_OK;
}

