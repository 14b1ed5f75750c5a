// fig2_pipeline.cu -- the paper's own MMOOC pipeline (Figure 2; description :285-313),
// written against the exported hcl* runtime calls only, as the paper writes it against hclRuntime.
//
// kept beside the tuned scheduler (executor.cu) so the two can be timed against each other
// on the same machine -- the shape of the paper's own experiment (abstraction vs hand-tuned, :372, :394).
//
// What is reproduced, in the paper's notation:
//   * hclMatrixPartitioner: A in h equal horizontal slices, B in w equal vertical slices, C in h x w blocks,
//     one B slice + two A slices + two C blocks resident (:289, example :301);
//   * w*h steps in column-major order idx = i + j*h, one c_ij per step (:189-192, :293);
//   * TWO streams used round-robin: s[idx%2] waits for its inputs, runs DGEMM and sends c_ij back, while
//     s[(idx+1)%2] prefetches a_i and c_ij of step idx+1 into the opposite-parity buffers (:287, :313);
//   * FIVE event families: rA[idx], rB[j], rC[idx] "received", eA[idx] "DGEMM done", eC[idx] "c_ij stored"
//     (:187-188, :291); a buffer is overwritten only after the kernel/transfer that used it (:311);
//   * a SINGLE B buffer, reloaded at i == h-1 after eA[idx] -- not overlapped with computation (:236-242);
//   * the in-core switch: if A, B and C fit the device memory together, one upload, one DGEMM, one download
//     (:130 hclGetMemSize, :368 "switches to out-of-core when N > 22528").
// Where the listing is garbled (the `nsteps` conditions, :245, :259-263; G17/G18 in DESIGN.md) every call
// uploads C when beta != 0 and downloads every block.  Ragged sizes are not treated by the paper ("equal
// slices"), and not here: h divides M and w divides N by construction of hclMatrixPartitioner.
#include <chrono>
#include <vector>
#include "../../include/hclooc.h"

namespace {

struct Fig2Events {
    std::vector<hclEvent> eA, rA, rB, eC, rC;
    void resize(size_t steps, size_t w) {
        eA.assign(steps, nullptr); rA.assign(steps, nullptr); eC.assign(steps, nullptr); rC.assign(steps, nullptr);
        rB.assign(w, nullptr);
    }
    void destroy() {
        for (auto* v : {&eA, &rA, &rB, &eC, &rC})
            for (hclEvent e : *v)
                if (e) hclEventDestroy(e);
    }
};

int64_t even_up(int64_t x) { return (x + 1) & ~(int64_t)1; }

}  // namespace

#define F2(call) do { int rc__ = (call); if (rc__ != HCLOOC_OK) { status = rc__; goto done; } } while (0)

extern "C" int hclooc_dgemm_fig2(int64_t M, int64_t N, int64_t K, double alpha, const double* A, int64_t lda,
                                 const double* B, int64_t ldb, double beta, double* C, int64_t ldc,
                                 size_t device_budget_bytes, hclooc_stats* stats) {
    if (M <= 0) return -1;
    if (N <= 0) return -2;
    if (K <= 0) return -3;
    if (!A) return -5;
    if (lda < K) return -6;
    if (!B) return -7;
    if (ldb < N) return -8;
    if (!C) return -10;
    if (ldc < N) return -11;
    if (stats) *stats = hclooc_stats{};
    int status = HCLOOC_OK;
    size_t budget = device_budget_bytes;
    if (budget == 0) {
        size_t fr = 0;
        int rc = hclGetMemSize(0, &fr);                                   // :130
        if (rc) return rc;
        budget = fr > ((size_t)2 << 30) ? fr - ((size_t)1 << 30) : fr / 2;
    }
    // ---- in-core or out-of-core (:130, :368), then hclMatrixPartitioner (:186)
    int64_t h = 1, w = 1;
    const long double all = (long double)M * K + (long double)K * N + (long double)M * N;
    const bool in_core = all * 8 <= (long double)budget;
    if (!in_core) {
        int rc = hclMatrixPartitioner(M, N, K, (int64_t)(budget / 8), &h, &w);
        if (rc) return rc;
    }
    const int64_t mb = M / h, nb = N / w, steps = h * w;
    const bool cload = (beta != 0.0);
    const int n_par = in_core ? 1 : 2;
    // device buffers: leading dimensions even so that every row start is 16-byte aligned (hclDgemmAsync)
    const int64_t ldA = even_up(K), ldB = even_up(nb), ldC = even_up(nb);
    const size_t bytes_a = (size_t)mb * ldA * 8, bytes_b = (size_t)K * ldB * 8, bytes_c = (size_t)mb * ldC * 8;
    if (bytes_b + n_par * (bytes_a + bytes_c) > budget) return HCLOOC_ERR_BUDGET;     // padding of odd widths did not fit
    double *dA[2] = {nullptr, nullptr}, *dC[2] = {nullptr, nullptr}, *dB = nullptr;
    hclStream s[2] = {nullptr, nullptr};
    Fig2Events ev;
    uint64_t bytes_h2d = 0, bytes_d2h = 0, n_h2d = 0, n_d2h = 0, n_kernels = 0;
    std::chrono::steady_clock::time_point t_enq0, t_enq1;
    ev.resize((size_t)steps, (size_t)w);
    F2(hclMalloc((void**)&dB, bytes_b));
    for (int p = 0; p < n_par; ++p) { F2(hclMalloc((void**)&dA[p], bytes_a)); F2(hclMalloc((void**)&dC[p], bytes_c)); }
    F2(hclStreamCreate(&s[0]));
    F2(hclStreamCreate(&s[1]));
    t_enq0 = std::chrono::steady_clock::now();
    {
        auto send_b = [&](int64_t j, hclStream st) {                       // S(b_j), :305
            bytes_h2d += (uint64_t)K * nb * 8; ++n_h2d;
            return hclMemcpy2DAsync(dB, (size_t)ldB * 8, B + j * nb, (size_t)ldb * 8, (size_t)nb * 8, (size_t)K, HCL_H2D, st, &ev.rB[j]);
        };
        auto send_a = [&](int64_t i, int par, int64_t idx, hclStream st) { // S(a_i), :306
            bytes_h2d += (uint64_t)mb * K * 8; ++n_h2d;
            return hclMemcpy2DAsync(dA[par], (size_t)ldA * 8, A + i * mb * lda, (size_t)lda * 8, (size_t)K * 8, (size_t)mb, HCL_H2D, st, &ev.rA[idx]);
        };
        auto send_c = [&](int64_t i, int64_t j, int par, int64_t idx, hclStream st) {   // S(c_ij), :307
            bytes_h2d += (uint64_t)mb * nb * 8; ++n_h2d;
            return hclMemcpy2DAsync(dC[par], (size_t)ldC * 8, C + i * mb * ldc + j * nb, (size_t)ldc * 8, (size_t)nb * 8, (size_t)mb, HCL_H2D, st, &ev.rC[idx]);
        };
        for (int64_t j = 0; j < w; ++j) {
            for (int64_t i = 0; i < h; ++i) {
                const int64_t idx = i + j * h;                             // :191
                const int cur = (int)(idx % n_par), nxt = (int)((idx + 1) % n_par);
                if (idx == 0) {                                            // lines 12-16 of the listing
                    F2(send_b(0, s[cur]));
                    F2(send_a(0, cur, 0, s[cur]));
                    if (cload) F2(send_c(0, 0, cur, 0, s[cur]));
                }
                // stream idx%2: Wait(rB[j]), Wait(rA[idx]), Wait(rC[idx]); DGEMM -> eA[idx]   (lines 18-22)
                F2(hclWaitEvent(s[cur], ev.rB[j]));
                F2(hclWaitEvent(s[cur], ev.rA[idx]));
                if (cload) F2(hclWaitEvent(s[cur], ev.rC[idx]));
                F2(hclDgemmAsync(mb, nb, K, alpha, dA[cur], ldA, dB, ldB, beta, dC[cur], ldC, s[cur], &ev.eA[idx]));   // :308
                ++n_kernels;
                if (idx < steps - 1) {
                    // the other stream prefetches step idx+1 into the opposite-parity buffers (lines 23-34)
                    const int64_t i1 = (idx + 1) % h, j1 = (idx + 1) / h;
                    if (idx > 0) F2(hclWaitEvent(s[nxt], ev.eA[idx - 1]));                 // a-buffer free (:311)
                    F2(send_a(i1, nxt, idx + 1, s[nxt]));
                    if (idx > 0) F2(hclWaitEvent(s[nxt], ev.eC[idx - 1]));                 // c-buffer drained
                    if (cload) F2(send_c(i1, j1, nxt, idx + 1, s[nxt]));
                    if (i == h - 1) {                                                      // lines 35-39: B reload, not overlapped
                        F2(hclWaitEvent(s[nxt], ev.eA[idx]));
                        if (idx > 0) F2(hclWaitEvent(s[nxt], ev.eA[idx - 1]));
                        F2(send_b(j1, s[nxt]));
                    }
                }
                // R(c_ij) on the step's own stream -> eC[idx]   (line 41, :309)
                bytes_d2h += (uint64_t)mb * nb * 8; ++n_d2h;
                F2(hclMemcpy2DAsync(C + i * mb * ldc + j * nb, (size_t)ldc * 8, dC[cur], (size_t)ldC * 8, (size_t)nb * 8, (size_t)mb, HCL_D2H, s[cur], &ev.eC[idx]));
            }
        }
    }
    t_enq1 = std::chrono::steady_clock::now();
    F2(hclStreamSynchronize(s[0]));                                        // :268-269
    F2(hclStreamSynchronize(s[1]));
    if (stats) {
        // t_total_s: first enqueue to both streams drained -- like hclooc_dgemm_ex with a ready context, device
        // allocation and release are outside (G16)
        stats->t_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_enq0).count();
        stats->plan.M = M; stats->plan.N = N; stats->plan.K = K;
        stats->plan.mb = mb; stats->plan.nb = nb; stats->plan.kb = K;
        stats->plan.h = h; stats->plan.w = w; stats->plan.kpanels = 1; stats->plan.n_steps = steps;
        stats->plan.n_sets = n_par; stats->plan.n_abuf = n_par; stats->plan.n_bbuf = 1; stats->plan.ksplit = 0;
        stats->plan.beta_nonzero = cload ? 1 : 0;
        stats->plan.lda_dev = ldA; stats->plan.ldb_dev = ldB; stats->plan.ldc_dev = ldC;
        stats->plan.bytes_a_buf = bytes_a; stats->plan.bytes_b_buf = bytes_b; stats->plan.bytes_c_buf = bytes_c;
        stats->plan.workspace_bytes = bytes_b + n_par * (bytes_a + bytes_c);
        stats->plan.bytes_h2d = bytes_h2d; stats->plan.bytes_d2h = bytes_d2h;
        stats->plan.n_copies_h2d = n_h2d; stats->plan.n_copies_d2h = n_d2h;
        stats->plan.flops = 2.0 * (double)M * (double)N * (double)K;
        stats->bytes_h2d = bytes_h2d; stats->bytes_d2h = bytes_d2h;
        stats->n_kernels = n_kernels; stats->n_copies_h2d = n_h2d; stats->n_copies_d2h = n_d2h;
        stats->t_enqueue_s = std::chrono::duration<double>(t_enq1 - t_enq0).count();
    }
done:
    if (s[0]) { hclStreamSynchronize(s[0]); }
    if (s[1]) { hclStreamSynchronize(s[1]); }
    ev.destroy();
    if (s[0]) hclStreamDestroy(s[0]);
    if (s[1]) hclStreamDestroy(s[1]);
    for (int p = 0; p < 2; ++p) { if (dA[p]) hclFree(dA[p]); if (dC[p]) hclFree(dC[p]); }
    if (dB) hclFree(dB);
    return status;
}
