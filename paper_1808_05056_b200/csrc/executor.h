// executor.h -- the context and the entry points of executor.cu that the other out-of-core routines (factor.cu) build on.
#pragma once
#include <chrono>
#include <mutex>
#include <utility>
#include <vector>
#include "internal.h"

constexpr int MAX_COMPUTE_STREAMS = 16;

struct hclooc_ctx {
    int device = 0;
    void* workspace = nullptr;
    size_t workspace_bytes = 0;
    bool owns_workspace = false;
    cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
    bool owns_h2d = false, owns_d2h = false;
    cudaStream_t s_compute[MAX_COMPUTE_STREAMS] = {};
    int n_compute = 0;
    bool owns_compute = false;
    std::vector<cudaEvent_t> events;
    std::vector<hclooc_op_t> ops;
    bool trace = false;
    int direct_mode = -1;                         // -1 cost model decides, 0 never, 1 whenever the operands allow it
    // plans of recent calls: the search over candidates costs 0.2 ms (config 1) to 9 ms (config 4) of host time
    // before the first copy can be issued, and a blocked algorithm repeats the same shapes over and over
    struct PlanKey { int64_t M, N, K; int beta_nz, alpha_zero, where; size_t budget; };
    std::vector<std::pair<PlanKey, hclooc_plan_t>> plan_cache;
    std::vector<cudaEvent_t> trace_events;        // 2 per traced op (+1 base), timing enabled
    std::vector<hclooc_trace_rec> trace_recs;     // filled after the final synchronisation
    // the schedule of the last call captured as a CUDA graph (short, latency-bound schedules; same call again
    // -> one graph launch instead of hundreds of enqueues)
    cudaGraphExec_t graph_exec = nullptr;
    bool graph_valid = false;                     // graph_exec is the schedule of graph_key
    std::vector<int64_t> graph_key;               // the previous call
    std::vector<cudaEvent_t> join_events;
    // nsteps mode (hclooc_dgemm_nsteps): C kept in device memory between the calls of one sequence
    double* res_c = nullptr;
    int64_t res_ld = 0, res_M = 0, res_N = 0, res_ldc = 0;
    const double* res_host = nullptr;
    size_t res_bytes = 0;
    // bytes at the front of the workspace that a routine running several DGEMM calls keeps for itself (a resident panel of
    // hclooc_dpotrf / hclooc_dtrsm_side): dgemm_core_locked carves its buffers behind them and plans with the rest of the budget
    size_t reserved_bytes = 0;
    // streams, events and a pinned status word of the routines with a look-ahead (factor.cu): their own device work runs beside
    // the DGEMM pipeline, so it must not sit on the pipeline's streams (dgemm_core synchronises those); created on first use
    cudaStream_t s_aux[4] = {};
    cudaEvent_t ev_aux[8] = {};
    long long* h_word = nullptr;
    // debug shaker (hclooc_ctx_set_debug / HCLOOC_DEBUG_JITTER): random spin kernels in front of copies and kernels, NaN in every
    // device buffer region the moment the schedule declares it free to overwrite
    uint64_t dbg_rng = 0;                         // 0 = off, else the xorshift state
    int dbg_poison = 0;
    std::mutex mu;
};

namespace hclooc {

int default_ctx(hclooc_ctx** out);
// 0 = ok, HCLOOC_ERR_NOT_PINNED if pageable host memory; *on_device is cleared unless p is device memory;
// *dev_alias (nullable) = the address under which kernels on the device reach p (NULL if they cannot)
int check_resident(const void* p, bool* on_device, const void** dev_alias = nullptr);
bool overlaps(const double* a, int64_t rows_a, int64_t cols_a, int64_t lda, const double* b, int64_t rows_b, int64_t cols_b, int64_t ldb);
int copy2d(void* dst, size_t dpitch, const void* src, size_t spitch, size_t width, size_t rows, cudaStream_t s);
// the budget a call works under: the caller's figure, clipped to a caller-owned workspace, or all free device memory less 1 GiB
int resolve_budget(hclooc_ctx* ctx, size_t device_budget_bytes, size_t* budget, bool* library_owned);
int ensure_workspace(hclooc_ctx* ctx, size_t bytes);
int ensure_aux(hclooc_ctx* ctx);        // ctx->s_aux, ev_aux, h_word
// debug shaker (runtime.cu): a spin kernel of random length in `s` (with probability 1/2) when ctx->dbg_rng != 0 ...
void debug_jitter(hclooc_ctx* ctx, cudaStream_t s);
// ... and NaN over a rows x cols region (leading dimension ld) in `s` when ctx->dbg_poison != 0: called where a buffer is about
// to be overwritten -- after the schedule's waits -- so that a reader the waits failed to cover sees NaN instead of stale data
void debug_poison(hclooc_ctx* ctx, double* p, int64_t ld, int64_t rows, int64_t cols, cudaStream_t s);

// C = alpha*op(A)*op(B) + beta*C through the pipeline (executor.cu).  tri != 0: only the lower (1) / upper (2) triangle of this
// call's C -- element (0, 0) on the diagonal -- is referenced (hclooc_dsyrk, the Cholesky panel).  Takes ctx->mu itself.
int dgemm_core(hclooc_ctx* ctx, int transa, int transb, int64_t M, int64_t N, int64_t K, double alpha, const double* A,
               int64_t lda, const double* B, int64_t ldb, double beta, double* C, int64_t ldc,
               size_t device_budget_bytes, hclooc_stats* stats, int tri = 0);
// Extras of a DGEMM call made by a routine that keeps a panel in device memory: the initial C is read from C_src (a host
// matrix, leading dimension ldc_src) while the result goes to C (device memory) -- the pipeline itself brings the panel up,
// block by block under its kernels; and the FIRST write into C waits for these events (the previous tenant of the buffer).
struct DgemmExtra {
    const double* C_src = nullptr;
    int64_t ldc_src = 0;
    cudaEvent_t wait_before_store[2] = {nullptr, nullptr};
    // a triangular operand (hclooc_dtrmm, hclooc_dsymm): op(A)[r][k] counts iff k <= r + adiag (amask = 1) / k >= r + adiag (2);
    // op(B)[k][c] counts iff c <= k + bdiag (bmask = 1) / c >= k + bdiag (2); what lies outside is never read into a product
    int amask = 0, adiag = 0, bmask = 0, bdiag = 0;
    // C may overlap an operand (hclooc_dtrmm works in place): legal only with one K panel -- every step then reads device
    // copies made before the first block of its column is stored -- so a plan with K panels is refused (HCLOOC_ERR_BUDGET)
    bool in_place = false;
};
// the same with ctx->mu already held by the caller (ctx not NULL)
int dgemm_core_locked(hclooc_ctx* ctx, int transa, int transb, int64_t M, int64_t N, int64_t K, double alpha, const double* A,
                      int64_t lda, const double* B, int64_t ldb, double beta, double* C, int64_t ldc,
                      size_t device_budget_bytes, hclooc_stats* stats, int tri = 0, const DgemmExtra* extra = nullptr);

// The resident schedule of hclooc_dgemm (resident.cu): A, B and C fit the budget, K is streamed in panels, C finished row block
// by row block.  resident_applies says whether the call takes it (shape, memory, cost model against the slice plan's t_model_s;
// HCLOOC_RESIDENT=0 / 1 forces the answer) and fills the shape; dgemm_resident runs it (ctx->mu held by the caller).
constexpr int RESIDENT_MAX_PANELS = 128;
struct ResidentShape {
    int64_t mb, h, kb, npanels, p_switch;          // row blocks of mb rows, K panels of at most kb, phase 2 starts with panel p_switch
    int64_t pk0[RESIDENT_MAX_PANELS], pkk[RESIDENT_MAX_PANELS];   // panel p = columns [pk0, pk0 + pkk) of A, the same rows of B
    int64_t ldA, ldB, ldC;                         // leading dimensions of the device copies
    size_t bytesA, bytesB, bytesC, bytes_stage, bytes_scratch, total;
    int ring;                                      // staging buffers for the initial C (0 when beta == 0)
    double t_flop_s, t_link_s, t_model_s;
};
bool resident_applies(int64_t M, int64_t N, int64_t K, bool beta_nonzero, size_t budget, double t_slice_model_s, ResidentShape* out);
int dgemm_resident(hclooc_ctx* ctx, const ResidentShape& S, int64_t M, int64_t N, int64_t K, double alpha, const double* A, int64_t lda,
                   const double* B, int64_t ldb, double beta, double* C, int64_t ldc, hclooc_stats* stats,
                   std::chrono::steady_clock::time_point t_begin);

// hclooc_dtrsm (side = Left) with two resident block rows and a look-ahead of one (factor.cu); ctx->mu held by the caller
int dtrsm_left_lookahead(hclooc_ctx* ctx, int uplo, int trans, int diag, int64_t M, int64_t N, double alpha, const double* A, int64_t lda,
                         double* B, int64_t ldb, size_t budget, bool own, int64_t NB, hclooc_stats* stats);

// X <- op(T)^-1 (scale X) (right = 0: X is n x w) / X <- (scale X) op(T)^-1 (right = 1: X is w x n) in device memory by recursive
// halving (factor.cu dev_trsm); lower: op(T) is lower triangular; trans: op(T)[r][c] is stored at T[c][r]
int dev_trsm_ctx(hclooc_ctx* dbg, int right, const double* dT, int64_t ldt, int lower, int trans, int unit, double* X, int64_t ld, int64_t w,
                 int64_t n, double scale, cudaStream_t st, uint64_t* n_kernels);

// the block kernels of the LU factorization (getrf_sm100.cu)
size_t getrf_slot_bytes(int gcap);            // scratch of the panel kernel for launches of at most gcap CTAs; its first 8 bytes: the barrier counter
int getrf_panel_shape(long long m, int* G_out, int* rpc_out);
int launch_getrf_panel(double* dA, int64_t lda, int64_t m, int w, long long* ipiv_out, long long row_base, long long* d_info,
                       long long info_base, void* slots, int gcap, unsigned long long* bar_base, cudaStream_t stream);
int launch_row_permute(double* X, int64_t ld, int64_t ncols, int nt, const int* src, const int* dst, double* tmp, size_t tmp_elems,
                       cudaStream_t stream, uint64_t* n_kernels);
int launch_row_gather_all(const double* X, int64_t ldx, int64_t ncols, int64_t nrows, const int* perm, double* Y, int64_t ldy, cudaStream_t stream);

}  // namespace hclooc
