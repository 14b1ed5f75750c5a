// internal.h -- declarations shared by the translation units of libhclooc_b200 (not installed).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/hclooc.h"

struct CUtensorMap_st;   // <cuda.h>

namespace hclooc {

// last CUDA error seen on this thread (hclooc_last_cuda_error)
void set_last_cuda_error(int e);
inline int cuda_fail(cudaError_t e) { set_last_cuda_error((int)e); return HCLOOC_ERR_CUDA; }

#define HCL_CUDA(call)                                        \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) return ::hclooc::cuda_fail(e__); \
    } while (0)

// Link and FP64 figures the planner's cost model uses (measured on the B200 box, see DESIGN.md
// "Measured peaks"); overridable through HCLOOC_* environment variables for experiments.
struct MachineModel {
    double fp64_flops;      // sustained DMMA rate, flop/s
    double h2d_Bps;         // host -> device alone
    double d2h_Bps;         // device -> host alone
    double duplex_Bps;      // sum of both directions when both are busy
    double copy_latency_s;  // fixed cost per enqueued copy
    double launch_latency_s;
};
const MachineModel& machine_model();
void set_machine_link(double h2d_Bps, double d2h_Bps, double duplex_Bps);   // hclooc_calibrate_link

// Launch the tile kernel: dC = alpha*dA*dB + beta*dC on device pointers (row-major).
// Preconditions (checked by callers): pointers 16-byte aligned, leading dimensions even.
int launch_dgemm_tiles(int64_t M, int64_t N, int64_t K, double alpha, const double* dA, int64_t lda,
                       const double* dB, int64_t ldb, double beta, double* dC, int64_t ldc,
                       cudaStream_t stream, int ksplit,    // ksplit: 1, 2, 4; 0 = choose from the tile count;
                       void* streamk_scratch = nullptr,    // -1 = the launch has the GPU to itself: persistent stream-K
                                                           //      (scratch: streamk_scratch_bytes(), or NULL = library pool)
                       int transa = 0, int transb = 0,     // dA is stored K x M / dB is stored N x K (hclooc_dgemm_t)
                       int tri = 0, int doff = 0,          // hclooc_dsyrk: store only col <= row + doff (1) / col >= row + doff (2)
                       int opmask = 0, int adoff = 0, int bdoff = 0);   // hclooc_dtrmm / dsymm: op(A) / op(B) is a triangle of the stored
                                                           // operand: opmask = am | bm << 2; am = 1: op(A)[r][k] counts iff k <= r + adoff,
                                                           // 2: iff k >= r + adoff; bm = 1: op(B)[k][c] counts iff c <= k + bdoff, 2: iff >=

// The persistent stream-K kernel (dgemm_streamk_sm100.cu).  Returns 1 if it does not apply (no scratch buffer
// free, shape out of range): the caller then launches one CTA per tile.
int launch_dgemm_streamk(int64_t M, int64_t N, int64_t K, double alpha, const ::CUtensorMap_st& tmA, const ::CUtensorMap_st& tmB,
                         double beta, double* dC, int64_t ldc, cudaStream_t stream, void* scratch, int transa = 0, int transb = 0);
size_t streamk_scratch_bytes();     // one scratch buffer (partial-tile slots + counters), rounded to 1 KiB
size_t streamk_counter_offset();    // the counters inside it must be zero before the first launch
size_t streamk_counter_bytes();
// Work split of a stream-K launch: G persistent CTAs, dp_waves whole-tile waves, tail_tiles tiles cut along K.
bool streamk_layout(int64_t M, int64_t N, int64_t K, int num_sms, int* G, int* dp_waves, int* tail_tiles);

// K split (cluster size) worth using when `tiles_in_flight` tiles can run concurrently
int dgemm_auto_ksplit(int64_t tiles_in_flight, int64_t K);

// Where the chunks of a prefetched B slice sit inside the previous column of steps (two B buffers): the
// first chunk goes out with the i0-th step of that column -- late enough that the kernels of the column
// before it, the last readers of the target buffer, have normally drained -- and one chunk follows per step.
// Shared by the planner (copy counts) and the executor (the schedule) so the two cannot disagree.
inline void prefetch_layout(int64_t h, int64_t kk, int n_sets, int64_t* i0, int64_t* nchunks) {
    const int64_t first = h > 1 ? (h - 1 < (int64_t)n_sets ? h - 1 : (int64_t)n_sets) : 0;
    int64_t n = h - first;
    if (n > kk) n = kk;
    if (n < 1) n = 1;
    *i0 = first;
    *nchunks = n;
}

// With a single B buffer, the uploads of this many steps of the next column are issued BEFORE the B reload
// (they keep the link busy while the previous column's kernels drain); the rest of the C buffers stay free so
// that uploads can continue right after the reload while those first kernels run.
inline int64_t early_uploads(int64_t h, int n_sets, int n_abuf) {
    int64_t pre = n_sets - 4;
    if (pre > n_abuf - 1) pre = n_abuf - 1;
    if (pre > h) pre = h;
    return pre < 0 ? 0 : pre;
}

// 2-D FP64 tensor map (box_rows x 16 columns, 128-byte swizzle, zero fill out of bounds) over a row-major matrix
int make_tensor_map(::CUtensorMap_st* map, const double* base, int64_t rows, int64_t cols, int64_t ld, int box_rows);

// Direct mode with thread-block clusters sharing their loads by TMA multicast (dgemm_direct_sm100.cu)
void direct_cluster_shape(int64_t M, int64_t N, int max_cluster, int* cm, int* cn);   // pure arithmetic
void set_planner_max_cluster(int n);                                                 // the planner's copy of direct_max_cluster()
int direct_max_cluster();                                                            // 16 if a 4 x 4 cluster can launch here, else 8
int launch_dgemm_direct(int64_t M, int64_t N, int64_t K, double alpha, const double* A, int64_t lda, const double* B, int64_t ldb,
                        double beta, double* C, int64_t ldc, cudaStream_t stream, int cm, int cn);

// hclooc_plan_ex with the operand layouts of hclooc_dgemm_t (planner.cpp)
int plan_impl(int64_t M, int64_t N, int64_t K, int beta_nonzero, int alpha_zero, size_t device_budget_bytes,
              int operands_on_device, int transa, int transb, hclooc_plan_t* out);

// Diagonal-block solve of hclooc_dtrsm (trsm_sm100.cu): dX (ib x ncols, ib <= 128) <- op(T)^-1 * (scale * dX) in place
// right != 0: dX is ncols x ib and dX <- (scale * dX) * op(T)^-1 (one thread per row)
int launch_trsm_block(const double* dT, int64_t ldt, int ib, double* dX, int64_t ldx, int64_t ncols, int lower, int trans,
                      int unit, double scale, cudaStream_t stream, int right = 0);

// Cholesky factorization of one diagonal block of at most 128 x 128 in device memory (potrf_sm100.cu): the `lower` (1) or upper
// (0) triangle of dA is overwritten by its factor; *d_info (device, int64) receives info_base + j + 1 if the pivot of column j is
// not positive and *d_info was 0 (the block is then left partly factored).
int launch_potrf_block(double* dA, int64_t lda, int n, int lower, long long* d_info, long long info_base, cudaStream_t stream);

// number of CTAs the tile kernel uses for an M x N output (for stats / tests)
int64_t dgemm_tile_count(int64_t M, int64_t N);

}  // namespace hclooc
