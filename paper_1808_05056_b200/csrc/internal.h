// internal.h -- declarations shared by the translation units of libhclooc_b200 (not installed).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/hclooc.h"

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

// Launch the tile kernel: dC = alpha*dA*dB + beta*dC on device pointers (row-major).
// Preconditions (checked by callers): pointers 16-byte aligned, leading dimensions even.
int launch_dgemm_tiles(int64_t M, int64_t N, int64_t K, double alpha, const double* dA, int64_t lda,
                       const double* dB, int64_t ldb, double beta, double* dC, int64_t ldc,
                       cudaStream_t stream, int ksplit);   // ksplit: 1, 2, 4, or 0 = choose from the tile count

// K split (cluster size) worth using when `tiles_in_flight` tiles can run concurrently
int dgemm_auto_ksplit(int64_t tiles_in_flight, int64_t K);

// number of CTAs the tile kernel uses for an M x N output (for stats / tests)
int64_t dgemm_tile_count(int64_t M, int64_t N);

}  // namespace hclooc
