// runtime.cu -- the uniform runtime the paper abstracts, CUDA only,
// as plain C functions: no factory, no virtual dispatch (the paper attributes part of its 4-10 %
// overhead to the virtual-table lookups, :164).
#include <cstring>
#include <algorithm>
#include <chrono>
#include <thread>
#include "internal.h"
#include "executor.h"
#include <algorithm>

using namespace hclooc;

namespace {
int finish_async(cudaStream_t s, hclEvent* ev) {
    if (!ev) return HCLOOC_OK;
    if (*ev == nullptr) {   // "an uninitialised hclEvent ... will create and initialise the event" (:146)
        cudaEvent_t e;
        HCL_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        *ev = (hclEvent)e;
    }
    HCL_CUDA(cudaEventRecord((cudaEvent_t)*ev, s));
    return HCLOOC_OK;
}
cudaMemcpyKind kind_of(int dir) { return dir == HCL_H2D ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToHost; }
}  // namespace

// ---------------------------------------------------------------------------------------------
// FP64 issue-rate probe (hclooc_probe_fp64): independent chains of DMMA.8x8x4 (kind 0) or DFMA (kind 1) in registers,
// no memory traffic -- the measured denominator of the roofline (148 SMs x 128 flop/clk x clock).
namespace {
__global__ void __launch_bounds__(256) probe_dmma_kernel(double* out, int iters) {
    double c[8][2];
    #pragma unroll
    for (int i = 0; i < 8; ++i) { c[i][0] = 0.0; c[i][1] = 0.0; }
    double a = 1.0 + 1e-9 * threadIdx.x, b = 1.0 - 1e-9 * threadIdx.x;
    for (int it = 0; it < iters; ++it) {
        #pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0.0;
    #pragma unroll
    for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
    if (s == 123.456) out[0] = s;        // keep the chains alive
}
__global__ void __launch_bounds__(256) probe_dfma_kernel(double* out, int iters) {
    double c[16];
    #pragma unroll
    for (int i = 0; i < 16; ++i) c[i] = 1e-3 * i;
    const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9 * threadIdx.x;
    for (int it = 0; it < iters; ++it) {
        #pragma unroll
        for (int i = 0; i < 16; ++i) c[i] = __fma_rn(c[i], a, b);
    }
    double s = 0.0;
    #pragma unroll
    for (int i = 0; i < 16; ++i) s += c[i];
    if (s == 123.456) out[0] = s;
}
}  // namespace

namespace {
__global__ void debug_spin_kernel(long long cycles) {
    const long long t0 = clock64();
    while (clock64() - t0 < cycles) { }
}
__global__ void debug_fill_kernel(double* p, long long ld, long long rows, long long cols, double v) {
    const long long n = rows * cols;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x)
        p[(e / cols) * ld + e % cols] = v;
}
}  // namespace

namespace hclooc {
void debug_jitter(hclooc_ctx* ctx, cudaStream_t s) {
    if (!ctx || !ctx->dbg_rng) return;
    uint64_t x = ctx->dbg_rng;
    x ^= x << 13; x ^= x >> 7; x ^= x << 17;
    ctx->dbg_rng = x ? x : 0x9E3779B97F4A7C15ull;
    if (x & 1) debug_spin_kernel<<<1, 1, 0, s>>>((long long)((x >> 8) % 300000));       // up to ~150 us at 1.965 GHz
}
void debug_poison(hclooc_ctx* ctx, double* p, int64_t ld, int64_t rows, int64_t cols, cudaStream_t s) {
    if (!ctx || !ctx->dbg_poison || !p || rows <= 0 || cols <= 0) return;
    const long long n = (long long)rows * cols;
    const unsigned grid = (unsigned)std::min<long long>(1184, (n + 255) / 256);
    const unsigned long long bits = 0x7ff8000000000badull;              // a quiet NaN with a recognisable payload
    double nan_v;
    memcpy(&nan_v, &bits, sizeof(nan_v));
    debug_fill_kernel<<<grid, 256, 0, s>>>(p, (long long)ld, (long long)rows, (long long)cols, nan_v);
}
}  // namespace hclooc

extern "C" {

int hclMalloc(void** dptr, size_t bytes) {
    if (!dptr) return -1;
    *dptr = nullptr;
    if (bytes == 0) return HCLOOC_OK;
    cudaError_t e = cudaMalloc(dptr, bytes);
    if (e == cudaErrorMemoryAllocation) { set_last_cuda_error((int)e); cudaGetLastError(); return HCLOOC_ERR_NOMEM; }
    if (e != cudaSuccess) return cuda_fail(e);
    return HCLOOC_OK;
}
int hclFree(void* dptr) {
    if (!dptr) return HCLOOC_OK;
    HCL_CUDA(cudaFree(dptr));
    return HCLOOC_OK;
}
int hclGetMemSize(int device, size_t* free_bytes) {
    if (device < 0) return -1;
    if (!free_bytes) return -2;
    int cur = 0;
    HCL_CUDA(cudaGetDevice(&cur));
    if (cur != device) HCL_CUDA(cudaSetDevice(device));
    size_t fr = 0, tot = 0;
    cudaError_t e = cudaMemGetInfo(&fr, &tot);
    if (cur != device) cudaSetDevice(cur);
    if (e != cudaSuccess) return cuda_fail(e);
    *free_bytes = fr;
    return HCLOOC_OK;
}
int hclStreamCreate(hclStream* s) {
    if (!s) return -1;
    cudaStream_t st;
    HCL_CUDA(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));
    *s = (hclStream)st;
    return HCLOOC_OK;
}
int hclStreamDestroy(hclStream s) {
    if (!s) return HCLOOC_OK;
    HCL_CUDA(cudaStreamDestroy((cudaStream_t)s));
    return HCLOOC_OK;
}
int hclEventDestroy(hclEvent e) {
    if (!e) return HCLOOC_OK;
    HCL_CUDA(cudaEventDestroy((cudaEvent_t)e));
    return HCLOOC_OK;
}
int hclMemcpy(void* dst, const void* src, size_t bytes, int dir) {
    if (bytes == 0) return HCLOOC_OK;
    if (!dst) return -1;
    if (!src) return -2;
    if (dir != HCL_H2D && dir != HCL_D2H) return -4;
    HCL_CUDA(cudaMemcpy(dst, src, bytes, kind_of(dir)));
    return HCLOOC_OK;
}
int hclMemcpyAsync(void* dst, const void* src, size_t bytes, int dir, hclStream s, hclEvent* ev) {
    if (bytes != 0) {
        if (!dst) return -1;
        if (!src) return -2;
        if (dir != HCL_H2D && dir != HCL_D2H) return -4;
        HCL_CUDA(cudaMemcpyAsync(dst, src, bytes, kind_of(dir), (cudaStream_t)s));
    }
    return finish_async((cudaStream_t)s, ev);
}
int hclMemcpy2DAsync(void* dst, size_t dpitch, const void* src, size_t spitch, size_t width_bytes, size_t rows,
                     int dir, hclStream s, hclEvent* ev) {
    if (width_bytes != 0 && rows != 0) {
        if (!dst) return -1;
        if (dpitch < width_bytes) return -2;
        if (!src) return -3;
        if (spitch < width_bytes) return -4;
        if (dir != HCL_H2D && dir != HCL_D2H) return -7;
        HCL_CUDA(cudaMemcpy2DAsync(dst, dpitch, src, spitch, width_bytes, rows, kind_of(dir), (cudaStream_t)s));
    }
    return finish_async((cudaStream_t)s, ev);
}
int hclDgemmAsyncEx(int64_t M, int64_t N, int64_t K, double alpha, const double* dA, int64_t lda, const double* dB,
                  int64_t ldb, double beta, double* dC, int64_t ldc, hclStream s, hclEvent* ev, int variant) {
    if (M < 0) return -1;
    if (N < 0) return -2;
    if (K < 0) return -3;
    const int ccm = (variant - 100) / 10, ccn = (variant - 100) % 10;
    const bool cluster = variant > 100 && (ccm == 1 || ccm == 2 || ccm == 4) && (ccn == 1 || ccn == 2 || ccn == 4);
    if (variant != HCL_DGEMM_AUTO && variant != -1 && variant != 1 && variant != 2 && variant != 4 && !cluster) return -14;
    const bool noab = (alpha == 0.0 || K == 0);
    if (M > 0 && N > 0) {
        if (!noab) {
            if (!dA) return -5;
            if (lda < K) return -6;
            if (!dB) return -7;
            if (ldb < N) return -8;
            if (((uintptr_t)dA & 15u) || ((uintptr_t)dB & 15u) || (lda & 1) || (ldb & 1)) return HCLOOC_ERR_ALIGN;
        }
        if (!dC) return -10;
        if (ldc < N) return -11;
        int rc = (cluster && !noab)
                     ? launch_dgemm_direct(M, N, K, alpha, dA, lda, dB, ldb, beta, dC, ldc, (cudaStream_t)s, ccm, ccn)
                     : launch_dgemm_tiles(M, N, K, alpha, dA, lda, dB, ldb, beta, dC, ldc, (cudaStream_t)s,
                                          variant == HCL_DGEMM_AUTO ? (dgemm_tile_count(M, N) >= 148 ? -1 : 0) : (cluster ? 1 : variant));
        if (rc) return rc;
    }
    return finish_async((cudaStream_t)s, ev);
}
int hclDgemmAsyncT(int transa, int transb, int64_t M, int64_t N, int64_t K, double alpha, const double* dA, int64_t lda,
                   const double* dB, int64_t ldb, double beta, double* dC, int64_t ldc, hclStream s, hclEvent* ev, int variant) {
    if (transa != HCL_OP_N && transa != HCL_OP_T) return -15;
    if (transb != HCL_OP_N && transb != HCL_OP_T) return -16;
    if (!transa && !transb) return hclDgemmAsyncEx(M, N, K, alpha, dA, lda, dB, ldb, beta, dC, ldc, s, ev, variant);
    if (M < 0) return -1;
    if (N < 0) return -2;
    if (K < 0) return -3;
    if (variant != HCL_DGEMM_AUTO && variant != -1 && variant != 1 && variant != 2 && variant != 4) return -14;
    const bool noab = (alpha == 0.0 || K == 0);
    if (M > 0 && N > 0) {
        if (!noab) {
            if (!dA) return -5;
            if (lda < (transa ? M : K)) return -6;
            if (!dB) return -7;
            if (ldb < (transb ? K : N)) return -8;
            if (((uintptr_t)dA & 15u) || ((uintptr_t)dB & 15u) || (lda & 1) || (ldb & 1)) return HCLOOC_ERR_ALIGN;
        }
        if (!dC) return -10;
        if (ldc < N) return -11;
        int rc = launch_dgemm_tiles(M, N, K, alpha, dA, lda, dB, ldb, beta, dC, ldc, (cudaStream_t)s,
                                    variant == HCL_DGEMM_AUTO ? (dgemm_tile_count(M, N) >= 148 ? -1 : 0) : variant, nullptr, transa, transb);
        if (rc) return rc;
    }
    return finish_async((cudaStream_t)s, ev);
}
int hclDgemmAsync(int64_t M, int64_t N, int64_t K, double alpha, const double* dA, int64_t lda, const double* dB, int64_t ldb,
                  double beta, double* dC, int64_t ldc, hclStream s, hclEvent* ev) {
    return hclDgemmAsyncEx(M, N, K, alpha, dA, lda, dB, ldb, beta, dC, ldc, s, ev, HCL_DGEMM_AUTO);
}
int hclWaitEvent(hclStream s, hclEvent e) {
    if (!e) return -2;
    HCL_CUDA(cudaStreamWaitEvent((cudaStream_t)s, (cudaEvent_t)e, 0));
    return HCLOOC_OK;
}
int hclStreamSynchronize(hclStream s) {
    HCL_CUDA(cudaStreamSynchronize((cudaStream_t)s));
    return HCLOOC_OK;
}
int hclDeviceSynchronize(int device) {
    if (device < 0) return -1;
    int cur = 0;
    HCL_CUDA(cudaGetDevice(&cur));
    if (cur != device) HCL_CUDA(cudaSetDevice(device));
    cudaError_t e = cudaDeviceSynchronize();
    if (cur != device) cudaSetDevice(cur);
    if (e != cudaSuccess) return cuda_fail(e);
    return HCLOOC_OK;
}

void* hclooc_host_alloc(size_t bytes) {
    void* p = nullptr;
    if (bytes == 0) return nullptr;
    // Pinning can fail transiently with cudaErrorOperatingSystem (304) although the host has the memory -- seen on the B200
    // boxes about once in eight fresh processes, succeeding two seconds later -- so a failed attempt is retried a few times.
    cudaError_t e = cudaSuccess;
    for (int attempt = 0; attempt < 6; ++attempt) {
        e = cudaHostAlloc(&p, bytes, cudaHostAllocDefault);
        if (e == cudaSuccess) return p;
        cudaGetLastError();
        if (e != cudaErrorOperatingSystem && e != cudaErrorMemoryAllocation) break;
        std::this_thread::sleep_for(std::chrono::seconds(2));
    }
    set_last_cuda_error((int)e);
    return nullptr;
}
int hclooc_host_free(void* p) {
    if (!p) return HCLOOC_OK;
    HCL_CUDA(cudaFreeHost(p));
    return HCLOOC_OK;
}
int hclooc_host_register(void* p, size_t bytes) {
    if (!p) return -1;
    if (bytes == 0) return -2;
    cudaError_t e = cudaSuccess;
    for (int attempt = 0; attempt < 6; ++attempt) {          // transient cudaErrorOperatingSystem: see hclooc_host_alloc
        e = cudaHostRegister(p, bytes, cudaHostRegisterDefault);
        if (e == cudaSuccess) return HCLOOC_OK;
        cudaGetLastError();
        if (e != cudaErrorOperatingSystem && e != cudaErrorMemoryAllocation) break;
        std::this_thread::sleep_for(std::chrono::seconds(2));
    }
    return cuda_fail(e);
}
int hclooc_host_unregister(void* p) {
    if (!p) return -1;
    HCL_CUDA(cudaHostUnregister(p));
    return HCLOOC_OK;
}

const char* hclooc_strerror(int status) {
    if (status == HCLOOC_OK) return "success";
    if (status < 0) return "invalid argument (the value is minus the 1-based argument number)";
    switch (status) {
        case HCLOOC_ERR_BUDGET: return "device budget below the minimum working set";
        case HCLOOC_ERR_NOT_PINNED: return "A, B or C is pageable host memory (pin it: hclooc_host_alloc / hclooc_host_register)";
        case HCLOOC_ERR_CUDA: return "a CUDA call failed (see hclooc_last_cuda_error)";
        case HCLOOC_ERR_NOMEM: return "out of device or host memory";
        case HCLOOC_ERR_ALIGN: return "device operand must be 16-byte aligned with an even leading dimension";
        case HCLOOC_ERR_INTERNAL: return "internal invariant violated";
        case HCLOOC_ERR_NOALLOC_LIMIT: return "hclDgemmNoAlloc: shape beyond the maximum its static scratch array serves (M, N, K <= 2^31 - 1, at most 2^30 - 1 tiles of 128 x 128)";
        default: return "unknown status";
    }
}
int hclooc_probe_fp64(int kind, int ctas_per_sm, double seconds, double* tflops) {
    if (kind != 0 && kind != 1) return -1;
    if (ctas_per_sm < 1 || ctas_per_sm > 8) return -2;
    if (!(seconds > 0.0) || seconds > 30.0) return -3;
    if (!tflops) return -4;
    int dev = 0, sms = 0;
    HCL_CUDA(cudaGetDevice(&dev));
    HCL_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double* d = nullptr;
    HCL_CUDA(cudaMalloc(&d, 8));
    cudaEvent_t e0, e1;
    HCL_CUDA(cudaEventCreate(&e0));
    HCL_CUDA(cudaEventCreate(&e1));
    const int grid = sms * ctas_per_sm;
    // flop per thread per iteration: DMMA: 8 chains x 512 flop per warp-wide instruction / 32 lanes; DFMA: 16 chains x 2
    const double flop_it = (kind == 0 ? 8.0 * 512.0 / 32.0 : 32.0) * 256.0 * grid;
    int iters = 1 << 14;
    double best = 0.0, total = 0.0;
    for (int rep = 0; rep < 64 && total < seconds; ++rep) {
        cudaEventRecord(e0, 0);
        if (kind == 0) probe_dmma_kernel<<<grid, 256>>>(d, iters); else probe_dfma_kernel<<<grid, 256>>>(d, iters);
        cudaEventRecord(e1, 0);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { cudaFree(d); return cuda_fail(e); }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0) { total += ms * 1e-3; best = std::max(best, flop_it * iters / (ms * 1e-3)); }
        if (ms < 20.f && iters < (1 << 24)) iters *= 2;         // launches of >= 20 ms
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
    *tflops = best / 1e12;
    return HCLOOC_OK;
}
const char* hclooc_version(void) { return "hclooc-b200 0.1 (sm_100a, DMMA tile kernel)"; }

}  // extern "C"
