// dgemm_streamk_sm100.cu -- the S5 kernel for launches that should fill the whole GPU by themselves: a
// PERSISTENT tile kernel with a stream-K tail (the in-core case, and hclDgemmAsync).
//
//   dC = alpha * dA * dB + beta * dC
//
// Why: with one CTA per 128 x 128 tile, a launch of T tiles on G = 148 SMs runs ceil(T/G) waves; the last
// wave is partly empty (T = 1408: 9.51 waves run as 10, 95 %).  Here G persistent CTAs (one per SM) share
// the work evenly:
//   * data-parallel part: the first `dp_waves` waves, CTA c computes tiles c, c + G, c + 2G, ... whole;
//   * stream-K tail: the remaining G..2G-1 tiles (or all tiles if T < G) are laid end to end as a sequence
//     of k blocks and cut into G equal contiguous ranges, so a tile may be shared by two or more CTAs.
//     Every sharer stores its partial accumulators to a scratch slot and bumps the tile's counter; the CTA
//     that arrives LAST adds the partials up in k order (so the result does not depend on who is last) and
//     runs the epilogue.  Nobody ever waits for another CTA, so no co-residency is needed.
//   * the TMA producer warp runs through the same work list and keeps the 3-stage ring full across tile
//     boundaries: the loads of the next tile overlap the epilogue of this one.
// Inner loop, fragment layout and epilogue are those of dgemm_sm100.cu (dgemm_device.cuh).
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <mutex>
#include "internal.h"
#include "dgemm_device.cuh"

namespace hclooc {

using namespace dev;

namespace {

constexpr int SK_SLOT_BYTES = BM * BN * 8;                 // one partial tile: 128 KiB
constexpr int SK_MAX_CTAS = 148;
constexpr int SK_MAX_TAIL_TILES = 2 * SK_MAX_CTAS;
constexpr size_t SK_SCRATCH_BYTES = (size_t)2 * SK_MAX_CTAS * SK_SLOT_BYTES + SK_MAX_TAIL_TILES * sizeof(unsigned);
constexpr int SK_MIN_KBLOCKS = 256 / BK;                   // do not cut pieces shorter than 256 deep

struct SkParams {
    int tiles_m, tiles_n, nk;        // tile grid and k blocks per tile
    int G;                           // persistent CTAs
    int dp_waves;                    // whole-tile waves before the tail
    int tail_tiles;                  // tiles in the stream-K tail (0, or G .. 2G-1, or all T if T < G)
    long long tail_iters;            // tail_tiles * nk
};

// One unit of work: k blocks [kb0, kb1) of tile `tile`.
struct WorkItem {
    int tile, kb0, kb1, tail_index;  // tail_index = index of the tile inside the tail, -1 in the data-parallel part
};

// Enumerates the work items of CTA c in the order both the producer and the consumers follow.
struct WorkIter {
    const SkParams& P;
    int c, wave;
    long long pos, end;              // position inside the tail's k-block sequence
    __device__ WorkIter(const SkParams& p, int cta) : P(p), c(cta), wave(0) {
        pos = P.tail_iters * c / P.G;
        end = P.tail_iters * (c + 1) / P.G;
    }
    __device__ bool next(WorkItem& w) {
        if (wave < P.dp_waves) {
            w.tile = wave * P.G + c; w.kb0 = 0; w.kb1 = P.nk; w.tail_index = -1;
            ++wave;
            return true;
        }
        if (pos >= end) return false;
        const int t = (int)(pos / P.nk);
        const long long t0 = (long long)t * P.nk;
        const long long hi = min(end, t0 + P.nk);
        w.tile = P.dp_waves * P.G + t; w.kb0 = (int)(pos - t0); w.kb1 = (int)(hi - t0); w.tail_index = t;
        pos = hi;
        return true;
    }
};

__device__ __forceinline__ void st_partial(double* p, double x, double y) {
    asm volatile("st.global.cg.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(x), "d"(y) : "memory");
}
__device__ __forceinline__ void ld_partial(const double* p, double& x, double& y) {
    asm volatile("ld.global.cg.v2.f64 {%0, %1}, [%2];" : "=d"(x), "=d"(y) : "l"(p) : "memory");
}

template <bool TA, bool TB>       // operand stored transposed (hclooc_dgemm_t): only TMA boxes and fragment addressing change
__global__ void __launch_bounds__(NUM_THREADS, 1)
hclooc_dgemm_streamk_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                            double* __restrict__ C, long long ldc, int M, int N, double alpha, double beta,
                            const SkParams P, double* __restrict__ partials, unsigned* __restrict__ counters) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_base = smem_base + STAGES * STAGE_BYTES;
    __shared__ unsigned s_arrival;
    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const int cta = blockIdx.x;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(bar_base + 8 * s, 1);
            mbar_init(bar_base + 8 * (STAGES + s), NUM_CONSUMER_WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp >= NUM_CONSUMER_WARPS) {
        // ------------------------------------------------------------ producer warpgroup: warp 0 drives TMA over the whole work list
        regs_release_producer();
        if (warp == NUM_CONSUMER_WARPS && lane == 0) {
            asm volatile("prefetch.tensormap [%0];" ::"l"(&tmA) : "memory");
            asm volatile("prefetch.tensormap [%0];" ::"l"(&tmB) : "memory");
            int stage = 0;
            uint32_t phase = 0;
            WorkIter it(P, cta);
            WorkItem w;
            while (it.next(w)) {
                int tile_m, tile_n;
                tile_coords(w.tile, P.tiles_m, P.tiles_n, tile_m, tile_n);
                const int m0 = tile_m * BM, n0 = tile_n * BN;
                for (int kb = w.kb0; kb < w.kb1; ++kb) {
                    const uint32_t full = bar_base + 8 * stage;
                    mbar_wait(bar_base + 8 * (STAGES + stage), phase ^ 1u);
                    mbar_expect_tx(full, STAGE_BYTES);
                    const uint32_t sa = smem_base + stage * STAGE_BYTES;
                    const uint32_t sb = sa + A_STAGE_BYTES;
                    const int k0 = kb * BK;
                    if (!TA) {
                        #pragma unroll
                        for (int hk = 0; hk < BK / 16; ++hk) tma_load_2d(sa + hk * A_HALF_BYTES, &tmA, k0 + 16 * hk, m0, full);
                    } else {
                        #pragma unroll
                        for (int b = 0; b < BM / 16; ++b) tma_load_2d(sa + b * B_BOX_BYTES, &tmA, m0 + 16 * b, k0, full);
                    }
                    if (!TB) {
                        #pragma unroll
                        for (int b = 0; b < BN / 16; ++b) tma_load_2d(sb + b * B_BOX_BYTES, &tmB, n0 + 16 * b, k0, full);
                    } else {
                        #pragma unroll
                        for (int hk = 0; hk < BK / 16; ++hk) tma_load_2d(sb + hk * A_HALF_BYTES, &tmB, k0 + 16 * hk, n0, full);
                    }
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
            }
        }
        return;
    }

    // ---------------------------------------------------------------- consumer warps: DMMA
    regs_take_consumer();
    FragLanesT<TA, TB> f;
    f.init(warp, lane);
    int stage = 0;
    uint32_t phase = 0;
    WorkIter it(P, cta);
    WorkItem w;
    while (it.next(w)) {
        double acc[4][4][2][2];
        #pragma unroll
        for (int u = 0; u < 4; ++u)
            #pragma unroll
            for (int bx = 0; bx < 4; ++bx)
                #pragma unroll
                for (int v = 0; v < 2; ++v) { acc[u][bx][v][0] = 0.0; acc[u][bx][v][1] = 0.0; }
        int tile_m, tile_n;
        tile_coords(w.tile, P.tiles_m, P.tiles_n, tile_m, tile_n);
        const int m0 = tile_m * BM, n0 = tile_n * BN;
        const int nu = edge_groups(M, m0 + f.wm * 32, 8), nbx = edge_groups(N, n0 + f.wn * 64, 16);
        if (nu != 0 && nbx != 0) {
            for (int kb = w.kb0; kb < w.kb1; ++kb) {
                mbar_wait(bar_base + 8 * stage, phase);
                mma_kblock(acc, smem_base + stage * STAGE_BYTES, f);
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_base + 8 * (STAGES + stage));
                if (++stage == STAGES) { stage = 0; phase ^= 1u; }
            }
        } else {                                  // this warp's part of the tile lies outside C: only keep the ring moving
            for (int kb = w.kb0; kb < w.kb1; ++kb) {
                mbar_wait(bar_base + 8 * stage, phase);
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_base + 8 * (STAGES + stage));
                if (++stage == STAGES) { stage = 0; phase ^= 1u; }
            }
        }
        if (w.kb0 != 0 || w.kb1 != P.nk) {
            // ---------------------------------------------------- this CTA holds only part of the tile's k range
            const long long t0 = (long long)w.tail_index * P.nk;
            // sharers of the tile: CTAs whose ranges [tail_iters*c/G, tail_iters*(c+1)/G) meet [t0, t0 + nk)
            int c_first = (int)((t0 * P.G) / P.tail_iters);
            while (P.tail_iters * (c_first + 1) / P.G <= t0) ++c_first;
            while (c_first > 0 && P.tail_iters * c_first / P.G > t0) --c_first;
            int c_last = (int)(((t0 + P.nk - 1) * P.G) / P.tail_iters);
            while (c_last + 1 < P.G && P.tail_iters * (c_last + 1) / P.G <= t0 + P.nk - 1) ++c_last;
            while (P.tail_iters * c_last / P.G > t0 + P.nk - 1) --c_last;
            const int n_sharers = c_last - c_first + 1;
            // slot: 2*cta + (0 if the piece starts this CTA's range, 1 otherwise); [i][tid] double2 layout, coalesced
            const bool first_piece = (t0 + w.kb0 == P.tail_iters * cta / P.G);
            double* mine = partials + ((size_t)(2 * cta + (first_piece ? 0 : 1)) * (SK_SLOT_BYTES / 8)) + 2 * threadIdx.x;
            #pragma unroll
            for (int u = 0; u < 4; ++u)
                #pragma unroll
                for (int bx = 0; bx < 4; ++bx)
                    #pragma unroll
                    for (int v = 0; v < 2; ++v)
                        st_partial(mine + ((u * 4 + bx) * 2 + v) * (NUM_CONSUMER_WARPS * 32 * 2), acc[u][bx][v][0], acc[u][bx][v][1]);
            __threadfence();
            asm volatile("bar.sync 1, %0;" ::"n"(NUM_CONSUMER_WARPS * 32) : "memory");
            if (threadIdx.x == 0) s_arrival = atomicAdd(&counters[w.tail_index], 1u);
            asm volatile("bar.sync 1, %0;" ::"n"(NUM_CONSUMER_WARPS * 32) : "memory");
            const bool last = (s_arrival == (unsigned)(n_sharers - 1));
            asm volatile("bar.sync 1, %0;" ::"n"(NUM_CONSUMER_WARPS * 32) : "memory");   // s_arrival may be rewritten next item
            if (!last) continue;
            __threadfence();
            if (threadIdx.x == 0) counters[w.tail_index] = 0;          // scratch is reusable by the next launch
            #pragma unroll
            for (int u = 0; u < 4; ++u)
                #pragma unroll
                for (int bx = 0; bx < 4; ++bx)
                    #pragma unroll
                    for (int v = 0; v < 2; ++v) { acc[u][bx][v][0] = 0.0; acc[u][bx][v][1] = 0.0; }
            #pragma unroll 1
            for (int cc = c_first; cc <= c_last; ++cc) {               // k order: deterministic sum
                const bool fp = (P.tail_iters * cc / P.G >= t0);       // the sharer's piece starts its own range
                const double* src = partials + ((size_t)(2 * cc + (fp ? 0 : 1)) * (SK_SLOT_BYTES / 8)) + 2 * threadIdx.x;
                #pragma unroll
                for (int u = 0; u < 4; ++u)
                    #pragma unroll
                    for (int bx = 0; bx < 4; ++bx)
                        #pragma unroll
                        for (int v = 0; v < 2; ++v) {
                            double p0, p1;
                            ld_partial(src + ((u * 4 + bx) * 2 + v) * (NUM_CONSUMER_WARPS * 32 * 2), p0, p1);
                            acc[u][bx][v][0] += p0;
                            acc[u][bx][v][1] += p1;
                        }
            }
        }
        epilogue_store(acc, C, ldc, M, N, m0, n0, alpha, beta, f);
    }
}

// ---------------------------------------------------------------------------------------------
// scratch pool: a stream-K launch needs partial slots and counters of its own while it runs
struct Scratch {
    void* mem = nullptr;
    cudaStream_t last_stream = nullptr;
    cudaEvent_t done = nullptr;
    bool used = false;
};
constexpr int POOL = 4;
Scratch g_pool[POOL];
std::mutex g_pool_mu;
int g_pool_device = -1;

// Returns a scratch buffer that no launch in flight on ANOTHER stream is using, or nullptr.
Scratch* acquire_scratch(cudaStream_t stream) {
    std::lock_guard<std::mutex> lk(g_pool_mu);
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return nullptr;
    if (g_pool_device >= 0 && g_pool_device != dev) return nullptr;       // pool lives on one device
    Scratch* pick = nullptr;
    for (Scratch& s : g_pool)
        if (s.mem && s.used && s.last_stream == stream) { pick = &s; break; }   // in-order with its previous user
    if (!pick)
        for (Scratch& s : g_pool)
            if (s.mem && (!s.used || cudaEventQuery(s.done) == cudaSuccess)) { pick = &s; break; }
    if (!pick)
        for (Scratch& s : g_pool)
            if (!s.mem) {
                if (cudaMalloc(&s.mem, SK_SCRATCH_BYTES) != cudaSuccess) { cudaGetLastError(); s.mem = nullptr; return nullptr; }
                if (cudaMemset((uint8_t*)s.mem + (size_t)2 * SK_MAX_CTAS * SK_SLOT_BYTES, 0, SK_MAX_TAIL_TILES * sizeof(unsigned)) != cudaSuccess ||
                    cudaEventCreateWithFlags(&s.done, cudaEventDisableTiming) != cudaSuccess) {
                    cudaGetLastError(); cudaFree(s.mem); s.mem = nullptr; return nullptr;
                }
                g_pool_device = dev;
                pick = &s;
                break;
            }
    cudaGetLastError();                                                   // cudaEventQuery's cudaErrorNotReady is not an error
    if (pick) { pick->last_stream = stream; pick->used = true; }
    return pick;
}

int ensure_attr() {
    static int status = -1;
    static std::once_flag once;
    std::call_once(once, [] {
        cudaError_t e = cudaFuncSetAttribute(hclooc_dgemm_streamk_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(hclooc_dgemm_streamk_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(hclooc_dgemm_streamk_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(hclooc_dgemm_streamk_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
        status = (e == cudaSuccess) ? 0 : cuda_fail(e);
    });
    return status;
}

}  // namespace

// Work split of a stream-K launch (host side, also used by the tests through hclooc_streamk_layout).
bool streamk_layout(int64_t M, int64_t N, int64_t K, int num_sms, int* G, int* dp_waves, int* tail_tiles) {
    const int64_t tm = (M + BM - 1) / BM, tn = (N + BN - 1) / BN, T = tm * tn, nk = (K + BK - 1) / BK;
    if (T <= 0 || nk <= 0 || T > 0x3fffffffLL) return false;
    const int sms = num_sms < SK_MAX_CTAS ? num_sms : SK_MAX_CTAS;
    int g = sms, waves = 0;
    int64_t tail = 0;
    if (T >= sms) {
        tail = T % sms;
        waves = (int)(T / sms);
        if (tail != 0) { tail += sms; --waves; }                          // one whole wave joins the tail: 1 <= tail/G < 2
    } else {
        tail = T;
        const int64_t pieces = (T * nk) / SK_MIN_KBLOCKS;                 // pieces of at least SK_MIN_KBLOCKS k blocks
        g = (int)(pieces < 1 ? 1 : (pieces < sms ? pieces : sms));
        if (g < T) g = (int)T;                                            // never fewer CTAs than tiles
        if (g > sms) return false;
    }
    *G = g; *dp_waves = waves; *tail_tiles = (int)tail;
    return true;
}

// Launch the persistent kernel if it applies (a scratch buffer is free, shapes fit); returns 1 if it did not
// apply (the caller falls back to one CTA per tile), 0 on success, an error code otherwise.
size_t streamk_scratch_bytes() { return (SK_SCRATCH_BYTES + 1023) / 1024 * 1024; }
size_t streamk_counter_offset() { return (size_t)2 * SK_MAX_CTAS * SK_SLOT_BYTES; }
size_t streamk_counter_bytes() { return SK_MAX_TAIL_TILES * sizeof(unsigned); }

int launch_dgemm_streamk(int64_t M, int64_t N, int64_t K, double alpha, const CUtensorMap& tmA, const CUtensorMap& tmB,
                         double beta, double* dC, int64_t ldc, cudaStream_t stream, void* scratch, int transa, int transb) {
    static int num_sms = 0;
    if (num_sms == 0) {
        int dev = 0, n = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 1;
        num_sms = n;
    }
    SkParams P;
    if (!streamk_layout(M, N, K, num_sms, &P.G, &P.dp_waves, &P.tail_tiles)) return 1;
    P.tiles_m = (int)((M + BM - 1) / BM); P.tiles_n = (int)((N + BN - 1) / BN); P.nk = (int)((K + BK - 1) / BK);
    P.tail_iters = (long long)P.tail_tiles * P.nk;
    int rc = ensure_attr();
    if (rc) return rc;
    // scratch given by the caller (a pipeline step: carved from the call's workspace, counters zeroed by the
    // executor, used by one stream only) or taken from the library's pool
    Scratch* sc = scratch ? nullptr : acquire_scratch(stream);
    if (!scratch && !sc) return 1;
    void* mem = scratch ? scratch : sc->mem;
    double* partials = (double*)mem;
    unsigned* counters = (unsigned*)((uint8_t*)mem + (size_t)2 * SK_MAX_CTAS * SK_SLOT_BYTES);
    if (transa && transb) hclooc_dgemm_streamk_kernel<true, true><<<P.G, NUM_THREADS, SMEM_BYTES, stream>>>(tmA, tmB, dC, (long long)ldc, (int)M, (int)N, alpha, beta, P, partials, counters);
    else if (transa) hclooc_dgemm_streamk_kernel<true, false><<<P.G, NUM_THREADS, SMEM_BYTES, stream>>>(tmA, tmB, dC, (long long)ldc, (int)M, (int)N, alpha, beta, P, partials, counters);
    else if (transb) hclooc_dgemm_streamk_kernel<false, true><<<P.G, NUM_THREADS, SMEM_BYTES, stream>>>(tmA, tmB, dC, (long long)ldc, (int)M, (int)N, alpha, beta, P, partials, counters);
    else hclooc_dgemm_streamk_kernel<false, false><<<P.G, NUM_THREADS, SMEM_BYTES, stream>>>(tmA, tmB, dC, (long long)ldc, (int)M, (int)N, alpha, beta, P, partials, counters);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && sc) e = cudaEventRecord(sc->done, stream);
    if (e != cudaSuccess) return cuda_fail(e);
    return HCLOOC_OK;
}

}  // namespace hclooc

// ---------------------------------------------------------------------------------------------
// hclDgemmNoAlloc: the persistent stream-K kernel for callers that cannot allocate (CUDA graph capture, serving loops, harnesses
// that forbid cudaMalloc).  The kernel is the one above, unchanged; the partial-tile slots and tile counters it needs sit in a
// file-scope device array instead of the cudaMalloc'ed pool of acquire_scratch.  Every GPU that loads the library holds the array
// (HCL_NOALLOC_SCRATCH_BYTES, 37.0 MiB) until the process exits.  In host code `g_noalloc_scratch` is only a stand-in for the
// symbol: the device address comes from cudaGetSymbolAddress, once per device, with that device current.
namespace hclooc {
namespace {

constexpr size_t NA_PARTIAL_BYTES = (size_t)2 * SK_MAX_CTAS * SK_SLOT_BYTES;                    // 2 slots per persistent CTA
constexpr size_t NA_COUNTER_BYTES = SK_MAX_TAIL_TILES * sizeof(unsigned);
constexpr size_t NA_SCRATCH_BYTES = (NA_PARTIAL_BYTES + NA_COUNTER_BYTES + 255) / 256 * 256;
static_assert(NA_SCRATCH_BYTES == HCL_NOALLOC_SCRATCH_BYTES, "include/hclooc.h states the size of the static scratch");
static_assert(NA_PARTIAL_BYTES % 256 == 0, "the counters start on a 256-byte boundary");

static __device__ __align__(256) unsigned char g_noalloc_scratch[NA_SCRATCH_BYTES];

constexpr int NA_MAX_DEVICES = 64;
struct NoAllocDevice {
    void* scratch = nullptr;        // device address of g_noalloc_scratch on this device
    int num_sms = 0;
    bool ready = false;
};
NoAllocDevice g_na_dev[NA_MAX_DEVICES];
std::mutex g_na_mu;

// Set-up of the CURRENT device (once per device): the array's device address, the SM count, the kernel's shared-memory limit.
int noalloc_setup(NoAllocDevice** out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e);
    if (dev < 0 || dev >= NA_MAX_DEVICES) return HCLOOC_ERR_INTERNAL;
    std::lock_guard<std::mutex> lk(g_na_mu);
    NoAllocDevice& d = g_na_dev[dev];
    if (!d.ready) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess) return cuda_fail(e);
        if (!p || ((uintptr_t)p & 255u)) return HCLOOC_ERR_INTERNAL;
        int n = 0;
        e = cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(hclooc_dgemm_streamk_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
        if (e != cudaSuccess) return cuda_fail(e);
        d.scratch = p; d.num_sms = n; d.ready = true;
    }
    *out = &d;
    return HCLOOC_OK;
}

}  // namespace
}  // namespace hclooc

extern "C" size_t hclDgemmNoAllocScratchBytes(void) { return hclooc::NA_SCRATCH_BYTES; }

extern "C" int hclDgemmNoAlloc(int64_t M, int64_t N, int64_t K, double alpha, const double* dA, int64_t lda, const double* dB,
                               int64_t ldb, double beta, double* dC, int64_t ldc, hclStream s) {
    using namespace hclooc;
    if (M < 0) return -1;
    if (N < 0) return -2;
    if (K < 0) return -3;
    // the maximum: what the kernel indexes with 32-bit integers and what the static array has slots and counters for
    if (M > HCL_NOALLOC_MAX_DIM || N > HCL_NOALLOC_MAX_DIM || K > HCL_NOALLOC_MAX_DIM) return HCLOOC_ERR_NOALLOC_LIMIT;
    if (((M + BM - 1) / BM) * ((N + BN - 1) / BN) > HCL_NOALLOC_MAX_TILES) return HCLOOC_ERR_NOALLOC_LIMIT;
    if (M == 0 || N == 0) return HCLOOC_OK;
    const bool noab = (alpha == 0.0 || K == 0);
    if (!noab) {
        if (!dA) return -5;
        if (lda < K) return -6;
        if (!dB) return -7;
        if (ldb < N) return -8;
        if (((uintptr_t)dA & 15u) || ((uintptr_t)dB & 15u) || (lda & 1) || (ldb & 1)) return HCLOOC_ERR_ALIGN;
    }
    if (!dC) return -10;
    if (ldc < N) return -11;
    cudaStream_t stream = (cudaStream_t)s;
    if (noab)                                        // dC = beta * dC: one CTA per tile, no scratch, nothing allocated either
        return launch_dgemm_tiles(M, N, 0, 0.0, nullptr, 2, nullptr, 2, beta, dC, ldc, stream, 1);
    NoAllocDevice* d = nullptr;
    int rc = noalloc_setup(&d);
    if (rc) return rc;
    SkParams P;
    if (!streamk_layout(M, N, K, d->num_sms, &P.G, &P.dp_waves, &P.tail_tiles)) return HCLOOC_ERR_NOALLOC_LIMIT;
    if (P.G > SK_MAX_CTAS || P.tail_tiles > SK_MAX_TAIL_TILES) return HCLOOC_ERR_NOALLOC_LIMIT;     // more than the array holds
    P.tiles_m = (int)((M + BM - 1) / BM); P.tiles_n = (int)((N + BN - 1) / BN); P.nk = (int)((K + BK - 1) / BK);
    P.tail_iters = (long long)P.tail_tiles * P.nk;
    CUtensorMap tmA, tmB;
    if ((rc = make_tensor_map(&tmA, dA, M, K, lda, BM))) return rc;
    if ((rc = make_tensor_map(&tmB, dB, K, N, ldb, BK))) return rc;
    double* partials = (double*)d->scratch;
    unsigned* counters = (unsigned*)((uint8_t*)d->scratch + NA_PARTIAL_BYTES);
    // the array keeps what the last call left: the partial slots are written before they are read, the counters must start at zero
    // (a launch resets the ones it used, but a launch that was aborted or is still running on another stream may not have)
    HCL_CUDA(cudaMemsetAsync(counters, 0, NA_COUNTER_BYTES, stream));
    hclooc_dgemm_streamk_kernel<false, false><<<P.G, NUM_THREADS, SMEM_BYTES, stream>>>(tmA, tmB, dC, (long long)ldc, (int)M, (int)N,
                                                                                        alpha, beta, P, partials, counters);
    HCL_CUDA(cudaGetLastError());
    return HCLOOC_OK;
}
