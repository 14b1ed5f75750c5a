// dgemm_sm100.cu -- the S5 step of the pipeline: the in-core FP64 tile kernel for sm_100a.
//
//   dC = alpha * dA * dB + beta * dC      ("DGEMM ... c_ij = alpha x a_i b_j + beta x c_ij";
//                                          the paper calls a vendor library here (:308), this is ours)
//
// Design:
//   * FP64 on B200 peaks on the DMMA pipe (mma.sync.m8n8k4.f64 -> SASS DMMA.8x8x4): measured
//     37.17 TFLOP/s vs 33.7 for DFMA, so the inner product is DMMA.  tcgen05 has no FP64 kind.
//   * CTA tile 128 x 128, K step 16, 8 consumer warps (4 along m x 2 along n, warp tile 32 x 64 =
//     4 x 8 DMMA tiles, 64 FP64 accumulators per thread) + 1 producer warp.
//   * A/B tiles are staged by TMA (cp.async.bulk.tensor.2d, 128-byte swizzle, zero fill outside the
//     matrix -> ragged M/N/K tails cost nothing in the main loop) into a 6-stage shared-memory ring
//     guarded by full/empty mbarriers; no __syncthreads in the main loop.
//   * Fragment loads are LDS.128 and bank-conflict free: inside a tile the 8 rows of a DMMA m-tile,
//     its 4 k indices and the 8 columns of an n-tile are PERMUTED (any permutation of m, n or k that
//     A, B and C agree on leaves the product unchanged) so that the swizzled 16-byte chunks of a
//     quarter warp fall on distinct banks, and one LDS.128 feeds two DMMAs.
//   * Epilogue fused: alpha*acc + beta*C straight from registers, C not read when beta == 0.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <mutex>
#include "internal.h"

namespace hclooc {

namespace {

constexpr int BM = 128;
constexpr int BN = 128;
constexpr int BK = 16;
constexpr int STAGES = 6;
constexpr int A_STAGE_BYTES = BM * BK * 8;          // 16 KiB: 128 rows x 128 B
constexpr int B_BOX_BYTES = BK * 16 * 8;            // 2 KiB: 16 k-rows x 128 B (16 columns)
constexpr int B_STAGE_BYTES = (BN / 16) * B_BOX_BYTES;  // 16 KiB
constexpr int STAGE_BYTES = A_STAGE_BYTES + B_STAGE_BYTES;
constexpr int NUM_CONSUMER_WARPS = 8;
constexpr int NUM_THREADS = (NUM_CONSUMER_WARPS + 1) * 32;
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*align slack*/ + 2 * STAGES * 8;
constexpr int RASTER_GROUP = 16;                     // m-tiles per rasterisation group

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE;\n"
        "bra WAIT_LOOP;\n"
        "DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
__device__ __forceinline__ void lds128(double& x, double& y, uint32_t addr) {
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(x), "=d"(y) : "r"(addr));
}
__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                 : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void ld_dsmem128(double& x, double& y, uint32_t local_addr, uint32_t rank) {
    uint32_t remote;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(local_addr), "r"(rank));
    asm volatile("ld.shared::cluster.v2.f64 {%0, %1}, [%2];" : "=d"(x), "=d"(y) : "r"(remote) : "memory");
}

// One CTA computes one 128 x 128 tile of C over the whole K range (KSPLIT == 1), or a cluster of KSPLIT
// CTAs shares the tile: CTA r of the cluster takes the r-th share of the k blocks, the partial
// accumulators are reduced through distributed shared memory in rank order (deterministic) and CTA 0
// runs the epilogue.  Used when a pipeline step has too few tiles to fill 148 SMs.
template <int KSPLIT>
__global__ void __launch_bounds__(NUM_THREADS, 1)
hclooc_dgemm_tile_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                         double* __restrict__ C, long long ldc, int M, int N, int K,
                         double alpha, double beta, int tiles_m, int tiles_n) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;   // 128B swizzle wants 1 KiB alignment
    const uint32_t bar_base = smem_base + STAGES * STAGE_BYTES;          // full[s] at +8s, empty[s] at +8(STAGES+s)
    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;

    // tile rasterisation: groups of RASTER_GROUP m-tiles, m fastest inside a group, so CTAs that run
    // together share B column panels and a bounded set of A row panels in L2
    int tile_m, tile_n;
    {
        const int per_group = RASTER_GROUP * tiles_n;
        const int tile = (KSPLIT == 1) ? (int)blockIdx.x : (int)(blockIdx.x / KSPLIT);
        const int grp = tile / per_group;
        const int rem = tile - grp * per_group;
        const int gm0 = grp * RASTER_GROUP;
        const int gsz = min(RASTER_GROUP, tiles_m - gm0);
        tile_m = gm0 + rem % gsz;
        tile_n = rem / gsz;
    }
    const int m0 = tile_m * BM;
    const int n0 = tile_n * BN;
    const int num_kb_all = (K + BK - 1) / BK;
    const uint32_t crank = (KSPLIT == 1) ? 0u : cluster_ctarank();
    const int kb_begin = (KSPLIT == 1) ? 0 : (int)(((long long)num_kb_all * crank) / KSPLIT);
    const int kb_end = (KSPLIT == 1) ? num_kb_all : (int)(((long long)num_kb_all * (crank + 1)) / KSPLIT);
    const int num_kb = kb_end - kb_begin;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(bar_base + 8 * s, 1);
            mbar_init(bar_base + 8 * (STAGES + s), NUM_CONSUMER_WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == NUM_CONSUMER_WARPS) {
        // ------------------------------------------------------------ producer warp: TMA
        if (lane == 0 && num_kb > 0) {
            asm volatile("prefetch.tensormap [%0];" ::"l"(&tmA) : "memory");
            asm volatile("prefetch.tensormap [%0];" ::"l"(&tmB) : "memory");
            int stage = 0;
            uint32_t phase = 0;
            for (int kb = 0; kb < num_kb; ++kb) {
                const uint32_t full = bar_base + 8 * stage;
                const uint32_t empty = bar_base + 8 * (STAGES + stage);
                mbar_wait(empty, phase ^ 1u);
                mbar_expect_tx(full, STAGE_BYTES);
                const uint32_t sa = smem_base + stage * STAGE_BYTES;
                const uint32_t sb = sa + A_STAGE_BYTES;
                const int k0 = (kb_begin + kb) * BK;
                tma_load_2d(sa, &tmA, k0, m0, full);
                #pragma unroll
                for (int b = 0; b < BN / 16; ++b) tma_load_2d(sb + b * B_BOX_BYTES, &tmB, n0 + 16 * b, k0, full);
                if (++stage == STAGES) { stage = 0; phase ^= 1u; }
            }
        }
        if (KSPLIT == 1) return;
        __syncwarp();
        cluster_sync_all();      // partials written
        cluster_sync_all();      // partials read: peers may exit
        return;
    }

    // ---------------------------------------------------------------- consumer warps: DMMA
    const int g = lane >> 2;                  // fragment row group
    const int t = lane & 3;                   // fragment k / column-pair index
    const int rp = 4 * (g & 1) + (g >> 1);    // row permutation inside an 8-row m-tile
    const int wm = warp & 3;                  // warp row   (32 rows each)
    const int wn = warp >> 2;                 // warp column (64 columns each)

    // per-lane shared-memory byte offsets inside a stage (see the header comment for the layout)
    const uint32_t a_lane = (uint32_t)((wm * 32 + rp) * 128 + ((t ^ rp) << 4));
    uint32_t b_lane[2];
    #pragma unroll
    for (int e = 0; e < 2; ++e)
        b_lane[e] = (uint32_t)(A_STAGE_BYTES + wn * 4 * B_BOX_BYTES + (2 * t + e) * 128 + ((g ^ (2 * t + e)) << 4));

    double acc[4][4][2][2];
    #pragma unroll
    for (int u = 0; u < 4; ++u)
        #pragma unroll
        for (int bx = 0; bx < 4; ++bx)
            #pragma unroll
            for (int v = 0; v < 2; ++v) { acc[u][bx][v][0] = 0.0; acc[u][bx][v][1] = 0.0; }

    {
        int stage = 0;
        uint32_t phase = 0;
        for (int kb = 0; kb < num_kb; ++kb) {
            mbar_wait(bar_base + 8 * stage, phase);
            const uint32_t sbase = smem_base + stage * STAGE_BYTES;
            #pragma unroll
            for (int kg = 0; kg < 2; ++kg) {
                double a[4][2];
                #pragma unroll
                for (int u = 0; u < 4; ++u) lds128(a[u][0], a[u][1], sbase + ((a_lane ^ (kg << 6)) + u * 1024));
                #pragma unroll
                for (int e = 0; e < 2; ++e) {
                    double b[4][2];
                    #pragma unroll
                    for (int bx = 0; bx < 4; ++bx)
                        lds128(b[bx][0], b[bx][1], sbase + b_lane[e] + kg * 1024 + bx * B_BOX_BYTES);
                    #pragma unroll
                    for (int u = 0; u < 4; ++u)
                        #pragma unroll
                        for (int bx = 0; bx < 4; ++bx) {
                            dmma(acc[u][bx][0], a[u][e], b[bx][0]);
                            dmma(acc[u][bx][1], a[u][e], b[bx][1]);
                        }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_base + 8 * (STAGES + stage));
            if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
    }

    // ---------------------------------------------------------------- split-K reduction over the cluster (DSMEM)
    if (KSPLIT > 1) {
        // every consumer warp of this CTA is done reading the stage buffers before they are reused
        asm volatile("bar.sync 1, %0;" ::"n"(NUM_CONSUMER_WARPS * 32) : "memory");
        const uint32_t slot = smem_base + threadIdx.x * 16;          // [i][tid] double2 layout: conflict free
        if (crank != 0) {
            #pragma unroll
            for (int u = 0; u < 4; ++u)
                #pragma unroll
                for (int bx = 0; bx < 4; ++bx)
                    #pragma unroll
                    for (int v = 0; v < 2; ++v)
                        asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(slot + ((u * 4 + bx) * 2 + v) * (NUM_CONSUMER_WARPS * 32 * 16)),
                                     "d"(acc[u][bx][v][0]), "d"(acc[u][bx][v][1]) : "memory");
        }
        __syncwarp();
        cluster_sync_all();
        if (crank == 0) {
            #pragma unroll 1
            for (uint32_t r = 1; r < (uint32_t)KSPLIT; ++r) {
                #pragma unroll
                for (int u = 0; u < 4; ++u)
                    #pragma unroll
                    for (int bx = 0; bx < 4; ++bx)
                        #pragma unroll
                        for (int v = 0; v < 2; ++v) {
                            double p0, p1;
                            ld_dsmem128(p0, p1, slot + ((u * 4 + bx) * 2 + v) * (NUM_CONSUMER_WARPS * 32 * 16), r);
                            acc[u][bx][v][0] += p0;
                            acc[u][bx][v][1] += p1;
                        }
            }
        }
        __syncwarp();
        cluster_sync_all();
        if (crank != 0) return;
    }

    // ---------------------------------------------------------------- fused epilogue
    const bool read_c = (beta != 0.0);
    const bool vec_ok = ((ldc & 1LL) == 0) && ((reinterpret_cast<uintptr_t>(C) & 15u) == 0);
    #pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int row = m0 + wm * 32 + u * 8 + rp;
        if (row >= M) continue;
        double* crow = C + (long long)row * ldc;
        #pragma unroll
        for (int bx = 0; bx < 4; ++bx) {
            const int col = n0 + wn * 64 + bx * 16 + 4 * t;
            // lane holds 4 consecutive columns: (v=0,c0) (v=1,c0) (v=0,c1) (v=1,c1)
            double x0 = alpha * acc[u][bx][0][0], x1 = alpha * acc[u][bx][1][0];
            double x2 = alpha * acc[u][bx][0][1], x3 = alpha * acc[u][bx][1][1];
            if (col + 3 < N && vec_ok) {
                double2* p = reinterpret_cast<double2*>(crow + col);
                if (read_c) {
                    const double2 c01 = p[0], c23 = p[1];
                    x0 += beta * c01.x; x1 += beta * c01.y; x2 += beta * c23.x; x3 += beta * c23.y;
                }
                p[0] = make_double2(x0, x1);
                p[1] = make_double2(x2, x3);
            } else {
                const double xs[4] = {x0, x1, x2, x3};
                #pragma unroll
                for (int q = 0; q < 4; ++q)
                    if (col + q < N) crow[col + q] = read_c ? xs[q] + beta * crow[col + q] : xs[q];
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = nullptr;
    static std::once_flag once;
    std::call_once(once, [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    });
    return fn;
}

// 2-D FP64 tensor map over a row-major matrix (rows x cols, leading dimension ld elements),
// box = box_rows x 16 columns (128 bytes), 128-byte swizzle, zero fill out of bounds.
int make_map(CUtensorMap* map, const double* base, int64_t rows, int64_t cols, int64_t ld, int box_rows) {
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return HCLOOC_ERR_CUDA;
    cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    cuuint64_t strides[1] = {(cuuint64_t)ld * 8};
    cuuint32_t box[2] = {16, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double*>(base), dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { set_last_cuda_error(1000 + (int)r); return HCLOOC_ERR_CUDA; }
    return HCLOOC_OK;
}

int ensure_kernel_attr() {
    static int status = -1;
    static std::once_flag once;
    std::call_once(once, [] {
        cudaError_t e = cudaFuncSetAttribute(hclooc_dgemm_tile_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(hclooc_dgemm_tile_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(hclooc_dgemm_tile_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
        status = (e == cudaSuccess) ? 0 : cuda_fail(e);
    });
    return status;
}

template <int KSPLIT>
cudaError_t launch_split(unsigned tiles, cudaStream_t stream, const CUtensorMap& tmA, const CUtensorMap& tmB, double* dC,
                         long long ldc, int M, int N, int K, double alpha, double beta, int tm, int tn) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(tiles * KSPLIT, 1, 1);
    cfg.blockDim = dim3(NUM_THREADS, 1, 1);
    cfg.dynamicSmemBytes = SMEM_BYTES;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = KSPLIT;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, hclooc_dgemm_tile_kernel<KSPLIT>, tmA, tmB, dC, ldc, M, N, K, alpha, beta, tm, tn);
}

}  // namespace

int64_t dgemm_tile_count(int64_t M, int64_t N) { return ((M + BM - 1) / BM) * ((N + BN - 1) / BN); }

int dgemm_auto_ksplit(int64_t tiles_in_flight, int64_t K) {
    // split K over a 2- or 4-CTA cluster when the tiles that can run together leave most SMs idle
    if (K >= 2048 && tiles_in_flight * 4 <= 148) return 4;
    if (K >= 1024 && tiles_in_flight * 2 <= 148) return 2;
    return 1;
}

int launch_dgemm_tiles(int64_t M, int64_t N, int64_t K, double alpha, const double* dA, int64_t lda,
                       const double* dB, int64_t ldb, double beta, double* dC, int64_t ldc, cudaStream_t stream,
                       int ksplit) {
    if (M == 0 || N == 0) return HCLOOC_OK;
    if (alpha == 0.0) K = 0;                       // A and B are not referenced (BLAS convention)
    int rc = ensure_kernel_attr();
    if (rc) return rc;
    CUtensorMap tmA, tmB;
    if (K > 0) {
        if ((rc = make_map(&tmA, dA, M, K, lda, BM))) return rc;
        if ((rc = make_map(&tmB, dB, K, N, ldb, BK))) return rc;
    } else {
        memset(&tmA, 0, sizeof(tmA));
        memset(&tmB, 0, sizeof(tmB));
    }
    const int64_t tm = (M + BM - 1) / BM, tn = (N + BN - 1) / BN;
    if (tm * tn > 0x7fffffffLL || M > 0x7fffffffLL || N > 0x7fffffffLL || K > 0x7fffffffLL) return HCLOOC_ERR_INTERNAL;
    if (ksplit <= 0) ksplit = dgemm_auto_ksplit(tm * tn, K);
    if (K == 0) ksplit = 1;
    cudaError_t e;
    if (ksplit >= 4) e = launch_split<4>((unsigned)(tm * tn), stream, tmA, tmB, dC, (long long)ldc, (int)M, (int)N, (int)K, alpha, beta, (int)tm, (int)tn);
    else if (ksplit >= 2) e = launch_split<2>((unsigned)(tm * tn), stream, tmA, tmB, dC, (long long)ldc, (int)M, (int)N, (int)K, alpha, beta, (int)tm, (int)tn);
    else {
        hclooc_dgemm_tile_kernel<1><<<(unsigned)(tm * tn), NUM_THREADS, SMEM_BYTES, stream>>>(
            tmA, tmB, dC, (long long)ldc, (int)M, (int)N, (int)K, alpha, beta, (int)tm, (int)tn);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) return cuda_fail(e);
    return HCLOOC_OK;
}

}  // namespace hclooc
