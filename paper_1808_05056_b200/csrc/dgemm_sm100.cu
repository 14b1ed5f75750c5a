// dgemm_sm100.cu -- the S5 step of the pipeline: the in-core FP64 tile kernel for sm_100a.
//
//   dC = alpha * dA * dB + beta * dC      ("DGEMM ... c_ij = alpha x a_i b_j + beta x c_ij";
//                                          the paper calls a vendor library here (:308), this is ours)
//
// Design:
//   * FP64 on B200 peaks on the DMMA pipe (mma.sync.m8n8k4.f64 -> SASS DMMA.8x8x4): measured
//     37.17 TFLOP/s vs 33.7 for DFMA, so the inner product is DMMA.  tcgen05 has no FP64 kind.
//   * CTA tile 128 x 128, K step 32, 8 consumer warps (4 along m x 2 along n, warp tile 32 x 64 =
//     4 x 8 DMMA tiles, 64 FP64 accumulators per thread) + 1 producer warp.
//   * A/B tiles are staged by TMA (cp.async.bulk.tensor.2d, 128-byte swizzle, zero fill outside the
//     matrix -> ragged M/N/K tails cost nothing in the main loop) into a 3-stage (3 x 64 KiB) shared-memory ring
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
#include <cstdlib>
#include <cstring>
#include "internal.h"
#include "dgemm_device.cuh"

namespace hclooc {

namespace {

using namespace dev;

// One CTA computes one 128 x 128 tile of C over the whole K range (KSPLIT == 1), or a cluster of KSPLIT
// CTAs shares the tile: CTA r of the cluster takes the r-th share of the k blocks, the partial
// accumulators are reduced through distributed shared memory in rank order (deterministic) and CTA 0
// runs the epilogue.  Used when a pipeline step has too few tiles to fill 148 SMs.
// TA / TB: the operand is stored transposed (A as K x M, B as N x K; hclooc_dgemm_t): only the TMA boxes and the fragment
// addressing change (dgemm_device.cuh), the DMMA loop and the order of summation over k do not.
// MASK (KSPLIT == 1 only; hclooc_dtrmm / hclooc_dsymm): op(A) and / or op(B) is a TRIANGLE of the stored operand -- opmask = am | bm << 2,
// am / bm = 0 none, 1: op(A)[r][k] counts iff k <= r + adoff resp. op(B)[k][c] iff c <= k + bdoff, 2: iff >= (indices of this launch).
// A tile runs only over the k blocks that can hold counted elements, and the blocks that cross a diagonal zero the rest by a
// select in registers (mma_kblock<.., MASK>): what lies outside the triangle is never multiplied, NaN there is harmless.
template <int KSPLIT, bool TA = false, bool TB = false, bool MASK = false>
__global__ void __launch_bounds__(NUM_THREADS, 1)
hclooc_dgemm_tile_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                         double* __restrict__ C, long long ldc, int M, int N, int K,
                         double alpha, double beta, int tiles_m, int tiles_n, int tri, int doff,
                         int opmask = 0, int adoff = 0, int bdoff = 0) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;   // 128B swizzle wants 1 KiB alignment
    const uint32_t bar_base = smem_base + STAGES * STAGE_BYTES;          // full[s] at +8s, empty[s] at +8(STAGES+s)
    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;

    int tile_m, tile_n;
    tile_coords((KSPLIT == 1) ? (int)blockIdx.x : (int)(blockIdx.x / KSPLIT), tiles_m, tiles_n, tile_m, tile_n);
    const int m0 = tile_m * BM;
    const int n0 = tile_n * BN;
    // hclooc_dsyrk: a tile that lies entirely in the triangle of C that is not referenced has nothing to do (every CTA of a
    // split-K cluster shares the tile, so the whole cluster leaves together, before any barrier exists)
    if (tri == 1 && n0 > min(m0 + BM, M) - 1 + doff) return;
    if (tri == 2 && min(n0 + BN, N) - 1 < m0 + doff) return;
    const int num_kb_all = (K + BK - 1) / BK;
    const uint32_t crank = (KSPLIT == 1) ? 0u : cluster_ctarank();
    int kb_begin = (KSPLIT == 1) ? 0 : (int)(((long long)num_kb_all * crank) / KSPLIT);
    int kb_end = (KSPLIT == 1) ? num_kb_all : (int)(((long long)num_kb_all * (crank + 1)) / KSPLIT);
    const int am = MASK ? (opmask & 3) : 0, bm = MASK ? ((opmask >> 2) & 3) : 0;
    if (MASK) {
        // the k range in which this tile's rows of op(A) / columns of op(B) can hold counted elements
        long long klo = 0, khi = K;
        const int m1 = min(m0 + BM, M) - 1, n1 = min(n0 + BN, N) - 1;
        if (am == 1) khi = min(khi, (long long)m1 + adoff + 1);
        if (am == 2) klo = max(klo, (long long)m0 + adoff);
        if (bm == 1) klo = max(klo, (long long)n0 - bdoff);          // c <= k + bdoff  <=>  k >= c - bdoff
        if (bm == 2) khi = min(khi, (long long)n1 - bdoff + 1);
        kb_begin = (int)(max(klo, 0LL) / BK);
        kb_end = khi <= 0 ? 0 : (int)((khi + BK - 1) / BK);
        if (kb_end < kb_begin) kb_end = kb_begin;
    }
    const int num_kb = kb_end - kb_begin;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(bar_base + 8 * s, 1);
            mbar_init(bar_base + 8 * (STAGES + s), NUM_CONSUMER_WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp >= NUM_CONSUMER_WARPS) {
        // ------------------------------------------------------------ producer warpgroup: warp 0 drives TMA
        regs_release_producer();
        if (warp == NUM_CONSUMER_WARPS && lane == 0 && num_kb > 0) {
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
                if (!TA) {
                    #pragma unroll
                    for (int hk = 0; hk < BK / 16; ++hk) tma_load_2d(sa + hk * A_HALF_BYTES, &tmA, k0 + 16 * hk, m0, full);
                } else {        // stored K x M: eight boxes of 32 k-rows x 16 m
                    #pragma unroll
                    for (int b = 0; b < BM / 16; ++b) tma_load_2d(sa + b * B_BOX_BYTES, &tmA, m0 + 16 * b, k0, full);
                }
                if (!TB) {
                    #pragma unroll
                    for (int b = 0; b < BN / 16; ++b) tma_load_2d(sb + b * B_BOX_BYTES, &tmB, n0 + 16 * b, k0, full);
                } else {        // stored N x K: two 16-k halves of 128 n-rows
                    #pragma unroll
                    for (int hk = 0; hk < BK / 16; ++hk) tma_load_2d(sb + hk * A_HALF_BYTES, &tmB, k0 + 16 * hk, n0, full);
                }
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
    regs_take_consumer();
    FragLanesT<TA, TB> f;
    f.init(warp, lane);

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
        const int nu = edge_groups(M, m0 + f.wm * 32, 8), nbx = edge_groups(N, n0 + f.wn * 64, 16);
        if (nu != 0 && nbx != 0) {
            for (int kb = 0; kb < num_kb; ++kb) {
                mbar_wait(bar_base + 8 * stage, phase);
                if (MASK) {
                    // tile-local offsets of the diagonals in this k block; the block needs the select only if it crosses one
                    const int k0 = (kb_begin + kb) * BK;
                    const int da = m0 + adoff - k0, db = k0 + bdoff - n0;
                    const bool cross = (am == 1 && BK - 1 > da) || (am == 2 && 0 < BM - 1 + da) || (bm == 1 && BN - 1 > db) || (bm == 2 && 0 < BK - 1 + db);
                    if (cross) mma_kblock<TA, TB, true>(acc, smem_base + stage * STAGE_BYTES, f, am, da, bm, db);
                    else mma_kblock(acc, smem_base + stage * STAGE_BYTES, f);
                } else {
                    mma_kblock(acc, smem_base + stage * STAGE_BYTES, f);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_base + 8 * (STAGES + stage));
                if (++stage == STAGES) { stage = 0; phase ^= 1u; }
            }
        } else {                                  // this warp's part of the tile lies outside C: only keep the ring moving
            for (int kb = 0; kb < num_kb; ++kb) {
                mbar_wait(bar_base + 8 * stage, phase);
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_base + 8 * (STAGES + stage));
                if (++stage == STAGES) { stage = 0; phase ^= 1u; }
            }
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
    epilogue_store(acc, C, ldc, M, N, m0, n0, alpha, beta, f, tri, doff);
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

}  // namespace

// 2-D FP64 tensor map over a row-major matrix (rows x cols, leading dimension ld elements),
// box = box_rows x 16 columns (128 bytes), 128-byte swizzle, zero fill out of bounds.
int make_tensor_map(CUtensorMap* map, const double* base, int64_t rows, int64_t cols, int64_t ld, int box_rows) {
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

namespace {
inline int make_map(CUtensorMap* map, const double* base, int64_t rows, int64_t cols, int64_t ld, int box_rows) {
    return make_tensor_map(map, base, rows, cols, ld, box_rows);
}

template <bool TA, bool TB>
cudaError_t set_attr_all_splits() {
    cudaError_t e = cudaFuncSetAttribute(hclooc_dgemm_tile_kernel<1, TA, TB>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(hclooc_dgemm_tile_kernel<2, TA, TB>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(hclooc_dgemm_tile_kernel<4, TA, TB>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(hclooc_dgemm_tile_kernel<1, TA, TB, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    return e;
}

int ensure_kernel_attr() {
    static int status = -1;
    static std::once_flag once;
    std::call_once(once, [] {
        cudaError_t e = set_attr_all_splits<false, false>();
        if (e == cudaSuccess) e = set_attr_all_splits<true, false>();
        if (e == cudaSuccess) e = set_attr_all_splits<false, true>();
        if (e == cudaSuccess) e = set_attr_all_splits<true, true>();
        status = (e == cudaSuccess) ? 0 : cuda_fail(e);
    });
    return status;
}

template <int KSPLIT, bool TA, bool TB>
cudaError_t launch_split(unsigned tiles, cudaStream_t stream, const CUtensorMap& tmA, const CUtensorMap& tmB, double* dC,
                         long long ldc, int M, int N, int K, double alpha, double beta, int tm, int tn, int tri, int doff) {
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
    return cudaLaunchKernelEx(&cfg, hclooc_dgemm_tile_kernel<KSPLIT, TA, TB>, tmA, tmB, dC, ldc, M, N, K, alpha, beta, tm, tn, tri, doff, 0, 0, 0);
}

template <bool TA, bool TB>
cudaError_t launch_any_split(int ksplit, unsigned tiles, cudaStream_t stream, const CUtensorMap& tmA, const CUtensorMap& tmB, double* dC,
                             long long ldc, int M, int N, int K, double alpha, double beta, int tm, int tn, int tri, int doff,
                             int opmask = 0, int adoff = 0, int bdoff = 0) {
    if (opmask) {      // a triangular operand: one CTA per tile, each over its own k range
        hclooc_dgemm_tile_kernel<1, TA, TB, true><<<tiles, NUM_THREADS, SMEM_BYTES, stream>>>(tmA, tmB, dC, ldc, M, N, K, alpha, beta, tm, tn, tri, doff, opmask, adoff, bdoff);
        return cudaGetLastError();
    }
    if (ksplit >= 4) return launch_split<4, TA, TB>(tiles, stream, tmA, tmB, dC, ldc, M, N, K, alpha, beta, tm, tn, tri, doff);
    if (ksplit >= 2) return launch_split<2, TA, TB>(tiles, stream, tmA, tmB, dC, ldc, M, N, K, alpha, beta, tm, tn, tri, doff);
    hclooc_dgemm_tile_kernel<1, TA, TB><<<tiles, NUM_THREADS, SMEM_BYTES, stream>>>(tmA, tmB, dC, ldc, M, N, K, alpha, beta, tm, tn, tri, doff);
    return cudaGetLastError();
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
                       int ksplit, void* streamk_scratch, int transa, int transb, int tri, int doff, int opmask, int adoff, int bdoff) {
    if (M == 0 || N == 0) return HCLOOC_OK;
    if (alpha == 0.0) K = 0;                       // A and B are not referenced (BLAS convention)
    int rc = ensure_kernel_attr();
    if (rc) return rc;
    CUtensorMap tmA, tmB;
    if (K > 0) {
        if ((rc = transa ? make_map(&tmA, dA, K, M, lda, BK) : make_map(&tmA, dA, M, K, lda, BM))) return rc;
        if ((rc = transb ? make_map(&tmB, dB, N, K, ldb, BN) : make_map(&tmB, dB, K, N, ldb, BK))) return rc;
    } else {
        memset(&tmA, 0, sizeof(tmA));
        memset(&tmB, 0, sizeof(tmB));
        transa = transb = 0;
    }
    const int64_t tm = (M + BM - 1) / BM, tn = (N + BN - 1) / BN;
    if (tm * tn > 0x7fffffffLL || M > 0x7fffffffLL || N > 0x7fffffffLL || K > 0x7fffffffLL) return HCLOOC_ERR_INTERNAL;
    static const bool no_streamk = getenv("HCLOOC_NO_STREAMK") != nullptr;   // experiment knob
    if (tri != 0 && (doff > 0x3fffffff || doff < -0x3fffffff)) return HCLOOC_ERR_INTERNAL;
    if (ksplit < 0 && tri != 0) ksplit = 0;                    // the persistent kernel has no triangle mask
    if (K == 0) opmask = 0;
    if (opmask) {
        ksplit = 1;
        if (adoff > 0x3fffffff || adoff < -0x3fffffff || bdoff > 0x3fffffff || bdoff < -0x3fffffff) return HCLOOC_ERR_INTERNAL;
    }
    if (ksplit < 0 && K > 0 && !no_streamk) {
        // A launch that has the GPU to itself.  One CTA per tile runs its main loop ~1 % faster than the persistent
        // kernel (measured 0.981 against 0.969 of peak on whole waves) but leaves the last wave partly empty, so
        // the persistent stream-K kernel is used unless the tiles fill their waves to 98.8 % or better.  A caller
        // that passes its own scratch (a pipeline step planned as stream-K) always gets it.
        const int64_t T = tm * tn, waves = (T + 147) / 148;
        const bool whole_waves = (double)T >= 0.988 * (double)(waves * 148);
        if (streamk_scratch || !whole_waves) {
            rc = launch_dgemm_streamk(M, N, K, alpha, tmA, tmB, beta, dC, ldc, stream, streamk_scratch, transa, transb);
            if (rc != 1) return rc;
        }
    }
    if (ksplit <= 0) ksplit = dgemm_auto_ksplit(tm * tn, K);
    if (K == 0) ksplit = 1;
    const unsigned tiles = (unsigned)(tm * tn);
    cudaError_t e;
    if (transa && transb) e = launch_any_split<true, true>(ksplit, tiles, stream, tmA, tmB, dC, (long long)ldc, (int)M, (int)N, (int)K, alpha, beta, (int)tm, (int)tn, tri, doff, opmask, adoff, bdoff);
    else if (transa) e = launch_any_split<true, false>(ksplit, tiles, stream, tmA, tmB, dC, (long long)ldc, (int)M, (int)N, (int)K, alpha, beta, (int)tm, (int)tn, tri, doff, opmask, adoff, bdoff);
    else if (transb) e = launch_any_split<false, true>(ksplit, tiles, stream, tmA, tmB, dC, (long long)ldc, (int)M, (int)N, (int)K, alpha, beta, (int)tm, (int)tn, tri, doff, opmask, adoff, bdoff);
    else e = launch_any_split<false, false>(ksplit, tiles, stream, tmA, tmB, dC, (long long)ldc, (int)M, (int)N, (int)K, alpha, beta, (int)tm, (int)tn, tri, doff, opmask, adoff, bdoff);
    if (e != cudaSuccess) return cuda_fail(e);
    return HCLOOC_OK;
}

}  // namespace hclooc
