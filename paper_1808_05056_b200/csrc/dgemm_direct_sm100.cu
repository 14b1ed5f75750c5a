// dgemm_direct_sm100.cu -- the kernel of the DIRECT mode (plan.direct): C = alpha*A*B + beta*C with A, B and C in mapped
// pinned HOST memory, no device buffer.  Every byte a tile needs crosses the host link inside a TMA load, so the tiles
// of a thread-block CLUSTER share them: a cluster of CM x CN CTAs computes CM x CN neighbouring tiles; the A panel of a
// tile row is needed by the CN CTAs of that row, the B panel of a tile column by the CM CTAs of that column.  Each CTA
// loads 1/CN of its row's A stage and 1/CM of its column's B stage and MULTICASTS them (cp.async.bulk.tensor ...
// .multicast::cluster) into the shared memory of the whole row / column, so A is read over the link ceil(tiles_n/CN)
// times and B ceil(tiles_m/CM) times instead of tiles_n and tiles_m times -- once each for BASELINE config 1
// (4 x 4 tiles in one 16-CTA cluster: the compulsory traffic).
//
// Same tile geometry, fragment layout, DMMA loop and epilogue as the tile kernel (dgemm_device.cuh): same bits.
// What differs is the barrier protocol: a stage of CTA X is written by every CTA of X's row and column, so the consumer
// warps of X release a stage by arriving on the `empty` barrier of each of those CTAs (remote mbarrier arrive), and a
// producer refills a stage only when all CTAs it writes to have released it.  Nobody exits before the cluster is done.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <mutex>
#include <cstring>
#include "internal.h"
#include "dgemm_device.cuh"

namespace hclooc {

namespace {

using namespace dev;

__device__ __forceinline__ void tma_load_2d_multicast(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar, uint16_t mask) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1, {%2, %3}], [%4], %5;"
        ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar), "h"(mask) : "memory");
}
__device__ __forceinline__ void mbar_arrive_remote(uint32_t local_bar, uint32_t rank) {
    uint32_t remote;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(local_bar), "r"(rank));
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(remote) : "memory");
}
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP_C:\n"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_C;\n"
        "bra WAIT_LOOP_C;\n"
        "DONE_C:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}

template <int CM, int CN>
__global__ void __launch_bounds__(NUM_THREADS, 1)
hclooc_dgemm_direct_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                           double* __restrict__ C, long long ldc, int M, int N, int K,
                           double alpha, double beta, int ctiles_n) {
    constexpr int CSIZE = CM * CN;
    constexpr int A_ROWS = BM / CN;                       // rows of the A stage this CTA loads for its row
    constexpr int B_BOXES = (BN / 16) / CM;               // 16-column boxes of the B stage this CTA loads for its column
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_base = smem_base + STAGES * STAGE_BYTES;
    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const uint32_t crank = (CSIZE == 1) ? 0u : cluster_ctarank();
    const int cr_m = (int)crank / CN, cr_n = (int)crank % CN;
    const int cluster_id = (int)blockIdx.x / CSIZE;
    const int tile_m = (cluster_id / ctiles_n) * CM + cr_m, tile_n = (cluster_id % ctiles_n) * CN + cr_n;
    const int m0 = tile_m * BM, n0 = tile_n * BN;         // may lie outside C (cluster padding): loads zero fill, nothing stored
    const int num_kb = (K + BK - 1) / BK;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(bar_base + 8 * s, 1);
            mbar_init(bar_base + 8 * (STAGES + s), NUM_CONSUMER_WARPS * (CM + CN - 1));
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    cluster_sync_all();                                   // every barrier of the cluster exists before anyone signals it

    if (warp >= NUM_CONSUMER_WARPS) {
        regs_release_producer();
        if (warp == NUM_CONSUMER_WARPS && lane == 0 && num_kb > 0) {
            asm volatile("prefetch.tensormap [%0];" ::"l"(&tmA) : "memory");
            asm volatile("prefetch.tensormap [%0];" ::"l"(&tmB) : "memory");
            uint16_t row_mask = 0, col_mask = 0;
            #pragma unroll
            for (int j = 0; j < CN; ++j) row_mask |= (uint16_t)(1u << (cr_m * CN + j));
            #pragma unroll
            for (int i = 0; i < CM; ++i) col_mask |= (uint16_t)(1u << (i * CN + cr_n));
            int stage = 0;
            uint32_t phase = 0;
            for (int kb = 0; kb < num_kb; ++kb) {
                const uint32_t full = bar_base + 8 * stage;
                mbar_wait_cluster(bar_base + 8 * (STAGES + stage), phase ^ 1u);      // my row and column released the stage
                mbar_expect_tx(full, STAGE_BYTES);
                const uint32_t sa = smem_base + stage * STAGE_BYTES;
                const uint32_t sb = sa + A_STAGE_BYTES;
                const int k0 = kb * BK;
                #pragma unroll
                for (int hk = 0; hk < BK / 16; ++hk) {
                    const uint32_t dst = sa + hk * A_HALF_BYTES + cr_n * A_ROWS * 128;
                    if (CN == 1) tma_load_2d(dst, &tmA, k0 + 16 * hk, m0, full);
                    else tma_load_2d_multicast(dst, &tmA, k0 + 16 * hk, m0 + cr_n * A_ROWS, full, row_mask);
                }
                #pragma unroll
                for (int q = 0; q < B_BOXES; ++q) {
                    const int b = cr_m * B_BOXES + q;
                    if (CM == 1) tma_load_2d(sb + b * B_BOX_BYTES, &tmB, n0 + 16 * b, k0, full);
                    else tma_load_2d_multicast(sb + b * B_BOX_BYTES, &tmB, n0 + 16 * b, k0, full, col_mask);
                }
                if (++stage == STAGES) { stage = 0; phase ^= 1u; }
            }
        }
        __syncwarp();
        cluster_sync_all();                               // peers may still write my stages / signal my barriers until here
        return;
    }

    regs_take_consumer();
    FragLanes f;
    f.init(warp, lane);
    double acc[4][4][2][2];
    #pragma unroll
    for (int u = 0; u < 4; ++u)
        #pragma unroll
        for (int bx = 0; bx < 4; ++bx)
            #pragma unroll
            for (int v = 0; v < 2; ++v) { acc[u][bx][v][0] = 0.0; acc[u][bx][v][1] = 0.0; }
    {
        // CTAs that write into my stages: my row (A parts) and my column (B parts); lane l < CM + CN - 1 signals one of them
        uint32_t target = crank;
        if (lane < CN) target = (uint32_t)(cr_m * CN + lane);
        else if (lane < CN + CM - 1) { const int i = lane - CN; target = (uint32_t)((i < cr_m ? i : i + 1) * CN + cr_n); }
        int stage = 0;
        uint32_t phase = 0;
        const int nu = edge_groups(M, m0 + f.wm * 32, 8), nbx = edge_groups(N, n0 + f.wn * 64, 16);
        const bool work = (nu != 0 && nbx != 0);
        for (int kb = 0; kb < num_kb; ++kb) {
            mbar_wait(bar_base + 8 * stage, phase);
            if (work) mma_kblock(acc, smem_base + stage * STAGE_BYTES, f);
            __syncwarp();
            if (lane < CM + CN - 1) mbar_arrive_remote(bar_base + 8 * (STAGES + stage), target);
            if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
    }
    epilogue_store(acc, C, ldc, M, N, m0, n0, alpha, beta, f);
    __syncwarp();
    cluster_sync_all();
}

template <int CM, int CN>
int launch_cluster(int64_t M, int64_t N, int64_t K, double alpha, const double* A, int64_t lda, const double* B, int64_t ldb,
                   double beta, double* C, int64_t ldc, cudaStream_t stream, bool probe_only) {
    static int attr_status = -1;
    static std::once_flag once;
    std::call_once(once, [] {
        cudaError_t e = cudaFuncSetAttribute(hclooc_dgemm_direct_kernel<CM, CN>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
        if (e == cudaSuccess && CM * CN > 8)
            e = cudaFuncSetAttribute(hclooc_dgemm_direct_kernel<CM, CN>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        attr_status = (e == cudaSuccess) ? 0 : cuda_fail(e);
    });
    if (attr_status) return attr_status;
    const int64_t tm = (M + BM - 1) / BM, tn = (N + BN - 1) / BN;
    const int64_t ctm = (tm + CM - 1) / CM, ctn = (tn + CN - 1) / CN;
    if (ctm * ctn * CM * CN > 0x7fffffffLL) return HCLOOC_ERR_INTERNAL;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(ctm * ctn * CM * CN), 1, 1);
    cfg.blockDim = dim3(NUM_THREADS, 1, 1);
    cfg.dynamicSmemBytes = SMEM_BYTES;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CM * CN;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (probe_only) {
        int n = 0;
        cudaError_t e = cudaOccupancyMaxActiveClusters(&n, hclooc_dgemm_direct_kernel<CM, CN>, &cfg);
        if (e != cudaSuccess) { cudaGetLastError(); return 1; }
        return n > 0 ? HCLOOC_OK : 1;
    }
    CUtensorMap tmA, tmB;
    int rc;
    if ((rc = make_tensor_map(&tmA, A, M, K, lda, BM / CN))) return rc;
    if ((rc = make_tensor_map(&tmB, B, K, N, ldb, BK))) return rc;
    cudaError_t e = cudaLaunchKernelEx(&cfg, hclooc_dgemm_direct_kernel<CM, CN>, tmA, tmB, C, (long long)ldc, (int)M, (int)N, (int)K,
                                       alpha, beta, (int)ctn);
    if (e != cudaSuccess) return cuda_fail(e);
    return HCLOOC_OK;
}

}  // namespace

// Cluster shape of a direct-mode launch: as many tiles of a row / column share their loads as there are, up to 4 x 4
// (16 CTAs: the non-portable cluster size of sm_100; `max_cluster` = 8 caps it at 2 x 4).  Pure arithmetic: the planner
// counts the traffic with it and the launch uses it.
void direct_cluster_shape(int64_t M, int64_t N, int max_cluster, int* cm, int* cn) {
    const int64_t tm = (M + BM - 1) / BM, tn = (N + BN - 1) / BN;
    int n = tn >= 3 ? 4 : (tn == 2 ? 2 : 1);
    int m = tm >= 3 ? 4 : (tm == 2 ? 2 : 1);
    if (m * n > max_cluster) m = (max_cluster / n) < 1 ? 1 : (max_cluster / n >= 4 ? 4 : (max_cluster / n >= 2 ? 2 : 1));
    *cm = m; *cn = n;
}

int direct_max_cluster() {
    static int value = 0;
    static std::once_flag once;
    std::call_once(once, [] {
        value = (launch_cluster<4, 4>(128 * 4, 128 * 4, 32, 1.0, nullptr, 32, nullptr, 512, 0.0, nullptr, 512, nullptr, true) == HCLOOC_OK) ? 16 : 8;
    });
    return value;
}

// C = alpha*A*B + beta*C on pointers the device can address (mapped pinned host memory), K > 0.
int launch_dgemm_direct(int64_t M, int64_t N, int64_t K, double alpha, const double* A, int64_t lda, const double* B, int64_t ldb,
                        double beta, double* C, int64_t ldc, cudaStream_t stream, int cm, int cn) {
    if (M == 0 || N == 0) return HCLOOC_OK;
    if (M > 0x7fffffffLL || N > 0x7fffffffLL || K > 0x7fffffffLL || K <= 0) return HCLOOC_ERR_INTERNAL;
#define HCL_DIRECT_CASE(a, b) if (cm == a && cn == b) return launch_cluster<a, b>(M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, stream, false)
    HCL_DIRECT_CASE(1, 1); HCL_DIRECT_CASE(1, 2); HCL_DIRECT_CASE(1, 4);
    HCL_DIRECT_CASE(2, 1); HCL_DIRECT_CASE(2, 2); HCL_DIRECT_CASE(2, 4);
    HCL_DIRECT_CASE(4, 1); HCL_DIRECT_CASE(4, 2); HCL_DIRECT_CASE(4, 4);
#undef HCL_DIRECT_CASE
    return HCLOOC_ERR_INTERNAL;
}

}  // namespace hclooc
