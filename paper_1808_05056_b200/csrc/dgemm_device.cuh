// dgemm_device.cuh -- device-side building blocks shared by the two S5 kernels (dgemm_sm100.cu: one tile or one
// cluster per tile; dgemm_streamk_sm100.cu: persistent stream-K): tile geometry, mbarrier/TMA/DMMA wrappers,
// the permuted fragment layout and the fused alpha/beta epilogue.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace hclooc {
namespace dev {

constexpr int BM = 128;
constexpr int BN = 128;
constexpr int BK = 32;                              // k depth of a stage: two 128-byte k halves of A, 32 k-rows of B
constexpr int STAGES = 3;
constexpr int A_HALF_BYTES = BM * 16 * 8;           // 16 KiB: one TMA box of A, 128 rows x 128 B (16 k)
constexpr int A_STAGE_BYTES = (BK / 16) * A_HALF_BYTES;
constexpr int B_BOX_BYTES = BK * 16 * 8;            // 4 KiB: one TMA box of B, 32 k-rows x 128 B (16 columns)
constexpr int B_STAGE_BYTES = (BN / 16) * B_BOX_BYTES;
constexpr int STAGE_BYTES = A_STAGE_BYTES + B_STAGE_BYTES;
constexpr int NUM_CONSUMER_WARPS = 8;
// Two consumer warpgroups + one producer warpgroup of which only warp 0 works.  The register file is split per
// SM sub-partition (16384 registers for its 3 warps), so a flat allocation caps every thread at 168 registers
// and the 128 accumulator registers of a consumer leave too little for the loop state: the producer warpgroup
// gives its registers back (setmaxnreg.dec) and the consumers take them (setmaxnreg.inc).
constexpr int NUM_PRODUCER_WARPS = 4;
constexpr int NUM_THREADS = (NUM_CONSUMER_WARPS + NUM_PRODUCER_WARPS) * 32;
constexpr int PRODUCER_REGS = 40;
constexpr int CONSUMER_REGS = 232;
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

__device__ __forceinline__ void regs_release_producer() {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(PRODUCER_REGS));
}
__device__ __forceinline__ void regs_take_consumer() {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(CONSUMER_REGS));
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


// Tile rasterisation: groups of RASTER_GROUP m-tiles, m fastest inside a group, so CTAs that run together share
// B column panels and a bounded set of A row panels in L2.
__device__ __forceinline__ void tile_coords(int tile, int tiles_m, int tiles_n, int& tile_m, int& tile_n) {
    const int per_group = RASTER_GROUP * tiles_n;
    const int grp = tile / per_group;
    const int rem = tile - grp * per_group;
    const int gm0 = grp * RASTER_GROUP;
    const int gsz = min(RASTER_GROUP, tiles_m - gm0);
    tile_m = gm0 + rem % gsz;
    tile_n = rem / gsz;
}

// Per-lane shared-memory byte offsets of the DMMA fragments inside a stage.  Inside a tile the 8 rows of an
// m-tile, the 4 k indices of a k-step and the 8 columns of an n-tile are permuted (row g <-> 4(g&1)+(g>>1),
// k index t <-> 2t+e, columns interleaved in pairs) so that with the 128-byte swizzle every LDS.128 of a
// quarter warp hits distinct banks and feeds two DMMAs.
//
// Transposed operands (hclooc_dgemm_t) change only how a stage is laid out and read, never the DMMA loop:
//   operand stored with k contiguous   (A, or B^T = stored N x K): two 16-k halves of 128 rows x 128 B; one LDS.128 of
//        lane (g, t) at row 8*tile + rp(g), chunk t gives k = 2t and 2t+1 of that row -> the operands of k-steps e = 0, 1;
//   operand stored with k as the row   (B, or A^T = stored K x M): eight boxes of 32 k-rows x 16 columns; one LDS.128 at
//        k-row 2t+e, chunk g gives columns 2g and 2g+1 -> the operands of two m- (or n-) tiles of k-step e.
// Which row (column) of C a DMMA tile's index g stands for follows from that and is undone in the epilogue:
//   A as stored M x K : row = 8u + rp(g)                      A^T (stored K x M): row = 16(u>>1) + 2g + (u&1)
//   B as stored K x N : col = 16bx + 2c' + v  (c' = DMMA col)  B^T (stored N x K): col = 8(2bx+v) + rp(c')
template <bool TA, bool TB>
struct FragLanesT {
    uint32_t a_lane, a_lane_t[2], b_lane[2], b_lane_t;
    int rp, t, g, wm, wn;
    __device__ __forceinline__ void init(int warp, int lane) {
        g = lane >> 2;
        t = lane & 3;
        rp = 4 * (g & 1) + (g >> 1);
        wm = warp & 3;
        wn = warp >> 2;
        a_lane = (uint32_t)((wm * 32 + rp) * 128 + ((t ^ rp) << 4));
        b_lane_t = (uint32_t)(A_STAGE_BYTES + (wn * 64 + rp) * 128 + ((t ^ rp) << 4));
        #pragma unroll
        for (int e = 0; e < 2; ++e) {
            b_lane[e] = (uint32_t)(A_STAGE_BYTES + wn * 4 * B_BOX_BYTES + (2 * t + e) * 128 + ((g ^ (2 * t + e)) << 4));
            a_lane_t[e] = (uint32_t)(wm * 2 * B_BOX_BYTES + (2 * t + e) * 128 + ((g ^ (2 * t + e)) << 4));
        }
    }
    // row of C (inside the CTA tile) that accumulator group u of this lane belongs to
    __device__ __forceinline__ int row_of(int u) const {
        return TA ? wm * 32 + (u >> 1) * 16 + 2 * g + (u & 1) : wm * 32 + u * 8 + rp;
    }
};
using FragLanes = FragLanesT<false, false>;

// One k block (BK deep) of the 32 x 64 warp tile: per group of 8 k, 12 LDS.128 feed 64 DMMA.8x8x4.
// MASK (hclooc_dtrmm, hclooc_dsymm: an operand that is a triangle of a stored matrix whose other triangle must not count): the
// fragments of the k blocks that cross the diagonal are zeroed where they fall outside the triangle --
//   am = 1: op(A)[r][k] counts iff k <= r + da,   am = 2: iff k >= r + da          (r, k: indices inside the tile / k block)
//   bm = 1: op(B)[k][c] counts iff c <= k + db,   bm = 2: iff c >= k + db
// -- by a select, never by a product (the other triangle may hold NaN).  Index maps: a[u][e] is row f.row_of(u), k = 8kg + 2t + e;
// b[bx][v] (k-step e) is column 16bx + 2g + v (B as stored) or 8(2bx + v) + rp (B^T) of the warp's 64, same k.
__device__ __forceinline__ bool mask_keep(int m, int major, int minor, int d) {      // m = 1: minor <= major + d, m = 2: minor >= major + d
    return m == 1 ? minor <= major + d : minor >= major + d;
}
template <bool TA, bool TB, bool MASK = false>
__device__ __forceinline__ void mma_kblock(double (&acc)[4][4][2][2], uint32_t sbase, const FragLanesT<TA, TB>& f,
                                           int am = 0, int da = 0, int bm = 0, int db = 0) {
    #pragma unroll
    for (int kg = 0; kg < BK / 8; ++kg) {
        double a[4][2];
        if (!TA) {
            const uint32_t abase = sbase + (kg >> 1) * A_HALF_BYTES + (f.a_lane ^ ((kg & 1) << 6));
            #pragma unroll
            for (int u = 0; u < 4; ++u) lds128(a[u][0], a[u][1], abase + u * 1024);
        } else {
            #pragma unroll
            for (int e = 0; e < 2; ++e)
                #pragma unroll
                for (int ub = 0; ub < 2; ++ub)
                    lds128(a[2 * ub][e], a[2 * ub + 1][e], sbase + f.a_lane_t[e] + kg * 1024 + ub * B_BOX_BYTES);
        }
        if (MASK && am) {
            #pragma unroll
            for (int u = 0; u < 4; ++u)
                #pragma unroll
                for (int e = 0; e < 2; ++e)
                    if (!mask_keep(am, f.row_of(u), kg * 8 + 2 * f.t + e, da)) a[u][e] = 0.0;
        }
        if (!TB) {
            #pragma unroll
            for (int e = 0; e < 2; ++e) {
                double b[4][2];
                #pragma unroll
                for (int bx = 0; bx < 4; ++bx)
                    lds128(b[bx][0], b[bx][1], sbase + f.b_lane[e] + kg * 1024 + bx * B_BOX_BYTES);
                if (MASK && bm) {
                    #pragma unroll
                    for (int bx = 0; bx < 4; ++bx)
                        #pragma unroll
                        for (int v = 0; v < 2; ++v)
                            if (!mask_keep(bm, kg * 8 + 2 * f.t + e, f.wn * 64 + 16 * bx + 2 * f.g + v, db)) b[bx][v] = 0.0;
                }
                #pragma unroll
                for (int u = 0; u < 4; ++u)
                    #pragma unroll
                    for (int bx = 0; bx < 4; ++bx) {
                        dmma(acc[u][bx][0], a[u][e], b[bx][0]);
                        dmma(acc[u][bx][1], a[u][e], b[bx][1]);
                    }
            }
        } else {
            const uint32_t bbase = sbase + (kg >> 1) * A_HALF_BYTES + (f.b_lane_t ^ ((kg & 1) << 6));
            #pragma unroll
            for (int half = 0; half < 2; ++half) {       // n-tiles j = 2bx + v, four at a time: both k-steps from one LDS.128
                double b[2][2][2];                        // [bx in half][v][e]
                #pragma unroll
                for (int q = 0; q < 4; ++q) lds128(b[q >> 1][q & 1][0], b[q >> 1][q & 1][1], bbase + (half * 4 + q) * 1024);
                if (MASK && bm) {
                    #pragma unroll
                    for (int q = 0; q < 4; ++q)
                        #pragma unroll
                        for (int e = 0; e < 2; ++e)
                            if (!mask_keep(bm, kg * 8 + 2 * f.t + e, f.wn * 64 + 8 * (half * 4 + q) + f.rp, db)) b[q >> 1][q & 1][e] = 0.0;
                }
                #pragma unroll
                for (int e = 0; e < 2; ++e)
                    #pragma unroll
                    for (int u = 0; u < 4; ++u)
                        #pragma unroll
                        for (int bq = 0; bq < 2; ++bq) {
                            dmma(acc[u][half * 2 + bq][0], a[u][e], b[bq][0][e]);
                            dmma(acc[u][half * 2 + bq][1], a[u][e], b[bq][1][e]);
                        }
            }
        }
    }
}

// How many 8-row groups / 16-column boxes of this warp's 32 x 64 tile lie inside the matrix (0..4 each).  A warp
// whose part of an edge tile is entirely zero fill skips its DMMAs (nobody reads those products).
__device__ __forceinline__ int edge_groups(int extent, int origin, int unit) {
    const int left = extent - origin;
    return left <= 0 ? 0 : (left >= 4 * unit ? 4 : (left + unit - 1) / unit);
}

// alpha*acc + beta*c with the rounding sequence of the definition (oracle: two products and one sum, each
// rounded): spelled with intrinsics so that no variant of the epilogue is contracted into an FMA differently from another.
__device__ __forceinline__ double axpby_tail(double alpha_acc, double beta, double c) {
    return __dadd_rn(alpha_acc, __dmul_rn(beta, c));
}

// Fused epilogue: C = alpha*acc + beta*C straight from registers; C is not read when beta == 0.
// tri != 0 (hclooc_dsyrk): only one triangle of C is referenced -- element (row, col) of this launch's C is stored iff
// col <= row + doff (tri == 1, lower) or col >= row + doff (tri == 2, upper); doff places the launch's block on the diagonal.
__device__ __forceinline__ bool tri_keep(int tri, int doff, int row, int col) {
    return tri == 0 || (tri == 1 ? col <= row + doff : col >= row + doff);
}

template <bool TA, bool TB>
__device__ __forceinline__ void epilogue_store(const double (&acc)[4][4][2][2], double* __restrict__ C, long long ldc,
                                               int M, int N, int m0, int n0, double alpha, double beta, const FragLanesT<TA, TB>& f,
                                               int tri = 0, int doff = 0) {
    const bool read_c = (beta != 0.0);
    const bool vec_ok = ((ldc & 1LL) == 0) && ((reinterpret_cast<uintptr_t>(C) & 15u) == 0);
    // 256-bit accesses (sm_100: LDG/STG.256): a lane's 4 consecutive columns are one 32-byte sector, a quarter warp's
    // 16 columns one 128-byte line -- what the host link wants when C lives in host memory (direct mode): 16-byte
    // stores into lines that were not read first (beta == 0) crossed the link at ~14 GB/s
    const bool vec4_ok = ((ldc & 3LL) == 0) && ((reinterpret_cast<uintptr_t>(C) & 31u) == 0);
    #pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int row = m0 + f.row_of(u);
        if (row >= M) continue;
        double* crow = C + (long long)row * ldc;
        // The common case -- C is read, 32-byte accesses are legal, no triangle mask, the lane's four segments of this row lie
        // inside C: the four loads of the row are issued back to back BEFORE the first use, so a lane makes 4 round trips to C
        // instead of 16 (what matters when C is host memory: direct mode spent a third of config 1 in these dependent reads).
        if (!TB && read_c && vec4_ok && tri == 0 && n0 + f.wn * 64 + 63 < N) {
            double c[4][4];
            #pragma unroll
            for (int bx = 0; bx < 4; ++bx) {
                const double* p = crow + n0 + f.wn * 64 + bx * 16 + 4 * f.t;
                asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(c[bx][0]), "=d"(c[bx][1]), "=d"(c[bx][2]), "=d"(c[bx][3]) : "l"(p));
            }
            #pragma unroll
            for (int bx = 0; bx < 4; ++bx) {
                double* p = crow + n0 + f.wn * 64 + bx * 16 + 4 * f.t;
                const double x0 = axpby_tail(__dmul_rn(alpha, acc[u][bx][0][0]), beta, c[bx][0]), x1 = axpby_tail(__dmul_rn(alpha, acc[u][bx][1][0]), beta, c[bx][1]);
                const double x2 = axpby_tail(__dmul_rn(alpha, acc[u][bx][0][1]), beta, c[bx][2]), x3 = axpby_tail(__dmul_rn(alpha, acc[u][bx][1][1]), beta, c[bx][3]);
                asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(x0), "d"(x1), "d"(x2), "d"(x3) : "memory");
            }
            continue;
        }
        #pragma unroll
        for (int bx = 0; bx < 4; ++bx) {
            if (!TB) {
                const int col = n0 + f.wn * 64 + bx * 16 + 4 * f.t;
                // lane holds 4 consecutive columns: (v=0,c0) (v=1,c0) (v=0,c1) (v=1,c1)
                double x0 = __dmul_rn(alpha, acc[u][bx][0][0]), x1 = __dmul_rn(alpha, acc[u][bx][1][0]);
                double x2 = __dmul_rn(alpha, acc[u][bx][0][1]), x3 = __dmul_rn(alpha, acc[u][bx][1][1]);
                const bool keep_lo = tri_keep(tri, doff, row, col), keep_hi = tri_keep(tri, doff, row, col + 3);
                if (!keep_lo && !keep_hi) continue;                      // the four columns lie in the other triangle
                const bool keep_all = keep_lo && keep_hi;
                if (!keep_all) {
                    const double xs[4] = {x0, x1, x2, x3};
                    #pragma unroll
                    for (int q = 0; q < 4; ++q)
                        if (col + q < N && tri_keep(tri, doff, row, col + q)) crow[col + q] = read_c ? axpby_tail(xs[q], beta, crow[col + q]) : xs[q];
                } else if (col + 3 < N && vec4_ok) {
                    double* p = crow + col;
                    if (read_c) {
                        double c0, c1, c2, c3;
                        asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(c0), "=d"(c1), "=d"(c2), "=d"(c3) : "l"(p) : "memory");
                        x0 = axpby_tail(x0, beta, c0); x1 = axpby_tail(x1, beta, c1);
                        x2 = axpby_tail(x2, beta, c2); x3 = axpby_tail(x3, beta, c3);
                    }
                    asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(x0), "d"(x1), "d"(x2), "d"(x3) : "memory");
                } else if (col + 3 < N && vec_ok) {
                    double2* p = reinterpret_cast<double2*>(crow + col);
                    if (read_c) {
                        const double2 c01 = p[0], c23 = p[1];
                        x0 = axpby_tail(x0, beta, c01.x); x1 = axpby_tail(x1, beta, c01.y);
                        x2 = axpby_tail(x2, beta, c23.x); x3 = axpby_tail(x3, beta, c23.y);
                    }
                    p[0] = make_double2(x0, x1);
                    p[1] = make_double2(x2, x3);
                } else {
                    const double xs[4] = {x0, x1, x2, x3};
                    #pragma unroll
                    for (int q = 0; q < 4; ++q)
                        if (col + q < N) crow[col + q] = read_c ? axpby_tail(xs[q], beta, crow[col + q]) : xs[q];
                }
            } else {
                // B^T: n-tile j = 2bx + v, DMMA column c' = 2t + c stands for column 8j + rp(c') = 8j + t + 4c
                #pragma unroll
                for (int v = 0; v < 2; ++v)
                    #pragma unroll
                    for (int c = 0; c < 2; ++c) {
                        const int col = n0 + f.wn * 64 + (2 * bx + v) * 8 + f.t + 4 * c;
                        const double x = __dmul_rn(alpha, acc[u][bx][v][c]);
                        if (col < N && tri_keep(tri, doff, row, col)) crow[col] = read_c ? axpby_tail(x, beta, crow[col]) : x;
                    }
            }
        }
    }
}

}  // namespace dev
}  // namespace hclooc
