// getrf_sm100.cu -- the block kernels of the LU factorization with partial pivoting (hclooc_dgetrf / hclDgetrf; PAPER.md:412
// names LU first among the out-of-core factorizations to be built on the DGEMM):
//
//   getrf_panel_kernel   factors ONE tall panel of m rows and w <= 128 columns that sits in device memory.  The flops of an LU
//                        factorization are DGEMM / DTRSM work on the tile kernel; what is left at the bottom of the recursion is
//                        this: per column a pivot search over ALL remaining rows, one row interchange, a division per row and a
//                        rank-1 update of at most 127 columns -- latency, not arithmetic.  So the panel is spread over up to one
//                        CTA per SM (cooperative launch): every CTA keeps its slab of rows in SHARED MEMORY for the whole panel
//                        (one read and one write of the panel in HBM), and a column costs ONE grid-wide barrier: before it every
//                        CTA publishes its best candidate (|value|, row, and the row's contents) and CTA 0 publishes row j; after
//                        it every CTA picks the same winner (largest |value|, smallest row on ties: the FIRST maximum, as IDAMAX
//                        and the oracle), the two CTAs that own row j and the pivot row exchange them from the published copies,
//                        and everybody eliminates in its own slab.
//   row_gather_kernel /  a sequence of row interchanges applied to OTHER columns as one permutation: the host folds the sequence
//   row_scatter_kernel   into (destination <- source) pairs; the rows are gathered into a scratch buffer and scattered back --
//                        two fully parallel passes instead of thousands of dependent row swaps.
#include <algorithm>
#include <cstdlib>
#include "internal.h"

namespace hclooc {
namespace {

constexpr int LU_T = 256;           // threads per CTA
constexpr int LU_W = 128;           // widest panel
constexpr int LU_MAXG = 192;        // most CTAs of a panel launch (>= SMs of the device, checked at launch)

__device__ __forceinline__ double lu_shfl_down(double v, int off) {
    int lo = __double2loint(v), hi = __double2hiint(v);
    lo = __shfl_down_sync(0xffffffffu, lo, off);
    hi = __shfl_down_sync(0xffffffffu, hi, off);
    return __hiloint2double(hi, lo);
}

__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

// candidate order: larger |value| first, smaller row on ties
__device__ __forceinline__ bool lu_better(double v, int r, double bv, int br) { return v > bv || (v == bv && r < br); }

// Global scratch of the panel launches.  TWO sets, used by the columns of even and of odd index: set j & 1 is written before the
// barrier of column j and read right after it; a CTA writes it again only after the barrier of column j+1, at which every CTA has
// arrived -- i.e. has finished those reads.
struct PanelSlots {
    double* cval;                   // [2][G]          best |a_ij| of CTA g in the column (-1: no row of it is still in play)
    int* crow;                      // [2][G]          its row (panel-local)
    double* ccont;                  // [2][G][LU_W]    that row's contents
    double* top;                    // [2][LU_W]       row j before the interchange of column j
    unsigned long long* counter;    // arrivals at the grid barrier, monotone across launches (bar_base = its value at launch)
};

__global__ void __launch_bounds__(LU_T, 1)
getrf_panel_kernel(double* __restrict__ A, long long lda, long long m, int w, int rpc, int G, long long* __restrict__ ipiv_out,
                   long long row_base, long long* __restrict__ info, long long info_base, PanelSlots sl, unsigned long long bar_base) {
    extern __shared__ __align__(16) double S[];     // S[r * SW + c]: this CTA's rows, odd stride (column access hits 32 banks)
    __shared__ double red_v[LU_T / 32];
    __shared__ int red_r[LU_T / 32];
    __shared__ double P_s[LU_W], T_s[LU_W];         // the pivot row / row j as published
    __shared__ int win_cta, win_row;
    const int g = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long r0 = (long long)g * rpc;
    const int nloc = (int)(m - r0 < (long long)rpc ? m - r0 : (long long)rpc);
    const int SW = w | 1;
    for (int r = warp; r < nloc; r += LU_T / 32)
        for (int c = lane; c < w; c += 32) S[r * SW + c] = A[(r0 + r) * lda + c];
    __syncthreads();
    const int nsteps = (int)(m < (long long)w ? m : (long long)w);
    // this thread's candidate for the pivot of the NEXT column: found at the end of a column's elimination, in the rows the thread
    // has just updated (column 0: here)
    double best = -1.0;
    int brow = 0x7fffffff;
    for (int r = tid; r < nloc; r += LU_T) {
        const double v = fabs(S[r * SW]);
        if (v > best) { best = v; brow = (int)(r0 + r); }
    }
    for (int j = 0; j < nsteps; ++j) {
        const int set = j & 1;
        // ---- this CTA's candidate for the pivot of column j
#pragma unroll
        for (int off = 16; off; off >>= 1) {
            const double ov = lu_shfl_down(best, off);
            const int orow = __shfl_down_sync(0xffffffffu, brow, off);
            if (lu_better(ov, orow, best, brow)) { best = ov; brow = orow; }
        }
        if (lane == 0) { red_v[warp] = best; red_r[warp] = brow; }
        __syncthreads();
        best = red_v[0]; brow = red_r[0];
#pragma unroll
        for (int k = 1; k < LU_T / 32; ++k)
            if (lu_better(red_v[k], red_r[k], best, brow)) { best = red_v[k]; brow = red_r[k]; }
        const size_t slot = (size_t)set * G + g;
        if (tid == 0) { sl.cval[slot] = best; sl.crow[slot] = brow; }
        if (tid < w && best >= 0.0) sl.ccont[slot * LU_W + tid] = S[(size_t)(brow - r0) * SW + tid];
        if (g == 0 && tid >= LU_W && tid < LU_W + w) sl.top[set * LU_W + tid - LU_W] = S[j * SW + tid - LU_W];
        // ---- the grid barrier of column j
        __threadfence();
        __syncthreads();
        if (tid == 0) {
            atomicAdd(sl.counter, 1ULL);
            const unsigned long long target = bar_base + (unsigned long long)G * (unsigned long long)(j + 1);
            while (ld_acquire_u64(sl.counter) < target) { }
        }
        __syncthreads();
        // ---- the same winner in every CTA: warp 0 picks it and fetches the two rows that change places
        if (warp == 0) {
            double bv = -2.0;
            int br = 0x7fffffff, bc = -1;
            for (int c = lane; c < G; c += 32) {
                const double v = __ldcg(&sl.cval[(size_t)set * G + c]);
                const int r = __ldcg(&sl.crow[(size_t)set * G + c]);
                if (lu_better(v, r, bv, br)) { bv = v; br = r; bc = c; }
            }
#pragma unroll
            for (int off = 16; off; off >>= 1) {
                const double ov = lu_shfl_down(bv, off);
                const int orow = __shfl_down_sync(0xffffffffu, br, off);
                const int oc = __shfl_down_sync(0xffffffffu, bc, off);
                if (lu_better(ov, orow, bv, br)) { bv = ov; br = orow; bc = oc; }
            }
            if (!(bv >= 0.0)) { br = j; bc = -1; }          // nothing comparable in the column (NaN): no interchange
            br = __shfl_sync(0xffffffffu, br, 0);
            bc = __shfl_sync(0xffffffffu, bc, 0);
            double tv[LU_W / 32], pv[LU_W / 32];          // all loads in flight before the first use: one L2 round trip, not four
#pragma unroll
            for (int i = 0; i < LU_W / 32; ++i) {
                const int c = lane + 32 * i;
                tv[i] = c < w ? __ldcg(&sl.top[set * LU_W + c]) : 0.0;
                pv[i] = c < w && bc >= 0 ? __ldcg(&sl.ccont[((size_t)set * G + bc) * LU_W + c]) : 0.0;
            }
#pragma unroll
            for (int i = 0; i < LU_W / 32; ++i) {
                const int c = lane + 32 * i;
                if (c < w) { T_s[c] = tv[i]; P_s[c] = bc < 0 ? tv[i] : pv[i]; }
            }
            if (lane == 0) { win_cta = bc; win_row = br; }
        }
        __syncthreads();
        const int wc = win_cta, pr = win_row;
        const double pivot = P_s[j];
        if (pr != j) {                               // rows j and pr change places, each owner taking the other's published copy
            if (g == wc && tid < w) S[(size_t)(pr - r0) * SW + tid] = T_s[tid];
            if (g == 0 && tid >= LU_W && tid < LU_W + w) S[j * SW + tid - LU_W] = P_s[tid - LU_W];
        }
        if (g == 0 && tid == 0) {
            ipiv_out[j] = row_base + pr;
            if (pivot == 0.0) atomicCAS((unsigned long long*)info, 0ULL, (unsigned long long)(info_base + j + 1));
        }
        __syncthreads();
        // ---- elimination, one thread per row: the multiplier (IEEE division, as the definition) stays in a register, then the
        // row's columns past j one after the other -- the lanes of a warp walk 32 consecutive rows (odd stride: no bank conflict),
        // the pivot row's element is a broadcast, and the iterations of a thread are independent, so the loads run ahead of the
        // arithmetic.  A zero pivot: the column is zero from row j down, nothing to eliminate.  The thread then looks at its rows'
        // entries in column j+1, which it has just written: its candidate for the next pivot (no barrier needed until the CTA
        // reduction at the top of the loop, which also orders these writes before anybody else's reads).
        best = -1.0;
        brow = 0x7fffffff;
        for (int r = tid; r < nloc; r += LU_T) {
            if (r0 + r > j) {
                double* __restrict__ row = S + (size_t)r * SW;
                if (pivot != 0.0) {
                    const double l = row[j] / pivot;
                    row[j] = l;
#pragma unroll 8
                    for (int c = j + 1; c < w; ++c) row[c] = __dsub_rn(row[c], __dmul_rn(l, P_s[c]));
                }
                if (j + 1 < nsteps) {
                    const double v = fabs(row[j + 1]);
                    if (v > best) { best = v; brow = (int)(r0 + r); }
                }
            }
        }
    }
    __syncthreads();
    for (int r = warp; r < nloc; r += LU_T / 32)
        for (int c = lane; c < w; c += 32) A[(r0 + r) * lda + c] = S[r * SW + c];
}

// rows on grid.x (as many as a permutation touches), 256 columns per CTA on grid.y
__global__ void __launch_bounds__(256)
row_gather_kernel(const double* __restrict__ X, long long ld, int ncols, const int* __restrict__ src, double* __restrict__ tmp, long long ldt) {
    __shared__ int s;
    if (threadIdx.x == 0) s = src[blockIdx.x];
    __syncthreads();
    const int c = blockIdx.y * 256 + threadIdx.x;
    if (c < ncols) tmp[(long long)blockIdx.x * ldt + c] = X[(long long)s * ld + c];
}

__global__ void __launch_bounds__(256)
row_scatter_kernel(double* __restrict__ X, long long ld, int ncols, const int* __restrict__ dst, const double* __restrict__ tmp, long long ldt) {
    __shared__ int d;
    if (threadIdx.x == 0) d = dst[blockIdx.x];
    __syncthreads();
    const int c = blockIdx.y * 256 + threadIdx.x;
    if (c < ncols) X[(long long)d * ld + c] = tmp[(long long)blockIdx.x * ldt + c];
}

}  // namespace

// device scratch of the panel kernel for launches of at most gcap CTAs: [counter 64 B][top][cval][ccont][crow]
size_t getrf_slot_bytes(int gcap) {
    return 64 + (size_t)2 * LU_W * 8 + (size_t)2 * gcap * 8 + (size_t)2 * gcap * LU_W * 8 + (size_t)2 * gcap * 4 + 64;
}

// Panel width the kernel can take for m rows on this device (128, or less when a CTA's slab of a tall panel would not fit
// its shared memory: 64 from ~32000 rows, 32 from ~63000), the CTAs it will use and their rows; 0 if even 8 columns do not fit.
int getrf_panel_shape(long long m, int* G_out, int* rpc_out) {
    static int sms = 0, smem_max = 0, coop = 0;
    if (!sms) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    }
    static const int g_env = [] { const char* e = getenv("HCLOOC_GETRF_MAXG"); const int v = e ? atoi(e) : 0; return v > 0 ? v : LU_MAXG; }();   // experiment knob
    const int maxg = std::min(sms < LU_MAXG ? sms : LU_MAXG, g_env);
    const size_t avail = (size_t)smem_max - 4096;                 // static shared memory and the runtime's share
    static const int w_env = [] { const char* e = getenv("HCLOOC_GETRF_BW"); const int v = e ? atoi(e) : 0; return v >= 8 ? v : LU_W; }();     // experiment knob
    for (int w = LU_W; w >= 8; w >>= 1) {
        if (w > w_env) continue;
        long long G = (m + 127) / 128;
        if (G > maxg) G = maxg;
        if (G < 1) G = 1;
        if (!coop) G = 1;
        long long rpc = (m + G - 1) / G;
        if (rpc < w) rpc = w;                                      // CTA 0 owns every row that can become row j
        G = (m + rpc - 1) / rpc;
        if ((size_t)rpc * (w | 1) * 8 <= avail) { *G_out = (int)G; *rpc_out = (int)rpc; return w; }
    }
    return 0;
}

// Factor the m x w panel at dA (device, row-major, leading dimension lda) in place; pivot rows (panel-local + row_base) go to
// ipiv_out[0 .. min(m, w)) -- memory the device can write, e.g. pinned host memory; *d_info (device) receives
// info_base + j + 1 for the first exactly-zero pivot if it was 0.  `slots`: getrf_slot_bytes(gcap) of device scratch whose barrier
// counter (its first 8 bytes) holds *bar_base on entry; *bar_base is advanced by the arrivals of this launch.
int launch_getrf_panel(double* dA, int64_t lda, int64_t m, int w, long long* ipiv_out, long long row_base, long long* d_info,
                       long long info_base, void* slots, int gcap, unsigned long long* bar_base, cudaStream_t stream) {
    if (m <= 0 || w <= 0) return HCLOOC_OK;
    int G = 0, rpc = 0;
    const int wmax = getrf_panel_shape(m, &G, &rpc);
    if (w > wmax || G > gcap) return HCLOOC_ERR_INTERNAL;
    static bool attr_set = false;
    static int smem_max = 0;
    if (!attr_set) {
        int dev = 0;
        HCL_CUDA(cudaGetDevice(&dev));
        HCL_CUDA(cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
        HCL_CUDA(cudaFuncSetAttribute(getrf_panel_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max - 4096));
        attr_set = true;
    }
    // with fewer columns than the shape was made for, the rows per CTA stay (they fit a fortiori); rpc >= w holds
    PanelSlots sl;
    uint8_t* p = (uint8_t*)slots;
    sl.counter = (unsigned long long*)p;  p += 64;
    sl.top = (double*)p;                  p += (size_t)2 * LU_W * 8;
    sl.cval = (double*)p;                 p += (size_t)2 * gcap * 8;
    sl.ccont = (double*)p;                p += (size_t)2 * gcap * LU_W * 8;
    sl.crow = (int*)p;
    long long lda_ll = lda, m_ll = m;
    unsigned long long base = *bar_base;
    const size_t smem = (size_t)rpc * (w | 1) * 8;
    void* args[] = {&dA, &lda_ll, &m_ll, &w, &rpc, &G, &ipiv_out, &row_base, &d_info, &info_base, &sl, &base};
    if (G > 1) HCL_CUDA(cudaLaunchCooperativeKernel((const void*)getrf_panel_kernel, dim3(G), dim3(LU_T), args, smem, stream));
    else HCL_CUDA(cudaLaunchKernel((const void*)getrf_panel_kernel, dim3(1), dim3(LU_T), args, smem, stream));
    *bar_base = base + (unsigned long long)G * (unsigned long long)(m < w ? m : w);
    return HCLOOC_OK;
}

// X[dst[i]][c] <- X[src[i]][c] for i < nt, c < ncols, all sources read before any destination is written: gathered into tmp
// (at least nt * min(ncols, tmp_elems / nt) doubles, in column chunks), then scattered.  src / dst: memory the device can read.
int launch_row_permute(double* X, int64_t ld, int64_t ncols, int nt, const int* src, const int* dst, double* tmp, size_t tmp_elems,
                       cudaStream_t stream, uint64_t* n_kernels) {
    if (nt <= 0 || ncols <= 0) return HCLOOC_OK;
    int64_t chunk = (int64_t)(tmp_elems / (size_t)nt) / 32 * 32;
    if (chunk < 32) return HCLOOC_ERR_BUDGET;
    if (chunk > ncols) chunk = ncols;
    for (int64_t c0 = 0; c0 < ncols; c0 += chunk) {
        const int nc = (int)(ncols - c0 < chunk ? ncols - c0 : chunk);
        const dim3 grid((unsigned)nt, (unsigned)((nc + 255) / 256));
        row_gather_kernel<<<grid, 256, 0, stream>>>(X + c0, ld, nc, src, tmp, chunk);
        row_scatter_kernel<<<grid, 256, 0, stream>>>(X + c0, ld, nc, dst, tmp, chunk);
        *n_kernels += 2;
    }
    HCL_CUDA(cudaGetLastError());
    return HCLOOC_OK;
}

// Y[i][c] <- X[perm[i]][c] for i < nrows (out of place; the final pass of hclooc_dgetrf)
namespace {
__global__ void __launch_bounds__(256)
row_gather_all_kernel(const double* __restrict__ X, long long ldx, int ncols, const int* __restrict__ perm, double* __restrict__ Y, long long ldy) {
    __shared__ int s;
    if (threadIdx.x == 0) s = perm[blockIdx.x];
    __syncthreads();
    const int c = blockIdx.y * 256 + threadIdx.x;
    if (c < ncols) Y[(long long)blockIdx.x * ldy + c] = X[(long long)s * ldx + c];
}
}  // namespace

int launch_row_gather_all(const double* X, int64_t ldx, int64_t ncols, int64_t nrows, const int* perm, double* Y, int64_t ldy, cudaStream_t stream) {
    if (nrows <= 0 || ncols <= 0) return HCLOOC_OK;
    const dim3 grid((unsigned)nrows, (unsigned)((ncols + 255) / 256));
    row_gather_all_kernel<<<grid, 256, 0, stream>>>(X, ldx, (int)ncols, perm, Y, ldy);
    HCL_CUDA(cudaGetLastError());
    return HCLOOC_OK;
}

}  // namespace hclooc
