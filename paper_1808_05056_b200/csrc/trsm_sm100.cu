// trsm_sm100.cu -- the diagonal-block kernel of the out-of-core DTRSM (hclooc_dtrsm; PAPER.md:412 names the routine as
// future work).  Solves  op(T) * X = scale * X  in place for one diagonal block T of at most 128 x 128
// and a row-major panel X of ib rows; everything off the diagonal blocks is DGEMM work and goes through the tile kernel.
//
// One thread owns one right-hand side (256 per CTA); the block is held in shared memory TRANSPOSED and in "logical" order -- for
// an upper triangle the rows and columns are reversed, which turns it into a lower one -- so that the coefficients one thread
// needs next (column p of the triangle, 32 consecutive rows) are contiguous: they are read as broadcast LDS.128.  Rounding: the
// division by t_ii is a multiplication by the rounded reciprocal (two roundings instead of one; exact for t_ii = +-2^k).
#include <cstdlib>
#include "internal.h"

namespace hclooc {
namespace {

constexpr int TB = 128;          // largest diagonal block
constexpr int TS = TB + 2;       // row stride of the staged triangle: even (LDS.128 alignment), 4-way instead of 32-way store conflicts
constexpr int HB = 64;           // rows solved in registers at a time (half a block)
constexpr int CH = 16;           // rows of the second half updated at a time
constexpr int TTHREADS = 256;    // threads per CTA = right-hand sides per CTA: all of them stage the triangle, each solves one
constexpr size_t TRSM_SMEM = (size_t)TB * TS * 8;   // 130 KiB: the triangle only (one CTA of 8 warps per SM)

// the 64 x 64 triangle at `tri` (tri[p * TS + q] = T'[q][p], reciprocal diagonal) against 64 values in registers, right-looking:
// x_t <- x_t * (1 / t_tt), then x_t2 <- x_t2 - T'[t2][t] x_t for t2 > t; the coefficients of column t are contiguous in q and are
// read as broadcast LDS.128 pairs (the pair that starts at an even q below t + 1 carries one unused value)
__device__ __forceinline__ void solve64(double (&x)[HB], const double* __restrict__ tri, int unit) {
#pragma unroll
    for (int t = 0; t < HB; ++t) {
        const double* tcol = tri + t * TS;
        const double xv = unit ? x[t] : x[t] * tcol[t];
        x[t] = xv;
        const int e0 = (t + 1) & ~1;
#pragma unroll
        for (int e = e0; e < HB; e += 2) {
            const double2 tv = *reinterpret_cast<const double2*>(tcol + e);
            if (e > t) x[e] = fma(-tv.x, xv, x[e]);
            x[e + 1] = fma(-tv.y, xv, x[e + 1]);
        }
    }
}

// Stage the triangle with all threads of the CTA: sTt[p * TS + q] = T'[q][p] for q >= p, T' = op(T) in logical (lower) order, 1 on a
// unit / padded diagonal, the diagonal kept as its reciprocal.  Ends with a barrier.
__device__ __forceinline__ void stage_triangle(double* __restrict__ sTt, const double* __restrict__ T, long long ldt, int ib, int lower, int trans,
                                               int unit, int tid) {
    // ---- stage the triangle with all threads: logical index q <-> actual index lower ? q : ib-1-q.  Consecutive
    // threads walk the direction that is contiguous in global memory (rows of T when it is stored untransposed, columns
    // when transposed); only the ib x ib corner is read, the rest of the 128 x 128 image is padding (0, diagonal 1).
    // (loads issued in batches of 16 per thread before their stores: the block comes from L2 / HBM at ~1 us per round trip)
    for (int base = 0; base < TB * TB; base += TTHREADS * 16) {
        double v[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const int e = base + j * TTHREADS + tid;
            const int hi = e / TB, lo_ = e % TB;
            const int p = trans ? hi : lo_, q = trans ? lo_ : hi;     // element T'[q][p], wanted for q >= p
            const bool need = q < ib && p < ib && (q > p || (q == p && !unit));
            const int r = lower ? q : ib - 1 - q, c = lower ? p : ib - 1 - p;         // op(T)[r][c]
            const long long at = need ? (trans ? (long long)c * ldt + r : (long long)r * ldt + c) : 0;
            v[j] = __ldg(T + at);             // UNCONDITIONAL (element 0 when not needed): a predicated load followed by its select
        }                                     // made ptxas wait for every load before issuing the next -- 64 round trips, 30 us
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const int e = base + j * TTHREADS + tid;
            const int hi = e / TB, lo_ = e % TB;
            const int p = trans ? hi : lo_, q = trans ? lo_ : hi;
            const bool need = q < ib && p < ib && (q > p || (q == p && !unit));
            if (q >= p) sTt[p * TS + q] = need ? v[j] : ((q == p) ? 1.0 : 0.0);
        }
    }
    __syncthreads();
    // the diagonal is kept as its reciprocal: x = b * (1/t) keeps the FP64 division out of the 128-step substitution chain
    // (128 divisions per CTA, after the staging: a select between v and 1/v per staged element made every thread divide 64 times)
    if (tid < ib && !unit) sTt[tid * TS + tid] = 1.0 / sTt[tid * TS + tid];
    __syncthreads();
}

// One thread owns one right-hand side: a column of the panel (side = Left: consecutive threads read consecutive addresses) or a
// row of it (side = Right: a thread's values are contiguous; VEC = 4 reads and writes them as 32-byte vectors -- one full sector
// per thread and instruction -- when the block is a whole 128 and the rows are 32-byte aligned).  Element q of the logical
// (lower) system sits at P0[q * step].  The 128 rows are two halves of 64: the first half is loaded into registers and solved
// there (solve64), stored, and -- still in registers -- subtracted from the second half 16 rows at a time (load, 16 x 64 FMAs against
// broadcast LDS.128 coefficients, store); then the second half is loaded and solved the same way.  Shared memory holds nothing but
// the triangle, so a CTA carries 256 solving threads; a right-hand side makes two round trips through L1/L2 instead of living
// in a per-thread staging buffer.  `scale` multiplies every value at its first load.
template <int VEC, bool FULL>
__global__ void __launch_bounds__(TTHREADS, 1)
trsm_block_kernel(const double* __restrict__ T, long long ldt, int ib, double* __restrict__ X, long long sq, long long si, int nitems,
                  int lower, int trans, int unit, double scale) {
    extern __shared__ __align__(16) double smem[];
    double* sTt = smem;                       // sTt[p * TS + q] = T'[q][p], T' = op(T) in logical (lower) order, 0 above, 1 on
    const int tid = threadIdx.x;              //                  a unit / padded diagonal; the diagonal is kept as its reciprocal
    stage_triangle(sTt, T, ldt, ib, lower, trans, unit, tid);
    const long long item = (long long)blockIdx.x * TTHREADS + tid;
    if (item >= nitems) return;               // no barrier follows
    double* P0 = X + item * si + (lower ? 0 : (long long)(ib - 1) * sq);
    const long long step = lower ? sq : -sq;
    double x[HB];
    for (int h = 0; h * HB < ib; ++h) {
        const int q0 = h * HB;
        const double sc = h == 0 ? scale : 1.0;          // the second half was scaled when the first half was subtracted from it
        if (VEC == 4) {     // contiguous and 32-byte aligned: ascending (lower) or descending (upper) in memory
#pragma unroll
            for (int t = 0; t < HB; t += 4) {
                const double* p = lower ? P0 + q0 + t : P0 - (q0 + t) - 3;
                double a, b, c, d;
                asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p) : "memory");
                x[t] = sc * (lower ? a : d); x[t + 1] = sc * (lower ? b : c); x[t + 2] = sc * (lower ? c : b); x[t + 3] = sc * (lower ? d : a);
            }
        } else {
            const double* pp = P0 + (long long)q0 * step;
#pragma unroll
            for (int t = 0; t < HB; ++t) { x[t] = (FULL || q0 + t < ib) ? *pp : 0.0; pp += step; }
            if (sc != 1.0) {
#pragma unroll
                for (int t = 0; t < HB; ++t) x[t] *= sc;
            }
        }
        solve64(x, sTt + q0 * TS + q0, unit);
        if (VEC == 4) {
#pragma unroll
            for (int t = 0; t < HB; t += 4) {
                double* p = lower ? P0 + q0 + t : P0 - (q0 + t) - 3;
                if (lower) asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(x[t]), "d"(x[t + 1]), "d"(x[t + 2]), "d"(x[t + 3]) : "memory");
                else asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(x[t + 3]), "d"(x[t + 2]), "d"(x[t + 1]), "d"(x[t]) : "memory");
            }
        } else {
            double* pp = P0 + (long long)q0 * step;
#pragma unroll
            for (int t = 0; t < HB; ++t) { if (FULL || q0 + t < ib) *pp = x[t]; pp += step; }
        }
        if (h == 0) {
            // the second half receives the first half's contribution, CH rows at a time: b_t -= sum_p T'[64 + t][p] x_p
            for (int q1 = HB; q1 < ib; q1 += CH) {
                double b[CH];
                if (VEC == 4) {
#pragma unroll
                    for (int t = 0; t < CH; t += 4) {
                        const double* p = lower ? P0 + q1 + t : P0 - (q1 + t) - 3;
                        double a, bb, c, d;
                        asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(a), "=d"(bb), "=d"(c), "=d"(d) : "l"(p) : "memory");
                        b[t] = sc * (lower ? a : d); b[t + 1] = sc * (lower ? bb : c); b[t + 2] = sc * (lower ? c : bb); b[t + 3] = sc * (lower ? d : a);
                    }
                } else {
                    const double* pp = P0 + (long long)q1 * step;
#pragma unroll
                    for (int t = 0; t < CH; ++t) { b[t] = (FULL || q1 + t < ib) ? *pp : 0.0; pp += step; }
                    if (sc != 1.0) {
#pragma unroll
                        for (int t = 0; t < CH; ++t) b[t] *= sc;
                    }
                }
#pragma unroll
                for (int p = 0; p < HB; ++p) {                 // fully unrolled: x[] stays in registers
                    const double xv = x[p];
                    const double2* trow = reinterpret_cast<const double2*>(sTt + p * TS + q1);
#pragma unroll
                    for (int t = 0; t < CH; t += 2) {
                        const double2 tv = trow[t / 2];
                        b[t] = fma(-tv.x, xv, b[t]);
                        b[t + 1] = fma(-tv.y, xv, b[t + 1]);
                    }
                }
                if (VEC == 4) {
#pragma unroll
                    for (int t = 0; t < CH; t += 4) {
                        double* p = lower ? P0 + q1 + t : P0 - (q1 + t) - 3;
                        if (lower) asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(b[t]), "d"(b[t + 1]), "d"(b[t + 2]), "d"(b[t + 3]) : "memory");
                        else asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(b[t + 3]), "d"(b[t + 2]), "d"(b[t + 1]), "d"(b[t]) : "memory");
                    }
                } else {
                    double* pp = P0 + (long long)q1 * step;
#pragma unroll
                    for (int t = 0; t < CH; ++t) { if (FULL || q1 + t < ib) *pp = b[t]; pp += step; }
                }
            }
        }
    }
}

// The same substitution for SMALL panels (fewer right-hand sides than 64 per SM): a right-hand side is shared by SPLIT = 4
// neighbouring lanes, so a CTA of 256 threads solves 64 of them and the 128-step chain costs a quarter of the FMAs per lane -- the
// launch is latency bound (a panel of the Cholesky / DTRSM recursion: 96 us with one thread per right-hand side, whatever the
// panel's size).  Lane j of a group owns the logical elements 16 i + 4 j + c (i < 8, c < 4): 32 values in registers, read and
// written as 32-byte vectors when the panel allows it.  Step t: the owner of x_t scales it by 1 / t_tt, a width-4 shuffle hands
// it to the group, every lane updates its own elements below t.  The operations on an element and their order are those of
// trsm_block_kernel, so the two kernels give the same bits.
constexpr int SPLIT = 4;
constexpr int SITEMS = TTHREADS / SPLIT;

template <int VEC, bool FULL>
__global__ void __launch_bounds__(TTHREADS, 1)
trsm_block_split_kernel(const double* __restrict__ T, long long ldt, int ib, double* __restrict__ X, long long sq, long long si, int nitems,
                        int lower, int trans, int unit, double scale) {
    extern __shared__ __align__(16) double smem[];
    double* sTt = smem;
    const int tid = threadIdx.x;
    stage_triangle(sTt, T, ldt, ib, lower, trans, unit, tid);
    const int j = tid & (SPLIT - 1);
    long long item = (long long)blockIdx.x * SITEMS + (tid >> 2);
    const bool live = item < nitems;          // a group past the end solves the last right-hand side again and stores nothing
    if (!live) item = nitems - 1;             // (the shuffles below name every lane of the warp)
    double* P0 = X + item * si + (lower ? 0 : (long long)(ib - 1) * sq);
    const long long step = lower ? sq : -sq;
    double x[32];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int q = 16 * i + 4 * j;
        if (VEC == 4) {
            const double* p = lower ? P0 + q : P0 - q - 3;
            double a, b, c, d;
            asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p) : "memory");
            x[4 * i] = scale * (lower ? a : d); x[4 * i + 1] = scale * (lower ? b : c); x[4 * i + 2] = scale * (lower ? c : b); x[4 * i + 3] = scale * (lower ? d : a);
        } else {
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const double v = (FULL || q + c < ib) ? P0[(long long)(q + c) * step] : 0.0;
                x[4 * i + c] = scale != 1.0 ? scale * v : v;
            }
        }
    }
    // Eight groups of 16 steps, ONE copy of the code (a fully unrolled chain is 96 KB of straight-line code: every instruction
    // a cache miss): after a group its 16 elements are final -- each lane stores its four and shifts the rest down, so the pivot
    // block is always x[0..3] and the live blocks are i < 8 - tb (a uniform branch per block).
#pragma unroll 1
    for (int tb = 0; tb < 8; ++tb) {
        const int nact = 8 - tb;
        const double* tbase = sTt + (16 * tb) * TS + 16 * tb;      // tbase[tt * TS + e] = T'[16 tb + e][16 tb + tt]
#pragma unroll
        for (int tt = 0; tt < 16; ++tt) {
            const int li = tt % 4, owner = tt / 4;
            const double* tcol = tbase + tt * TS;
            const double cand = unit ? x[li] : x[li] * tcol[tt];
            const double xv = __shfl_sync(0xffffffffu, cand, owner, SPLIT);
            if (j == owner) x[li] = xv;
            {                                     // the block that holds the pivot: only the elements below it (what lies above is not staged)
                const double2 t01 = *reinterpret_cast<const double2*>(tcol + 4 * j);
                const double2 t23 = *reinterpret_cast<const double2*>(tcol + 4 * j + 2);
                const int e = 4 * j - tt;         // element c is below the pivot iff e + c > 0
                if (e > 0) x[0] = fma(-t01.x, xv, x[0]);
                if (e + 1 > 0) x[1] = fma(-t01.y, xv, x[1]);
                if (e + 2 > 0) x[2] = fma(-t23.x, xv, x[2]);
                if (e + 3 > 0) x[3] = fma(-t23.y, xv, x[3]);
            }
#pragma unroll
            for (int i = 1; i < 8; ++i) {
                if (i < nact) {                   // uniform
                    const double2 t01 = *reinterpret_cast<const double2*>(tcol + 16 * i + 4 * j);
                    const double2 t23 = *reinterpret_cast<const double2*>(tcol + 16 * i + 4 * j + 2);
                    x[4 * i] = fma(-t01.x, xv, x[4 * i]);
                    x[4 * i + 1] = fma(-t01.y, xv, x[4 * i + 1]);
                    x[4 * i + 2] = fma(-t23.x, xv, x[4 * i + 2]);
                    x[4 * i + 3] = fma(-t23.y, xv, x[4 * i + 3]);
                }
            }
        }
        if (live) {
            const int q = 16 * tb + 4 * j;
            if (VEC == 4) {
                double* p = lower ? P0 + q : P0 - q - 3;
                if (lower) asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(x[0]), "d"(x[1]), "d"(x[2]), "d"(x[3]) : "memory");
                else asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(x[3]), "d"(x[2]), "d"(x[1]), "d"(x[0]) : "memory");
            } else {
#pragma unroll
                for (int c = 0; c < 4; ++c)
                    if (FULL || q + c < ib) P0[(long long)(q + c) * step] = x[c];
            }
        }
#pragma unroll
        for (int k = 0; k < 28; ++k) x[k] = x[k + 4];
    }
}

}  // namespace

// X (ib x ncols, row-major, ldx) <- op(T)^-1 * (scale * X) for the ib x ib diagonal block T (row-major as stored, ldt);
// lower = op(T) is lower triangular, trans = op(T)[r][c] is stored at T[c][r], unit = the diagonal is 1 and not read.
// right != 0 (DTRSM side = Right, and the Cholesky panel): X is ncols x ib and X <- (scale * X) * op(T)^-1.  Every ROW of X is
// then an independent system op(T)^T x^T = b^T: the same substitution with the triangle read transposed and one thread per row
// of X instead of one per column (only the addressing of X changes: element (q, item) sits at X[item*ldx + q]).
int launch_trsm_block(const double* dT, int64_t ldt, int ib, double* dX, int64_t ldx, int64_t ncols, int lower, int trans,
                      int unit, double scale, cudaStream_t stream, int right) {
    if (ib <= 0 || ncols <= 0) return HCLOOC_OK;
    if (ib > TB || ncols > 0x7fffffffLL) return HCLOOC_ERR_INTERNAL;
    static cudaError_t attr = cudaFuncSetAttribute(trsm_block_kernel<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TRSM_SMEM);
    if (attr != cudaSuccess) return cuda_fail(attr);
    const unsigned grid = (unsigned)((ncols + TTHREADS - 1) / TTHREADS);
    // small panels: four lanes per right-hand side (same bits, a quarter of the chain per lane) while that still fits one wave
    const char* split_e = getenv("HCLOOC_TRSM_SPLIT");       // 0: never, 1: always (tests: the two kernels must give the same bits)
    const int split_env = split_e ? atoi(split_e) : -1;
    static int split_items = 0;
    if (split_items == 0) {
        int dev = 0, sms = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) sms = 148;
        split_items = SITEMS * sms;
    }
    if (split_env != 0 && (split_env == 1 || ncols <= split_items)) {
        static cudaError_t sa = [] {
            cudaError_t e = cudaFuncSetAttribute(trsm_block_split_kernel<4, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TRSM_SMEM);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(trsm_block_split_kernel<1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TRSM_SMEM);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(trsm_block_split_kernel<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TRSM_SMEM);
            return e;
        }();
        if (sa != cudaSuccess) return cuda_fail(sa);
        const unsigned sgrid = (unsigned)((ncols + SITEMS - 1) / SITEMS);
        if (right) {
            const bool vec = ib == TB && (ldx % 4 == 0) && (((uintptr_t)dX & 31u) == 0);
            if (vec) trsm_block_split_kernel<4, true><<<sgrid, TTHREADS, TRSM_SMEM, stream>>>(dT, (long long)ldt, ib, dX, 1LL, (long long)ldx, (int)ncols, !lower, !trans, unit, scale);
            else if (ib == TB) trsm_block_split_kernel<1, true><<<sgrid, TTHREADS, TRSM_SMEM, stream>>>(dT, (long long)ldt, ib, dX, 1LL, (long long)ldx, (int)ncols, !lower, !trans, unit, scale);
            else trsm_block_split_kernel<1, false><<<sgrid, TTHREADS, TRSM_SMEM, stream>>>(dT, (long long)ldt, ib, dX, 1LL, (long long)ldx, (int)ncols, !lower, !trans, unit, scale);
        } else if (ib == TB) {
            trsm_block_split_kernel<1, true><<<sgrid, TTHREADS, TRSM_SMEM, stream>>>(dT, (long long)ldt, ib, dX, (long long)ldx, 1LL, (int)ncols, lower, trans, unit, scale);
        } else {
            trsm_block_split_kernel<1, false><<<sgrid, TTHREADS, TRSM_SMEM, stream>>>(dT, (long long)ldt, ib, dX, (long long)ldx, 1LL, (int)ncols, lower, trans, unit, scale);
        }
        HCL_CUDA(cudaGetLastError());
        return HCLOOC_OK;
    }
    static cudaError_t attr4 = cudaFuncSetAttribute(trsm_block_kernel<4, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TRSM_SMEM);
    if (attr4 != cudaSuccess) return cuda_fail(attr4);
    static cudaError_t attr1 = cudaFuncSetAttribute(trsm_block_kernel<1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TRSM_SMEM);
    if (attr1 != cudaSuccess) return cuda_fail(attr1);
    if (right) {    // the operator of the row systems is op(T)^T: lower where op(T) is upper, and read with `trans` flipped
        // a thread's row is contiguous: 32-byte vectors when the block is whole and every row starts on a 32-byte boundary
        const bool vec = ib == TB && (ldx % 4 == 0) && (((uintptr_t)dX & 31u) == 0);
        if (vec) trsm_block_kernel<4, true><<<grid, TTHREADS, TRSM_SMEM, stream>>>(dT, (long long)ldt, ib, dX, 1LL, (long long)ldx, (int)ncols, !lower, !trans, unit, scale);
        else if (ib == TB) trsm_block_kernel<1, true><<<grid, TTHREADS, TRSM_SMEM, stream>>>(dT, (long long)ldt, ib, dX, 1LL, (long long)ldx, (int)ncols, !lower, !trans, unit, scale);
        else trsm_block_kernel<1, false><<<grid, TTHREADS, TRSM_SMEM, stream>>>(dT, (long long)ldt, ib, dX, 1LL, (long long)ldx, (int)ncols, !lower, !trans, unit, scale);
    } else if (ib == TB) {
        trsm_block_kernel<1, true><<<grid, TTHREADS, TRSM_SMEM, stream>>>(dT, (long long)ldt, ib, dX, (long long)ldx, 1LL, (int)ncols, lower, trans, unit, scale);
    } else {
        trsm_block_kernel<1, false><<<grid, TTHREADS, TRSM_SMEM, stream>>>(dT, (long long)ldt, ib, dX, (long long)ldx, 1LL, (int)ncols, lower, trans, unit, scale);
    }
    HCL_CUDA(cudaGetLastError());
    return HCLOOC_OK;
}

}  // namespace hclooc
