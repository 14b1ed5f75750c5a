// trsm_sm100.cu -- the diagonal-block kernel of the out-of-core DTRSM (hclooc_dtrsm; PAPER.md:412 names the routine as
// future work).  Solves  op(T) * X = scale * X  in place for one diagonal block T of at most 128 x 128
// and a row-major panel X of ib rows; everything off the diagonal blocks is DGEMM work and goes through the tile kernel.
//
// One thread owns one column of the panel (64 solving threads per CTA -- 256 are launched, all of which stage the triangle --,
// consecutive columns: every global access is a coalesced 512-byte row segment).  The block is held in shared memory TRANSPOSED and in "logical" order -- for an upper triangle the
// rows and columns are reversed, which turns it into a lower one -- so that the coefficients one thread needs next
// (column p of the triangle, 32 consecutive rows) are contiguous: they are read as broadcast LDS.128.  The 128 rows are
// processed as 4 sub-blocks of 32 rows held in registers: a left-looking update from the rows already solved (32
// independent DFMA chains per solved row), then the 32 x 32 triangle by fully unrolled substitution.  Rounding: the
// division by t_ii is a multiplication by the rounded reciprocal (two roundings instead of one; exact for t_ii = +-2^k).
#include "internal.h"

namespace hclooc {
namespace {

constexpr int TB = 128;          // largest diagonal block
constexpr int TCOLS = 64;        // columns (solving threads) per CTA (32 was measured slower: staging the triangle dominates)
constexpr int TS = TB + 2;       // row stride of the staged triangle: even (LDS.128 alignment), 4-way instead of 32-way store conflicts
constexpr int SUB = 32;          // rows held in registers
constexpr int TSTAGE = 256;      // threads per CTA: all of them stage the triangle, the first TCOLS solve
constexpr size_t TRSM_SMEM = (size_t)TB * TS * 8 + (size_t)TB * TCOLS * 8;   // 130 KiB triangle + 64 KiB solved rows

__global__ void __launch_bounds__(TSTAGE, 1)
trsm_block_kernel(const double* __restrict__ T, long long ldt, int ib, double* __restrict__ X, long long sq, long long si, int ncols,
                  int lower, int trans, int unit, double scale) {
    extern __shared__ __align__(16) double smem[];
    double* sTt = smem;                       // sTt[p * TS + q] = T'[q][p], T' = op(T) in logical (lower) order, 0 above, 1 on
    double* xs = smem + TB * TS;              //                  a unit / padded diagonal
    const int tid = threadIdx.x;
    // ---- stage the triangle with all TSTAGE threads: logical index q <-> actual index lower ? q : ib-1-q.  Consecutive
    // threads walk the direction that is contiguous in global memory (rows of T when it is stored untransposed, columns
    // when transposed); only the ib x ib corner is read, the rest of the 128 x 128 image is padding (0, diagonal 1).
    // (loads issued in batches of 8 per thread before their stores: the block comes from L2 / HBM at ~1 us per round trip)
    for (int base = 0; base < TB * TB; base += TSTAGE * 8) {
        double v[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int e = base + j * TSTAGE + tid;
            const int hi = e / TB, lo_ = e % TB;
            const int p = trans ? hi : lo_, q = trans ? lo_ : hi;     // element T'[q][p], wanted for q >= p
            const bool need = q < ib && p < ib && (q > p || (q == p && !unit));
            const int r = lower ? q : ib - 1 - q, c = lower ? p : ib - 1 - p;         // op(T)[r][c]
            const long long at = need ? (trans ? (long long)c * ldt + r : (long long)r * ldt + c) : 0;
            const double t = need ? T[at] : 0.0;
            v[j] = need ? t : ((q == p) ? 1.0 : 0.0);
        }
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int e = base + j * TSTAGE + tid;
            const int hi = e / TB, lo_ = e % TB;
            const int p = trans ? hi : lo_, q = trans ? lo_ : hi;
            const bool need = q < ib && p < ib && q == p && !unit;
            if (q >= p) sTt[p * TS + q] = need ? 1.0 / v[j] : v[j];   // the diagonal is kept as its reciprocal: x = b * (1/t) keeps
        }                                                             // the FP64 division out of the 128-step substitution chain
    }
    __syncthreads();
    if (tid >= TCOLS) return;                 // the extra threads only helped staging (no barrier follows)
    const int col = blockIdx.x * TCOLS + tid;
    const bool live = col < ncols;
    double b[SUB];
    for (int q0 = 0; q0 < ib; q0 += SUB) {
#pragma unroll
        for (int t = 0; t < SUB; ++t) {
            const int q = q0 + t;
            const int r = lower ? q : ib - 1 - q;
            b[t] = (live && q < ib) ? scale * X[(long long)r * sq + (long long)col * si] : 0.0;
        }
        // left-looking: subtract the contribution of the rows solved so far (xs is private to this thread's column)
#pragma unroll 2
        for (int p = 0; p < q0; ++p) {
            const double xv = xs[p * TCOLS + tid];
            const double2* trow = reinterpret_cast<const double2*>(sTt + p * TS + q0);
#pragma unroll
            for (int t = 0; t < SUB; t += 2) {
                const double2 tv = trow[t / 2];
                b[t] = fma(-tv.x, xv, b[t]);
                b[t + 1] = fma(-tv.y, xv, b[t + 1]);
            }
        }
        // the 32 x 32 triangle on the diagonal, right-looking in registers
#pragma unroll
        for (int t = 0; t < SUB; ++t) {
            const double* tcol = sTt + (q0 + t) * TS + q0;
            const double x = unit ? b[t] : b[t] * tcol[t];
            b[t] = x;
#pragma unroll
            for (int t2 = t + 1; t2 < SUB; ++t2) b[t2] = fma(-tcol[t2], x, b[t2]);
        }
#pragma unroll
        for (int t = 0; t < SUB; ++t) {
            const int q = q0 + t;
            xs[q * TCOLS + tid] = b[t];
            if (live && q < ib) {
                const int r = lower ? q : ib - 1 - q;
                X[(long long)r * sq + (long long)col * si] = b[t];
            }
        }
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
    static cudaError_t attr = cudaFuncSetAttribute(trsm_block_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TRSM_SMEM);
    if (attr != cudaSuccess) return cuda_fail(attr);
    const unsigned grid = (unsigned)((ncols + TCOLS - 1) / TCOLS);
    if (right)      // the operator of the row systems is op(T)^T: lower where op(T) is upper, and read with `trans` flipped
        trsm_block_kernel<<<grid, TSTAGE, TRSM_SMEM, stream>>>(dT, (long long)ldt, ib, dX, 1LL, (long long)ldx, (int)ncols, !lower, !trans, unit, scale);
    else
        trsm_block_kernel<<<grid, TSTAGE, TRSM_SMEM, stream>>>(dT, (long long)ldt, ib, dX, (long long)ldx, 1LL, (int)ncols, lower, trans, unit, scale);
    HCL_CUDA(cudaGetLastError());
    return HCLOOC_OK;
}

}  // namespace hclooc
