// trsm_sm100.cu -- the diagonal-block kernel of the out-of-core DTRSM (hclooc_dtrsm; PAPER.md:412 names the routine as
// future work).  Solves  op(T) * X = scale * X  in place for one diagonal block T of at most 128 x 128
// and a row-major panel X of ib rows; everything off the diagonal blocks is DGEMM work and goes through the tile kernel.
//
// One thread owns one column of the panel (64 threads per CTA, consecutive columns: every global access is a coalesced
// 512-byte row segment).  The block is held in shared memory TRANSPOSED and in "logical" order -- for an upper triangle the
// rows and columns are reversed, which turns it into a lower one -- so that the coefficients one thread needs next
// (column p of the triangle, 32 consecutive rows) are contiguous: they are read as broadcast LDS.128.  The 128 rows are
// processed as 4 sub-blocks of 32 rows held in registers: a left-looking update from the rows already solved (32
// independent DFMA chains per solved row), then the 32 x 32 triangle by fully unrolled substitution.
#include "internal.h"

namespace hclooc {
namespace {

constexpr int TB = 128;          // largest diagonal block
constexpr int TCOLS = 64;        // columns (threads) per CTA
constexpr int SUB = 32;          // rows held in registers
constexpr size_t TRSM_SMEM = (size_t)TB * TB * 8 + (size_t)TB * TCOLS * 8;   // 128 KiB triangle + 64 KiB solved rows

__global__ void __launch_bounds__(TCOLS, 1)
trsm_block_kernel(const double* __restrict__ T, long long ldt, int ib, double* __restrict__ X, long long ldx, int ncols,
                  int lower, int trans, int unit, double scale) {
    extern __shared__ __align__(16) double smem[];
    double* sTt = smem;                       // sTt[p * TB + q] = T'[q][p], T' = op(T) in logical (lower) order, 0 above, 1 on
    double* xs = smem + TB * TB;              //                  a unit / padded diagonal
    const int tid = threadIdx.x;
    // ---- stage the triangle: logical index q <-> actual index lower ? q : ib-1-q
    for (int e = tid; e < TB * TB; e += TCOLS) {
        const int p = e / TB, q = e % TB;     // element T'[q][p], wanted for q >= p
        double v = 0.0;
        if (q < ib && p < ib) {
            if (q > p || (q == p && !unit)) {
                const int r = lower ? q : ib - 1 - q, c = lower ? p : ib - 1 - p;     // op(T)[r][c]
                v = trans ? T[(long long)c * ldt + r] : T[(long long)r * ldt + c];
            } else if (q == p) v = 1.0;
        } else if (q == p) v = 1.0;           // padding rows: x = b / 1
        sTt[e] = v;
    }
    __syncthreads();
    const int col = blockIdx.x * TCOLS + tid;
    const bool live = col < ncols;
    double b[SUB];
    for (int q0 = 0; q0 < ib; q0 += SUB) {
#pragma unroll
        for (int t = 0; t < SUB; ++t) {
            const int q = q0 + t;
            const int r = lower ? q : ib - 1 - q;
            b[t] = (live && q < ib) ? scale * X[(long long)r * ldx + col] : 0.0;
        }
        // left-looking: subtract the contribution of the rows solved so far (xs is private to this thread's column)
        for (int p = 0; p < q0; ++p) {
            const double xv = xs[p * TCOLS + tid];
            const double2* trow = reinterpret_cast<const double2*>(sTt + p * TB + q0);
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
            const double* tcol = sTt + (q0 + t) * TB + q0;
            const double x = unit ? b[t] : b[t] / tcol[t];
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
                X[(long long)r * ldx + col] = b[t];
            }
        }
    }
}

}  // namespace

// X (ib x ncols, row-major, ldx) <- op(T)^-1 * (scale * X) for the ib x ib diagonal block T (row-major as stored, ldt);
// lower = op(T) is lower triangular, trans = op(T)[r][c] is stored at T[c][r], unit = the diagonal is 1 and not read.
int launch_trsm_block(const double* dT, int64_t ldt, int ib, double* dX, int64_t ldx, int64_t ncols, int lower, int trans,
                      int unit, double scale, cudaStream_t stream) {
    if (ib <= 0 || ncols <= 0) return HCLOOC_OK;
    if (ib > TB || ncols > 0x7fffffffLL) return HCLOOC_ERR_INTERNAL;
    static cudaError_t attr = cudaFuncSetAttribute(trsm_block_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TRSM_SMEM);
    if (attr != cudaSuccess) return cuda_fail(attr);
    const unsigned grid = (unsigned)((ncols + TCOLS - 1) / TCOLS);
    trsm_block_kernel<<<grid, TCOLS, TRSM_SMEM, stream>>>(dT, (long long)ldt, ib, dX, (long long)ldx, (int)ncols, lower, trans, unit, scale);
    HCL_CUDA(cudaGetLastError());
    return HCLOOC_OK;
}

}  // namespace hclooc
