// transpose_sm100.cu -- staging step of the transposed-operand calls (hclooc_dgemm_t): a slice of op(A) = A^T or
// op(B) = B^T arrives from the host in the layout it is stored in (DMA cannot transpose) and is turned into the
// row-major slice the tile kernel's tensor maps expect.  HBM-bound and tiny beside the DGEMM of the step: a slice is
// read and written once (16 B per element at ~6.5 TB/s against 2*nb flops per element of an A slice).
//
//   dst[c * ldd + r] = src[r * lds + c]      r < rows, c < cols
//
// 32 x 32 tiles through shared memory (row pitch 33 doubles: conflict-free both ways), both sides coalesced.
#include <cuda_runtime.h>
#include <stdint.h>
#include "internal.h"

namespace hclooc {

namespace {

constexpr int TT = 32;

__global__ void __launch_bounds__(TT * 8)
hclooc_transpose_kernel(const double* __restrict__ src, long long lds, double* __restrict__ dst, long long ldd,
                        int rows, int cols, int tiles_c) {
    __shared__ double tile[TT][TT + 1];
    const int tr = blockIdx.x / tiles_c, tc = blockIdx.x - tr * tiles_c;
    const int r0 = tr * TT, c0 = tc * TT;
    const int x = threadIdx.x & 31, y = threadIdx.x >> 5;
    #pragma unroll
    for (int i = y; i < TT; i += 8) {
        const int r = r0 + i, c = c0 + x;
        if (r < rows && c < cols) tile[i][x] = src[(long long)r * lds + c];
    }
    __syncthreads();
    #pragma unroll
    for (int i = y; i < TT; i += 8) {
        const int c = c0 + i, r = r0 + x;
        if (r < rows && c < cols) dst[(long long)c * ldd + r] = tile[x][i];
    }
}

}  // namespace

int launch_transpose(const double* src, int64_t rows, int64_t cols, int64_t lds, double* dst, int64_t ldd, cudaStream_t stream) {
    if (rows <= 0 || cols <= 0) return HCLOOC_OK;
    const int64_t tr = (rows + TT - 1) / TT, tc = (cols + TT - 1) / TT;
    if (tr * tc > 0x7fffffffLL || rows > 0x7fffffffLL || cols > 0x7fffffffLL) return HCLOOC_ERR_INTERNAL;
    hclooc_transpose_kernel<<<(unsigned)(tr * tc), TT * 8, 0, stream>>>(src, (long long)lds, dst, (long long)ldd, (int)rows, (int)cols, (int)tc);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    return HCLOOC_OK;
}

}  // namespace hclooc
