// potrf_sm100.cu -- the diagonal-block kernel of the out-of-core Cholesky factorization (hclooc_dpotrf; PAPER.md:412 names
// the factorization as future work on top of the out-of-core DGEMM).  Factors ONE block of at most
// 128 x 128 that sits in device memory; everything off these blocks is DGEMM / DSYRK / DTRSM work on the tile kernel.
//
// One CTA of 256 threads.  The triangle is staged into shared memory as a lower triangle L' (an upper factor U is its
// transpose: U^T U = L' L'^T with L' = U^T, so only the addressing of the global block changes), row stride 129 doubles so that
// "thread i works on row i" touches 32 different banks.  Right-looking by columns: for column j the pivot s = a_jj must be
// positive (else info), d = sqrt(s), rows below are divided by d (true FP64 division and IEEE sqrt: one rounding each, as in
// the definition), then the trailing triangle receives a_ik -= l_ij * l_kj.  Two threads share a row: they take alternate
// columns of the trailing update.  ALU / latency bound by construction (a 128-step dependent chain); it holds n^3/3 = 0.7 Mflop.
#include "internal.h"

namespace hclooc {
namespace {

constexpr int PB = 128;            // largest block
constexpr int PS = PB + 1;         // shared-memory row stride (bank-conflict free column access)
constexpr int PT = 256;            // threads per CTA
constexpr size_t POTRF_SMEM = (size_t)PB * PS * 8;

__global__ void __launch_bounds__(PT, 1)
potrf_block_kernel(double* __restrict__ A, long long lda, int n, int lower, long long* __restrict__ info, long long info_base) {
    extern __shared__ __align__(16) double S[];      // S[i * PS + k] = element (i, k) of the lower triangle L'
    __shared__ int bad;
    const int tid = threadIdx.x;
    if (tid == 0) bad = -1;
    // stage: consecutive threads walk the direction that is contiguous in global memory (rows of A)
    for (int e = tid; e < n * n; e += PT) {
        const int r = e / n, c = e % n;              // global element A[r][c]
        const bool in = lower ? (c <= r) : (c >= r);
        if (in) {
            const double v = A[(long long)r * lda + c];
            if (lower) S[r * PS + c] = v; else S[c * PS + r] = v;
        }
    }
    __syncthreads();
    const int row2 = tid >> 1, half = tid & 1;       // two threads per row of the trailing update
    for (int j = 0; j < n; ++j) {
        const double s = S[j * PS + j];
        if (!(s > 0.0)) {                            // not positive (or NaN): the leading minor of order j+1 is not positive definite
            if (tid == 0) bad = j;
            break;                                   // uniform: every thread read the same s
        }
        const double d = sqrt(s);
        __syncthreads();                             // everybody has read a_jj
        if (tid == j) S[j * PS + j] = d;
        if (tid > j && tid < n) S[tid * PS + j] = S[tid * PS + j] / d;
        __syncthreads();
        // trailing update: a_ik -= l_ij * l_kj for j < k <= i < n
        const int i = j + 1 + row2;
        if (i < n) {
            const double lij = S[i * PS + j];
            for (int k = j + 1 + half; k <= i; k += 2) {
                const double p = lij * S[k * PS + j];
                S[i * PS + k] = S[i * PS + k] - p;
            }
        }
        __syncthreads();
    }
    __syncthreads();
    if (tid == 0 && bad >= 0 && *info == 0) *info = info_base + bad + 1;
    // store the triangle back (also after a failure: the columns before `bad` are the factor's, LAPACK leaves the rest undefined)
    for (int e = tid; e < n * n; e += PT) {
        const int r = e / n, c = e % n;
        const bool in = lower ? (c <= r) : (c >= r);
        if (in) A[(long long)r * lda + c] = lower ? S[r * PS + c] : S[c * PS + r];
    }
}

}  // namespace

int launch_potrf_block(double* dA, int64_t lda, int n, int lower, long long* d_info, long long info_base, cudaStream_t stream) {
    if (n <= 0) return HCLOOC_OK;
    if (n > PB || !d_info) return HCLOOC_ERR_INTERNAL;
    static cudaError_t attr = cudaFuncSetAttribute(potrf_block_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)POTRF_SMEM);
    if (attr != cudaSuccess) return cuda_fail(attr);
    potrf_block_kernel<<<1, PT, POTRF_SMEM, stream>>>(dA, (long long)lda, n, lower, d_info, info_base);
    HCL_CUDA(cudaGetLastError());
    return HCLOOC_OK;
}

}  // namespace hclooc
