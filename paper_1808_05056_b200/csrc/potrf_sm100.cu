// potrf_sm100.cu -- the diagonal-block kernel of the out-of-core Cholesky factorization (hclooc_dpotrf; PAPER.md:412 names
// the factorization as future work on top of the out-of-core DGEMM).  Factors ONE block of at most
// 128 x 128 that sits in device memory; everything off these blocks is DGEMM / DSYRK / DTRSM work on the tile kernel.
//
// One CTA of 256 threads; the triangle is staged into shared memory as a lower triangle L' (an upper factor U is its transpose:
// U^T U = L' L'^T with L' = U^T, so only the addressing of the global block changes), row stride 129 doubles so that "thread i
// works on row i" touches 32 different banks.  Blocked by 32 columns, right-looking:
//   (1) the 32 x 32 diagonal block is factored by ONE WARP in registers -- lane i holds row i; column j: the pivot travels by
//       shuffle, must be positive (else info), d = sqrt(pivot), the lanes below divide by d (IEEE sqrt and division: one rounding
//       each, as in the definition), and every later column k receives l_ij * l_kj with l_kj shuffled from lane k;
//   (2) the rows below it are solved against the block, one thread per row: x L_D^T = a, 32 steps in registers with the
//       coefficients broadcast from shared memory;
//   (3) the trailing triangle receives  a_ik -= sum_j l_ij l_kj  in 4 x 4 register tiles spread over all threads.
// Three barriers per 32 columns instead of three per column.  ALU / latency bound by construction; it holds n^3/3 = 0.7 Mflop.
#include "internal.h"

namespace hclooc {
namespace {

constexpr int PB = 128;            // largest block
constexpr int PS = PB + 1;         // shared-memory row stride (bank-conflict free column access)
constexpr int PT = 256;            // threads per CTA
constexpr int PW = 32;             // columns per step (one warp factors the diagonal block)
constexpr size_t POTRF_SMEM = (size_t)(PB + 4) * PS * 8;   // + 4 rows: the 4 x 4 tiles of a ragged block read past row n

__device__ __forceinline__ double shfl_f64(double v, int src) {
    int lo = __double2loint(v), hi = __double2hiint(v);
    lo = __shfl_sync(0xffffffffu, lo, src);
    hi = __shfl_sync(0xffffffffu, hi, src);
    return __hiloint2double(hi, lo);
}

// column J of the 32 x 32 diagonal block held one row per lane (compile-time recursion: d[] must stay in registers)
template <int J>
__device__ __forceinline__ void potrf_warp_col(double (&d)[PW], int lane, int& fail, double* __restrict__ rd) {
    double ajj = shfl_f64(d[J], J);
    if (fail < 0 && !(ajj > 0.0)) fail = J;                  // uniform: every lane holds the same ajj
    if (fail >= 0) ajj = 1.0;                                 // keep going on harmless values: the block is abandoned
    const double r = sqrt(ajj);
    const double rinv = 1.0 / r;                              // the rows below multiply by the rounded reciprocal (one rounding more
    const double lij = lane > J ? d[J] * rinv : (lane == J ? r : d[J]);   // than dividing: inside gamma_(N+2), G24; exact for l_jj = 2^k)
    d[J] = lij;
    if (lane == 0) rd[J] = rinv;

#pragma unroll
    for (int k = J + 1; k < PW; ++k) {
        const double lkj = shfl_f64(lij, k);
        const double p = lij * lkj;
        if (lane >= k) d[k] = d[k] - p;
    }
    if constexpr (J + 1 < PW) potrf_warp_col<J + 1>(d, lane, fail, rd);
}

__global__ void __launch_bounds__(PT, 1)
potrf_block_kernel(double* __restrict__ A, long long lda, int n, int lower, long long* __restrict__ info, long long info_base) {
    extern __shared__ __align__(16) double S[];      // S[i * PS + k] = element (i, k) of the lower triangle L'
    __shared__ int bad;
    __shared__ double rdiag[PB];                     // 1 / l_jj of the columns factored so far
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) bad = -1;
    // stage: consecutive threads walk the direction that is contiguous in global memory (rows of A); rows and columns beyond n are
    // padded with the identity so that the last step of a ragged block factors a full 32 x 32 block
    // (loads issued in batches of 16 per thread before their stores: one round trip to L2 / HBM per batch instead of one per element)
    for (int base = 0; base < PB * PB; base += PT * 16) {
        double v[16];
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            const int e = base + u * PT + tid;
            const int r = e / PB, c = e % PB;                // global element A[r][c] = logical (r, c) of a lower, (c, r) of an upper block
            const int i = lower ? r : c, k = lower ? c : r;  // logical element (i, k), wanted for k <= i
            v[u] = A[(k <= i && i < n) ? (long long)r * lda + c : 0];    // unconditional (element 0 when not wanted): the loads of a batch must not wait for each other
        }
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            const int e = base + u * PT + tid;
            const int r = e / PB, c = e % PB;
            const int i = lower ? r : c, k = lower ? c : r;
            if (k <= i) S[i * PS + k] = (i < n) ? v[u] : (i == k ? 1.0 : 0.0);
        }
    }
    __syncthreads();
    for (int c0 = 0; c0 < n; c0 += PW) {
        // ---- (1) the diagonal block, warp 0, lane i = row c0 + i
        if (warp == 0) {
            double d[PW];
#pragma unroll
            for (int k = 0; k < PW; ++k) d[k] = S[(c0 + lane) * PS + c0 + k];
            int fail = -1;
            potrf_warp_col<0>(d, lane, fail, rdiag + c0);
            if (fail >= 0 && lane == 0) bad = c0 + fail;
#pragma unroll
            for (int k = 0; k < PW; ++k) if (k <= lane) S[(c0 + lane) * PS + c0 + k] = d[k];
        }
        __syncthreads();
        if (bad >= 0) break;                                              // uniform: read after the barrier
        // ---- (2) the rows below: x L_D^T = a, one thread per row
        {
            const int r = c0 + PW + tid;
            if (r < n) {
                double a[PW];
#pragma unroll
                for (int k = 0; k < PW; ++k) a[k] = S[r * PS + c0 + k];
#pragma unroll
                for (int j = 0; j < PW; ++j) {
                    const double xj = a[j] * rdiag[c0 + j];
                    a[j] = xj;
#pragma unroll
                    for (int t = j + 1; t < PW; ++t) { const double p = xj * S[(c0 + t) * PS + c0 + j]; a[t] = a[t] - p; }
                }
#pragma unroll
                for (int k = 0; k < PW; ++k) S[r * PS + c0 + k] = a[k];
            }
        }
        __syncthreads();
        // ---- (3) the trailing triangle: a_ik -= sum_j l_ij l_kj, 4 x 4 register tiles, tile (ti, tk) with tk <= ti
        {
            const int m0 = c0 + PW, m = n - m0;
            if (m > 0) {
                const int nt = (m + 3) / 4;
                for (int t = tid; t < nt * nt; t += PT) {
                    const int ti = t / nt, tk = t % nt;
                    if (tk > ti) continue;
                    const int i0 = m0 + 4 * ti, k0 = m0 + 4 * tk;
                    double acc[4][4];
#pragma unroll
                    for (int a = 0; a < 4; ++a)
#pragma unroll
                        for (int b = 0; b < 4; ++b) acc[a][b] = 0.0;
#pragma unroll 8
                    for (int j = 0; j < PW; ++j) {
                        double li[4], lk[4];
#pragma unroll
                        for (int a = 0; a < 4; ++a) { li[a] = S[(i0 + a) * PS + c0 + j]; lk[a] = S[(k0 + a) * PS + c0 + j]; }   // rows < 128 + 3: padded
#pragma unroll
                        for (int a = 0; a < 4; ++a)
#pragma unroll
                            for (int b = 0; b < 4; ++b) acc[a][b] = fma(li[a], lk[b], acc[a][b]);
                    }
#pragma unroll
                    for (int a = 0; a < 4; ++a)
#pragma unroll
                        for (int b = 0; b < 4; ++b) {
                            const int i = i0 + a, k = k0 + b;
                            if (i < n && k <= i) S[i * PS + k] = S[i * PS + k] - acc[a][b];
                        }
                }
            }
        }
        __syncthreads();
    }
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
