/* synthgen.c -- seeded, counter-based synthetic matrix generator.
 *
 * Shared by the oracle tests, the GPU parity tests and bench.py.  It holds NO arithmetic of the
 * method (no products, no sums over k): it only maps (seed, matrix_id, i, j) -> one double, so any
 * element or sub-block of A, B or C0 can be regenerated at any time (C is overwritten in place by
 * the method, and at 214.7 GB a second copy is not affordable).
 *
 * Recipe:
 *   h      = splitmix64(seed ^ (matrix_id * 0x9E3779B97F4A7C15) ^ splitmix64(i * logical_cols + j))
 *   dist 0 : uniform [-1,1)      v = (h >> 11) * 2^-52 - 1
 *   dist 1 : integer {-4..4}     v = (double)((int)(h % 9) - 4)          (never -0.0)
 *   dist 2 : normal(0,1)         Box-Muller: u1 = ((h>>11)+1) * 2^-53, u2 = (splitmix64(h)>>11) * 2^-53,
 *                                v = sqrt(-2 ln u1) * cos(2 pi u2)       (host libm, generated once)
 */
#include <math.h>
#include <stdint.h>

static inline uint64_t splitmix64(uint64_t x) {
    x += 0x9E3779B97F4A7C15ull;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}

static inline double synth_value(uint64_t seed, uint64_t matrix_id, uint64_t lin, int dist) {
    uint64_t h = splitmix64(seed ^ (matrix_id * 0x9E3779B97F4A7C15ull) ^ splitmix64(lin));
    if (dist == 0) return (double)(h >> 11) * 0x1.0p-52 - 1.0;
    if (dist == 1) return (double)((int)(h % 9ull) - 4);
    {
        double u1 = ((double)(h >> 11) + 1.0) * 0x1.0p-53;
        double u2 = (double)(splitmix64(h) >> 11) * 0x1.0p-53;
        return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925286766559 * u2);
    }
}

/* Fill dst[r*ld + c], r < rows, c < cols, with logical element (row0 + r, col0 + c) of the matrix
 * `matrix_id` (1 = A, 2 = B, 3 = C) whose logical width is `logical_cols`.  Padding (c >= cols) is
 * not touched.  Returns 0, or -1 on a bad argument. */
int synth_fill(double* dst, int64_t rows, int64_t cols, int64_t ld, uint64_t seed, int matrix_id,
               int dist, int64_t row0, int64_t col0, int64_t logical_cols) {
    if (!dst || rows < 0 || cols < 0 || ld < cols || dist < 0 || dist > 2) return -1;
    #pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < rows; ++r) {
        double* row = dst + r * ld;
        uint64_t base = (uint64_t)(row0 + r) * (uint64_t)logical_cols + (uint64_t)col0;
        for (int64_t c = 0; c < cols; ++c) row[c] = synth_value(seed, (uint64_t)matrix_id, base + (uint64_t)c, dist);
    }
    return 0;
}

/* Fill every element of a buffer (including padding) with one bit pattern, e.g. a NaN poison. */
int synth_fill_const(double* dst, int64_t n, double v) {
    if (!dst || n < 0) return -1;
    #pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) dst[i] = v;
    return 0;
}
