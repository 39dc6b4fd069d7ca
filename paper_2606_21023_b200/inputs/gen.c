/*
 * gen.c -- seeded, counter-based synthetic input generator (harness code).
 *
 * Serves BOTH the oracle-side tests and the CUDA path's tests/bench.  It holds none of the
 * method's arithmetic (no split, no products, no accumulation): it only produces the FP32
 * activations and FP16/FP32 weights the BASELINE.json configs describe.
 *
 * The value of element (tensor_id, row, col) under `seed` is a pure function of that tuple:
 *   key  = mix64(seed * 0x9E3779B97F4A7C15 + tensor_id)
 *   c    = mix64(key ^ (row * 2^32 + col))          (cols < 2^32)
 *   u1   = mix64(c), u2 = mix64(c + 0x9E3779B97F4A7C15)   -> two uniforms in (0,1), 53 bits
 *   normal : sigma * sqrt(-2 ln u1) * cos(2 pi u2)   (Box-Muller, double) -> RNE to FP32
 *   uniform: lo + (hi - lo) * u1                     (double)              -> RNE to FP32
 * so any row subset can be regenerated, and the M=1/8/32 activations are row prefixes of the
 * larger ones (cross-M bit-identity tests compare like with like).
 * FP16 weights are the FP32 value converted once more by the compiler's float -> _Float16
 * cast (IEEE round-to-nearest-even).
 */
#include <stdint.h>
#include <math.h>
#include <string.h>

static inline uint64_t mix64(uint64_t z)
{
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

static inline double u01(uint64_t r)            /* (0,1), never 0 or 1 */
{
    return ((double)(r >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

static inline float gen_value(uint64_t key, int64_t row, int64_t col, int dist, double p0, double p1)
{
    uint64_t c = mix64(key ^ (((uint64_t)row << 32) + (uint64_t)col));
    double a = u01(mix64(c));
    if (dist == 0) {                            /* N(0, p0^2) */
        double b = u01(mix64(c + 0x9E3779B97F4A7C15ull));
        return (float)(p0 * sqrt(-2.0 * log(a)) * cos(6.283185307179586476925286766559 * b));
    }
    return (float)(p0 + (p1 - p0) * a);         /* U(p0, p1) */
}

uint64_t heal_inputs_key(uint64_t seed, uint64_t tensor_id)
{
    return mix64(seed * 0x9E3779B97F4A7C15ull + tensor_id);
}

/*
 * Fill out[r][c] (row-major, leading dimension ld, elements) for rows row0..row0+nrows-1 and
 * cols 0..ncols-1 of tensor `tensor_id`.
 *   dist: 0 = normal(sigma=p0), 1 = uniform(p0, p1)
 *   scale_cols / n_scale / factor: the listed columns are multiplied by `factor` (the
 *     "outlier channels" of PAPER.md:201 -- fixed channels, reading A9); NULL/0 = none.
 *   as_f16: 0 -> out is float*, 1 -> out is uint16_t* holding binary16 bit patterns.
 */
void heal_inputs_fill(void *out, int64_t ld, int64_t row0, int64_t nrows, int64_t ncols,
                      uint64_t seed, uint64_t tensor_id, int dist, double p0, double p1,
                      const int64_t *scale_cols, int64_t n_scale, double factor, int as_f16)
{
    uint64_t key = heal_inputs_key(seed, tensor_id);
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < nrows; ++r) {
        for (int64_t c = 0; c < ncols; ++c) {
            float v = gen_value(key, row0 + r, c, dist, p0, p1);
            for (int64_t t = 0; t < n_scale; ++t)
                if (scale_cols[t] == c) v = (float)((double)v * factor);
            if (as_f16) {
                _Float16 h = (_Float16)v;
                memcpy((uint16_t *)out + r * ld + c, &h, 2);
            } else {
                ((float *)out)[r * ld + c] = v;
            }
        }
    }
}

/* n distinct column indices in [0, ncols), a pure function of (seed, tensor_id); ascending. */
void heal_inputs_outlier_cols(int64_t *cols, int64_t n, int64_t ncols, uint64_t seed, uint64_t tensor_id)
{
    uint64_t key = mix64(heal_inputs_key(seed, tensor_id) ^ 0x6F75746C69657273ull);
    int64_t got = 0;
    uint64_t ctr = 0;
    while (got < n) {
        int64_t c = (int64_t)(mix64(key + ctr++) % (uint64_t)ncols);
        int dup = 0;
        for (int64_t t = 0; t < got; ++t) dup |= (cols[t] == c);
        if (!dup) cols[got++] = c;
    }
    for (int64_t i = 1; i < n; ++i) {           /* insertion sort */
        int64_t v = cols[i], j = i - 1;
        while (j >= 0 && cols[j] > v) { cols[j + 1] = cols[j]; --j; }
        cols[j + 1] = v;
    }
}
