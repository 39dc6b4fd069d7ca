/*
 * heal_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU reference for HEAL's algebraic error-compensated
 * GEMM (Section 3 "Mitigating GEMM Truncation via FP16 Promotion and
 * Algebraic Compensation", Eq. 10; three-product form from Eq. 9).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call this file.  It shares no code, header, table or helper with the CUDA
 * path under paper_2606_21023_b200/csrc/ and includes no CUDA header.  Built with gcc only.
 *
 * What is here (each pinned by tests/test_oracle_pins.py):
 *   O1  oracle_gemm_f64      the definition the method approximates: C = A.B with every input
 *                            widened exactly to double, one double accumulator per element,
 *                            k ascending (the left-hand side of Eq. 10).
 *   O2  oracle_round16,      r16(): round-to-nearest-even FP32 -> IEEE binary16 by integer bit
 *       oracle_split         manipulation ("unbiased Round-to-Nearest-Even");
 *                            split h = h_hi + h_lo / 2^s  (s = 0 is the
 *                            BASELINE.json north_star reading, s = 10 the paper's, A1).
 *   O3  oracle_gemm_split    the right-hand side of Eq. 10 evaluated in exact (double)
 *                            arithmetic: sum over k of exactly the products the mode keeps
 *                            (2P: hi.W + lo.W; 3P: hi.hi + hi.lo + lo.hi, Eq. 9
 *                            expansion PAPER.md:195 with the lo.lo term dropped, A3).
 *
 * Parity status: the paper prints no numeric GEMM example, so O1/O2/O3 are pinned by
 * mathematics (closed forms, exact-integer GEMMs, brute force, x86 F16C / numpy float16
 * conversions, numpy float64 matmul), not by paper-printed values.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- binary16 <-> wider formats, by bit manipulation only ------------------------------- */

/* Exact value of an IEEE binary16 bit pattern (FP16 has 10 explicit
 * significand bits; 5 exponent bits, bias 15). */
double oracle_f16_to_f64(uint16_t h)
{
    uint64_t sign = (uint64_t)(h >> 15) << 63;
    uint32_t e    = (h >> 10) & 0x1f;
    uint64_t m    = h & 0x3ff;
    uint64_t bits;
    double v;
    if (e == 0) {                                 /* zero / subnormal: m * 2^-24 (exact) */
        v = (double)m * 0x1p-24;
        memcpy(&bits, &v, 8);
        bits |= sign;
    } else if (e == 31) {                         /* Inf / NaN */
        bits = sign | 0x7ff0000000000000ull | (m << 42);
    } else {                                      /* (1 + m/1024) * 2^(e-15): rebias 15 -> 1023 */
        bits = sign | ((uint64_t)(e - 15 + 1023) << 52) | (m << 42);
    }
    memcpy(&v, &bits, 8);
    return v;
}

/* r16(x): FP32 -> binary16, round to nearest, ties to even, subnormals kept, overflow to
 * Inf (values >= 65520 round to Inf).  Pure integer arithmetic on the FP32 pattern. */
uint16_t oracle_round16(float x)
{
    uint32_t u;
    memcpy(&u, &x, 4);
    uint16_t sign = (uint16_t)((u >> 16) & 0x8000u);
    uint32_t abs  = u & 0x7fffffffu;
    if (abs > 0x7f800000u) return (uint16_t)(sign | 0x7e00u);           /* NaN  */
    if (abs == 0x7f800000u) return (uint16_t)(sign | 0x7c00u);          /* Inf  */
    int32_t e = (int32_t)(abs >> 23) - 127;                              /* unbiased */
    uint32_t m = abs & 0x7fffffu;
    if ((abs >> 23) == 0) return sign;           /* FP32 subnormal (< 2^-126): far below 2^-25 -> 0 */
    /* 24-bit significand with the hidden one */
    uint64_t sig = (uint64_t)(m | 0x800000u);    /* value = sig * 2^(e-23) */
    /* target: integer q in units of 2^q_exp, q_exp = max(e,-14) - 10 */
    int32_t q_exp = (e < -14 ? -14 : e) - 10;
    int32_t shift = q_exp - (e - 23);            /* >= 13 */
    uint64_t q, rem, half;
    if (shift >= 40) { q = 0; rem = 1; half = 2; }      /* far too small: rounds to zero */
    else {
        q    = sig >> shift;
        rem  = sig & (((uint64_t)1 << shift) - 1);
        half = (uint64_t)1 << (shift - 1);
    }
    if (rem > half || (rem == half && (q & 1))) q += 1;
    /* assemble: q is in [0, 2048]; 2048 means carry into the next binade */
    uint32_t out;
    if (e < -14) {
        out = (uint32_t)q;                       /* subnormal field; q==1024 becomes min normal */
    } else {
        uint32_t be = (uint32_t)(e + 15);
        out = (be << 10) + (uint32_t)(q - 1024); /* q==2048 carries into exponent */
    }
    if (out >= 0x7c00u) out = 0x7c00u;           /* overflow -> Inf */
    return (uint16_t)(sign | out);
}

/* Split:  hi = r16(x);  lo = r16((x - hi) * 2^s).
 * x - hi is evaluated in double (exact: both are FP32-representable and the difference needs
 * at most 24 bits), the scale by 2^s is exact, then rounded once to FP32 (exact again) and r16. */
void oracle_split(int64_t n, const float *x, uint16_t *hi, uint16_t *lo, int s)
{
    for (int64_t i = 0; i < n; ++i) {
        uint16_t h = oracle_round16(x[i]);
        double r = ((double)x[i] - oracle_f16_to_f64(h)) * ldexp(1.0, s);
        hi[i] = h;
        lo[i] = oracle_round16((float)r);
    }
}

/* ---- O1: the plain definition ------------------------------------------------------------ */

static inline double b_at(const void *B, int b_is_f16, int64_t idx)
{
    return b_is_f16 ? oracle_f16_to_f64(((const uint16_t *)B)[idx])
                    : (double)((const float *)B)[idx];
}

/*
 * Cref[r][j] = sum_{k=0}^{K-1} (double)A[rows[r]][k] * (double)B[k][j]      (k ascending)
 *   A      FP32 row-major, lda >= K
 *   B      FP16 bit patterns (b_is_f16=1) or FP32 (b_is_f16=0); row-major K x N with ldb >= N,
 *          or, if b_nk=1, N x K with ldb >= K (the paper's W^T storage)
 *   rows   optional list of nrows row indices (NULL: all M rows, nrows ignored)
 *   C      double, nrows_out x N, leading dimension N
 * Returns 0, or -1 on bad arguments.
 */
int oracle_gemm_f64(int64_t M, int64_t N, int64_t K,
                    const float *A, int64_t lda,
                    const void *B, int64_t ldb, int b_is_f16, int b_nk,
                    const int64_t *rows, int64_t nrows, double *C)
{
    if (M < 0 || N < 0 || K < 0) return -1;
    int64_t R = rows ? nrows : M;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t r = 0; r < R; ++r) {
        int64_t i = rows ? rows[r] : r;
        double *c = C + r * N;
        for (int64_t j = 0; j < N; ++j) c[j] = 0.0;
        if (b_nk) {
            for (int64_t j = 0; j < N; ++j) {
                double acc = 0.0;
                for (int64_t k = 0; k < K; ++k)
                    acc += (double)A[i * lda + k] * b_at(B, b_is_f16, j * ldb + k);
                c[j] = acc;
            }
        } else {
            /* i-k-j order over the double row buffer: each c[j] still receives its K terms
             * in ascending k, one accumulator per element. */
            for (int64_t k = 0; k < K; ++k) {
                double a = (double)A[i * lda + k];
                for (int64_t j = 0; j < N; ++j)
                    c[j] += a * b_at(B, b_is_f16, k * ldb + j);
            }
        }
    }
    return 0;
}

/* ---- O3: Eq. 10 / Eq. 9 evaluated exactly ------------------------------------------------- */

/*
 * n_prod = 1: sum_k hi(a).b                          (single FP16 GEMM, HEAL-Base)
 * n_prod = 2: sum_k (hi(a) + lo(a)/2^s).b           (Eq. 10; B must be FP16)
 * n_prod = 3: sum_k hi(a)hi(b) + hi(a)lo(b)/2^s + lo(a)hi(b)/2^s   (Eq. 9 expansion, B FP32)
 * n_prod = 4: n_prod 3 plus lo(a)lo(b)/4^s          (diagnostic)
 * For n_prod <= 2 with an FP32 B, b is first rounded to FP16 (hi(b)).
 * All products and sums in double: each product of two binary16 values is exact, the sum's
 * own rounding is ~K*2^-53.
 */
int oracle_gemm_split(int64_t M, int64_t N, int64_t K,
                      const float *A, int64_t lda,
                      const void *B, int64_t ldb, int b_is_f16, int b_nk,
                      int n_prod, int s,
                      const int64_t *rows, int64_t nrows, double *C)
{
    if (M < 0 || N < 0 || K < 0 || n_prod < 1 || n_prod > 4) return -1;
    if (n_prod >= 3 && b_is_f16) return -1;
    int64_t R = rows ? nrows : M;
    int64_t brow = b_nk ? N : K, bcol = b_nk ? K : N;
    double inv = ldexp(1.0, -s);
    /* planes of B as doubles: bh (hi) and bl (lo / 2^s) */
    double *bh = (double *)malloc(sizeof(double) * (size_t)(brow * bcol + 1));
    double *bl = (double *)malloc(sizeof(double) * (size_t)(brow * bcol + 1));
    if (!bh || !bl) { free(bh); free(bl); return -2; }
    for (int64_t p = 0; p < brow; ++p)
        for (int64_t q = 0; q < bcol; ++q) {
            if (b_is_f16) {
                bh[p * bcol + q] = oracle_f16_to_f64(((const uint16_t *)B)[p * ldb + q]);
                bl[p * bcol + q] = 0.0;
            } else {
                uint16_t h, l;
                oracle_split(1, (const float *)B + p * ldb + q, &h, &l, s);
                bh[p * bcol + q] = oracle_f16_to_f64(h);
                bl[p * bcol + q] = oracle_f16_to_f64(l) * inv;
            }
        }
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t r = 0; r < R; ++r) {
        int64_t i = rows ? rows[r] : r;
        double *c = C + r * N;
        /* planes of this row of A as doubles: ah (hi) and al (lo / 2^s) */
        double *ah = (double *)malloc(sizeof(double) * (size_t)(K + 1));
        double *al = (double *)malloc(sizeof(double) * (size_t)(K + 1));
        for (int64_t k = 0; k < K; ++k) {
            uint16_t h, l;
            oracle_split(1, A + i * lda + k, &h, &l, s);
            ah[k] = oracle_f16_to_f64(h);
            al[k] = oracle_f16_to_f64(l) * inv;
        }
        for (int64_t j = 0; j < N; ++j) {
            double acc = 0.0;
            for (int64_t k = 0; k < K; ++k) {
                int64_t bi = b_nk ? (j * bcol + k) : (k * bcol + j);
                double t = ah[k] * bh[bi];
                if (n_prod >= 2) t += al[k] * bh[bi];
                if (n_prod >= 3) t += ah[k] * bl[bi];
                if (n_prod >= 4) t += al[k] * bl[bi];
                acc += t;
            }
            c[j] = acc;
        }
        free(ah); free(al);
    }
    free(bh); free(bl);
    return 0;
}

/* ---- acceptance metric (BASELINE.json north_star) ----------------------------------------- */

/* sum of squares of a strided FP32 / FP16 / double matrix, in double */
double oracle_sumsq_f32(int64_t rows, int64_t cols, const float *X, int64_t ld)
{
    double s = 0.0;
    for (int64_t i = 0; i < rows; ++i)
        for (int64_t j = 0; j < cols; ++j) { double v = X[i * ld + j]; s += v * v; }
    return s;
}
double oracle_sumsq_f16(int64_t rows, int64_t cols, const uint16_t *X, int64_t ld)
{
    double s = 0.0;
    for (int64_t i = 0; i < rows; ++i)
        for (int64_t j = 0; j < cols; ++j) { double v = oracle_f16_to_f64(X[i * ld + j]); s += v * v; }
    return s;
}
/* sum over (r,j) of (C[r][j] - Cref[r][j])^2, C FP32 with leading dimension ldc and row list */
double oracle_diff_sumsq(int64_t R, int64_t N, const float *C, int64_t ldc,
                         const int64_t *rows, const double *Cref)
{
    double s = 0.0;
    for (int64_t r = 0; r < R; ++r) {
        int64_t i = rows ? rows[r] : r;
        for (int64_t j = 0; j < N; ++j) { double d = (double)C[i * ldc + j] - Cref[r * N + j]; s += d * d; }
    }
    return s;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
