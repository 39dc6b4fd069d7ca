/*
 * heal_fusions.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (same rules as heal_oracle.c: only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load or call it; no code,
 * header, table or helper shared with paper_2606_21023_b200/csrc/; gcc only).
 *
 * Plain FP64 definitions of the element-wise steps that sit around HEAL's compensated GEMMs in the decoder layer of
 * Algorithm 1 and that the CUDA path fuses into the GEMM's prologue / epilogue (
 * "FP32 residual flow": hidden states, residual tensors, normalization inputs/outputs and operator outputs stay FP32,
 * PAPER.md:563):
 *
 *   F1  oracle_rmsnorm_f64    Norm(.) of  "g, u <- GEMM(Norm(A_i), W_gate_up)".  The paper names the
 *                             operator only; its models (Qwen3, Llama-3.1) use RMSNorm:
 *                                 y[k] = x[k] / sqrt( (1/K) sum_k x[k]^2 + eps ) * gamma[k]
 *                             (reading A17: formula and eps are the models', eps is an argument).
 *   F2  oracle_silu_mul_f64   "SiLU(g) (.) u"  of  "H_{i+1} <- A_i + GEMM(SiLU(g) (.) u, W_down)":
 *                                 h[j] = g[j] / (1 + exp(-g[j])) * u[j]
 *                             with g and u interleaved column-wise in the gate_up GEMM's output, c[2j] = g[j],
 *                             c[2j+1] = u[j] (reading A18: the paper writes "g, u <- GEMM(...)" and says
 *                             nothing about the column order; interleaving puts a (g, u) pair into one epilogue thread).
 *   F3  oracle_gemm_dd        C = A.B with A already double (the output of F1 / F2 fed to the next GEMM of the chain),
 *                             B FP16 or FP32 widened exactly, one double accumulator per element, k ascending: the same
 *                             definition as O1 (left-hand side of Eq. 10) for a double first operand.
 *   F4  oracle_add_f64        the residual add "A_i + GEMM(...)", element-wise in double.
 *
 * Pins: tests/test_oracle_pins.py (hand values, closed forms -- silu(x) - silu(-x) = x, silu(ln 3) = 3/4 ln 3, unit mean
 * square after RMSNorm with gamma = 1 and eps = 0, scale invariance -- and index-order cases that fail if gate and up,
 * or rows and columns, are swapped; F3 against O1 bit for bit on FP32-valued doubles and against exact int64 GEMMs).
 * Parity status: the paper prints no numeric example of these steps; the pins are mathematical.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

double oracle_f16_to_f64(uint16_t h);       /* heal_oracle.c (same library) */

/* F1: Y[i][k] = X[i][k] / sqrt(mean_k X[i][k]^2 + eps) * gamma[k];  X FP32 (pitch ldx), gamma FP32 or NULL (= ones), Y double
 * rows x cols dense. */
void oracle_rmsnorm_f64(int64_t rows, int64_t cols, const float *X, int64_t ldx, const float *gamma, double eps, double *Y)
{
    for (int64_t i = 0; i < rows; ++i) {
        double ss = 0.0;
        for (int64_t k = 0; k < cols; ++k) { double v = X[i * ldx + k]; ss += v * v; }
        double rms = sqrt(ss / (double)cols + eps);
        for (int64_t k = 0; k < cols; ++k)
            Y[i * cols + k] = (double)X[i * ldx + k] / rms * (gamma ? (double)gamma[k] : 1.0);
    }
}

/* F2: H[i][j] = silu(C[i][2j]) * C[i][2j+1], j = 0..cols-1;  C double rows x 2cols dense (gate, up interleaved), H double
 * rows x cols dense. */
void oracle_silu_mul_f64(int64_t rows, int64_t cols, const double *C, double *H)
{
    for (int64_t i = 0; i < rows; ++i)
        for (int64_t j = 0; j < cols; ++j) {
            double g = C[i * 2 * cols + 2 * j], u = C[i * 2 * cols + 2 * j + 1];
            H[i * cols + j] = g / (1.0 + exp(-g)) * u;
        }
}

/* F3: C[r][j] = sum_k A[i][k] * B[k][j]  (B[j][k] if b_nk), A double M x K dense, B FP16 bits or FP32 with pitch ldb;
 * rows == NULL: all M rows, else the listed ones.  C double R x N dense. */
int oracle_gemm_dd(int64_t M, int64_t N, int64_t K, const double *A, const void *B, int64_t ldb, int b_is_f16, int b_nk,
                   const int64_t *rows, int64_t nrows, double *C)
{
    int64_t R = rows ? nrows : M;
    if (M < 0 || N < 0 || K < 0) return -1;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t r = 0; r < R; ++r) {
        int64_t i = rows ? rows[r] : r;
        for (int64_t j = 0; j < N; ++j) {
            double acc = 0.0;
            for (int64_t k = 0; k < K; ++k) {
                int64_t bi = b_nk ? (j * ldb + k) : (k * ldb + j);
                double b = b_is_f16 ? oracle_f16_to_f64(((const uint16_t *)B)[bi]) : (double)((const float *)B)[bi];
                acc += A[i * K + k] * b;
            }
            C[r * N + j] = acc;
        }
    }
    return 0;
}

/* F4: Z = X + Y element-wise, X FP32 (pitch ldx), Y and Z double rows x cols dense. */
void oracle_add_f64(int64_t rows, int64_t cols, const float *X, int64_t ldx, const double *Y, double *Z)
{
    for (int64_t i = 0; i < rows; ++i)
        for (int64_t j = 0; j < cols; ++j) Z[i * cols + j] = (double)X[i * ldx + j] + Y[i * cols + j];
}
