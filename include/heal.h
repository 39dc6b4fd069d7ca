/*
 * heal.h -- C ABI of the B200-native HEAL compensated GEMM library (libheal.so).
 *
 * The operation (Section 3 "Mitigating GEMM Truncation via FP16 Promotion and
 * Algebraic Compensation"): an FP32 activation matrix h is decomposed into two FP16 matrices,
 *      h = h_hi + h_lo / 2^s            hi = r16(h),  lo = r16((h - hi) * 2^s)
 * (r16 = round-to-nearest-even to IEEE binary16) and the GEMM is expanded into FP16 tensor-core
 * products accumulated in FP32 into an FP32 output (Eq. 10, 563, 571):
 *      2 products:  C = h_hi.W + h_lo.W                         W already FP16      (Eq. 10)
 *      3 products:  C = A_hi.B_hi + A_hi.B_lo + A_lo.B_hi       both operands FP32  (Eq. 9 expansion,
 *                                                               PAPER.md:195; lo.lo dropped)
 *      1 product :  C = h_hi.W                                  the "skipped layer" / HEAL-Base GEMM
 *
 * The default is s = 0 (BASELINE.json north_star: lo = r16(x - hi), all products into one
 * accumulator); the paper's s = 10 is the HEAL_LO_SCALED variant below (reading A1).
 *
 * Reduction order (fixed; a function of K and mode only, never of M, N, tile shape or launch):
 *   K is cut into segments of HEAL_K_SEGMENT = 512 consecutive k.  Within a segment the tensor core
 *   accumulates in FP32, k ascending in slices of 16, the products of one slice issued in the order
 *   listed above.  Segment partial sums are added in FP32 (round-to-nearest) in ascending segment
 *   order.  No split-K atomics.  Results are bit-identical run to run, across M and across row
 *   position.
 *
 * All matrices are row-major.  Unless a function says "host", pointers are DEVICE pointers, and
 * the call is asynchronous on `stream` (a cudaStream_t passed as void*; NULL = the legacy default
 * stream).  The library never prints and never aborts; every entry point returns a heal_status.
 * There is no CPU fallback: without an sm_100 device every compute call returns HEAL_ERR_CUDA /
 * HEAL_ERR_UNSUPPORTED_DEVICE.
 */
#ifndef HEAL_H_
#define HEAL_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    HEAL_OK = 0,
    HEAL_ERR_INVALID_VALUE = 1,      /* negative dimension, leading dimension too small            */
    HEAL_ERR_NULL_POINTER = 2,       /* NULL matrix pointer with a non-empty problem               */
    HEAL_ERR_MISALIGNED = 3,         /* pointer not 16-byte aligned / leading dimension not a
                                        multiple of 16 bytes (TMA and 128-bit loads need both)     */
    HEAL_ERR_UNSUPPORTED_MODE = 4,   /* unknown mode bits, or B dtype/mode mismatch                */
    HEAL_ERR_CUDA = 5,               /* a CUDA call failed; see heal_last_cuda_error()             */
    HEAL_ERR_WORKSPACE = 6,          /* caller-supplied workspace too small                        */
    HEAL_ERR_UNSUPPORTED_DEVICE = 7  /* current device is not sm_100, or differs from the device of the
                                        process's first call (one device per process)              */
} heal_status;

#define HEAL_K_SEGMENT 512

/* mode word ------------------------------------------------------------------------------------ */
#define HEAL_MODE_PRODUCTS_MASK 0x0fu
#define HEAL_MODE_1P 1u        /* hi.W                      B is FP16                              */
#define HEAL_MODE_2P 2u        /* hi.W + lo.W               B is FP16   (Eq. 10)     */
#define HEAL_MODE_3P 3u        /* hi.hi + hi.lo + lo.hi     B is FP32   (Eq. 9)      */
#define HEAL_MODE_4P 4u        /* 3P + lo.lo (diagnostic)   B is FP32                              */
#define HEAL_B_NK 0x10u        /* B is stored N x K (K contiguous) -- the paper's W^T /
                                  nn.Linear layout; default is K x N (N contiguous) */
#define HEAL_B_STATIC 0x20u    /* promise: B (static weights, the inference case) is not written by the
                                  operations enqueued on `stream` just before this call.  The kernel may
                                  then start streaming B while its stream predecessor is still finishing
                                  (programmatic dependent launch); everything that reads A or writes C
                                  still waits for the predecessor.  Same bits with or without the flag.  Ignored by
                                  heal_gemm in the FP32-B modes (3P/4P), whose B planes are produced on the fly. */

#define HEAL_EPI_SILU_MUL 0x80u   /* step E fused with the MLP activation of Algorithm 1, "SiLU(g) (.) u" (SURVEY.md 8(f)
                                     NEXT-3): the GEMM's N columns are (gate, up) pairs -- column 2j = g_j, column 2j+1 = u_j, i.e.
                                     the gate and up projection weights interleaved column-wise -- N must be even, and every
                                     output (C, C_hi/C_lo) is M x N/2 and receives  g_j / (1 + exp(-g_j)) * u_j  computed in FP32
                                     from the (2^-scale_exp scaled) GEMM results; with C_hi/C_lo this is the activation of the down
                                     projection, already split for heal_gemm_presplit.  ldc, ldc16 >= N/2. */
#define HEAL_EPI_ACCUMULATE 0x100u /* step E fused with the residual add of Algorithm 1, "A_i + GEMM(...)" (FP32 residual
                                     flow): C must hold the residual on entry and receives C + result (one FP32 RN add
                                     per element); the planes, if requested, are the split of that sum.  Needs C. */

#define HEAL_FUSE_SPLIT 0x200u     /* heal_gemm / heal_gemm_ex, M > 128, N > 128, two or three products: step S of the activations runs
                                     inside the GEMM kernel (FP32 tiles by TMA, converted in place in shared memory; SURVEY.md 8(f)
                                     NEXT-1(i)) -- no hi/lo planes in HBM, no workspace and one launch with FP16 weights.  Same bits.
                                     Slower than split + GEMM on B200 (0-13 %), hence opt-in; the library also
                                     takes this path by itself when a captured call finds no workspace.  Ignored elsewhere. */

#define HEAL_LO_SHIFT 10
#define HEAL_LO_SCALED 0x40u   /* the paper's scaled residual, Eq. 10 as printed: h = h_hi + h_lo / 2^10 with
                                  h_lo = r16((h - h_hi) * 2^10), C = GEMM(h_hi, W) + GEMM(h_lo / 2^10, W).  Two-product mode only.  One
                                  kernel, one accumulator: inside every 512-long K segment the tensor core first accumulates the h_lo.W
                                  products (k ascending), then scales that sum by 2^-10 (tcgen05.mma scale_input_d, an exact power of two)
                                  as it adds the first h_hi.W product, then accumulates the remaining h_hi.W products; segment sums are
                                  added in FP32 RN in ascending order as always.  Differs from the default (s = 0) only where h_lo would
                                  leave FP16's normal range, i.e. for |h| < 2^-3 (reading A1).  The weight tile travels twice per
                                  segment: about 8 % slower than the default on prefill shapes, 1.3-1.5x on decode shapes (M <= 32: the
                                  small-M kernel's form of the same two passes, second weight read out of L2; same bits for every M).  With
                                  heal_gemm_presplit(_ex) A_lo must hold the scaled residual (heal_split_scaled with lo_shift = 10). */

/*
 * C[M x N] (FP32) = A[M x K] (FP32) . B          one pass of the whole path: split, MMAs, epilogue.
 *   A    FP32, lda >= K elements; 16-byte aligned, lda % 4 == 0.  Read-only.
 *   B    FP16 (modes 1P, 2P) or FP32 (modes 3P, 4P).  K x N with ldb >= N, or N x K with ldb >= K
 *        if HEAL_B_NK.  16-byte aligned; ldb % 8 == 0 (FP16) / ldb % 4 == 0 (FP32).  Read-only.
 *   C    FP32, ldc >= N, 16-byte aligned, ldc % 4 == 0.  Overwritten (no beta).  Must not alias A/B.
 *   M == 0 or N == 0: no-op, HEAL_OK.  K == 0: C is zero-filled.
 * Ownership: the caller owns A, B, C and keeps them alive until `stream` has passed the call.  The
 * hi/lo planes live in a library-owned workspace -- one per stream (up to 8 streams; beyond that the
 * least recently used one is recycled after a device synchronise), grown on first use, so calls on
 * different streams may run concurrently.  A caller-supplied workspace (heal_set_workspace) is
 * shared by all streams: calls that use it must be issued on one stream at a time.  During stream
 * capture the library does not allocate: run the call once eagerly on that stream first (or supply
 * a workspace); a captured call that finds none returns HEAL_ERR_WORKSPACE, except for the shapes of HEAL_FUSE_SPLIT, which
 * then split inside the GEMM kernel.  Buffers that a captured graph may hold are never freed or handed to another stream.
 * With FP16 weights and decode-sized M (M <= 16 with K <= 16384; M <= 32 for problems of up to 32 Mi weights) the split
 * runs inside the GEMM kernel -- one launch, no workspace -- wherever that is the faster form: not for very wide weight
 * matrices (N of about 26 500 columns or more with K >= 2048, e.g. the LM head), which take split + GEMM on planes like larger M
 * (unless the call is being captured on a stream without a workspace: then the fused kernel, not HEAL_ERR_WORKSPACE).
 * Numerical contract: finite inputs with |x| <= 65504 (activations observed
 * < 1024); anything larger, Inf or NaN propagates to Inf/NaN in the affected rows/columns.
 */
int heal_gemm(int64_t M, int64_t N, int64_t K,
              const void *A, int64_t lda,
              const void *B, int64_t ldb,
              void *C, int64_t ldc,
              uint32_t mode, void *stream);

/*
 * Step S alone: hi[r][c] = r16(X[r][c]), lo[r][c] = r16(X[r][c] - hi[r][c]).
 *   X      FP32 rows x cols, ldx >= cols
 *   hi,lo  FP16 rows x cols, leading dimension ld >= cols (elements)
 * All pointers 16-byte aligned; ldx % 4 == 0 and ld % 8 == 0.  Used by tests and to pre-split
 * static FP32 weights once (three-product mode).
 */
int heal_split(int64_t rows, int64_t cols, const void *X, int64_t ldx,
               void *hi, void *lo, int64_t ld, void *stream);

/* Step S with a scaled residual: lo[r][c] = r16((X[r][c] - hi[r][c]) * 2^lo_shift), 0 <= lo_shift <= 16
 * (PAPER.md:203 uses 10).  heal_split(...) == heal_split_scaled(..., 0, stream). */
int heal_split_scaled(int64_t rows, int64_t cols, const void *X, int64_t ldx,
                      void *hi, void *lo, int64_t ld, int32_t lo_shift, void *stream);

/*
 * Norm -> step S in one pass ("GEMM(Norm(H_i), W)"; FP32 normalization): RMSNorm of
 * every row of X in FP32,   y[r][c] = (X[r][c] * rstd_r) * gamma[c],   rstd_r = 1 / sqrt(mean_c X[r][c]^2 + eps),
 * immediately split into hi = r16(y), lo = r16(y - hi) for heal_gemm_presplit -- the normalised FP32 activations are written
 * only if Y != NULL (pitch ldy >= cols, % 4 == 0).  gamma: FP32 vector of `cols` elements, 16-byte aligned, or NULL (= ones).
 * Other arguments as heal_split.  Deterministic: the result of a row does not depend on the other rows or on `rows`.
 */
int heal_rmsnorm_split(int64_t rows, int64_t cols, const void *X, int64_t ldx, const void *gamma, float eps,
                       void *hi, void *lo, int64_t ld, void *Y, int64_t ldy, void *stream);

/*
 * Steps G + E on pre-split planes: C = sum of the products `mode` keeps.
 *   A_hi, A_lo   FP16 M x K, leading dimension lda (elements, % 8 == 0).  A_lo may be NULL for 1P.
 *   B_hi, B_lo   FP16 K x N (or N x K with HEAL_B_NK), leading dimension ldb (% 8 == 0).
 *                B_lo is ignored (may be NULL) for 1P/2P.
 * Same alignment, aliasing and asynchrony rules as heal_gemm.  Never allocates.
 */
int heal_gemm_presplit(int64_t M, int64_t N, int64_t K,
                       const void *A_hi, const void *A_lo, int64_t lda,
                       const void *B_hi, const void *B_lo, int64_t ldb,
                       void *C, int64_t ldc,
                       uint32_t mode, void *stream);

/*
 * Extended epilogue (step E options):
 *   scale_exp   the result is multiplied by 2^-scale_exp before it is stored -- the inverse of the
 *               per-weight-matrix power-of-two scale 2^p the paper applies to the weights before the
 *               GEMM ("invert the scale after the GEMM output").  Exact (a power of two)
 *               unless the product leaves the FP32 normal range.  -126 <= scale_exp <= 126; 0 = none.
 *   C_hi, C_lo  optional FP16 M x N planes (leading dimension ldc16 >= N elements, % 8 == 0, 16-byte
 *               aligned; both or neither): the chained output -- hi = r16(c), lo = r16(c - hi) of every
 *               scaled result c, i.e. exactly heal_split() of the FP32 output, written by
 *               the GEMM epilogue so that the next compensated GEMM (heal_gemm_presplit) needs no pass
 *               over C.
 *   C           may be NULL when the planes are requested (then ldc is ignored); otherwise as heal_gemm.
 * Everything else as heal_gemm / heal_gemm_presplit; heal_gemm(...) == heal_gemm_ex(..., NULL, NULL, 0, 0, ...).
 */
int heal_gemm_ex(int64_t M, int64_t N, int64_t K,
                 const void *A, int64_t lda,
                 const void *B, int64_t ldb,
                 void *C, int64_t ldc,
                 void *C_hi, void *C_lo, int64_t ldc16, int32_t scale_exp,
                 uint32_t mode, void *stream);

int heal_gemm_presplit_ex(int64_t M, int64_t N, int64_t K,
                          const void *A_hi, const void *A_lo, int64_t lda,
                          const void *B_hi, const void *B_lo, int64_t ldb,
                          void *C, int64_t ldc,
                          void *C_hi, void *C_lo, int64_t ldc16, int32_t scale_exp,
                          uint32_t mode, void *stream);

/*
 * HOST-buffer variant of heal_gemm: A, B, C are HOST pointers (ideally pinned).  Copies A and B to
 * the device, runs the path, copies C back and synchronises `stream` before returning.  Same
 * layout rules as heal_gemm except that alignment applies to the internal device copies only.
 * Staging buffers are library-owned and reused between calls.  Large problems are pipelined over blocks of
 * weight columns on two library-owned copy streams (weights in while the previous block computes and the one
 * before travels out), with bit-identical results; calls are serialised inside the library.
 */
int heal_gemm_host(int64_t M, int64_t N, int64_t K,
                   const void *A_host, int64_t lda,
                   const void *B_host, int64_t ldb,
                   void *C_host, int64_t ldc,
                   uint32_t mode, void *stream);

/*
 * The inference form of the host variant: activations in, results out, WEIGHTS RESIDENT on the device.  A and C are HOST pointers
 * (ideally pinned), B is a DEVICE pointer with the layout and alignment rules of heal_gemm.  Pipelined over blocks of 512 token rows
 * on the library's two copy streams (activations in, compute, results out overlap); bit-identical to heal_gemm over all rows (the
 * reduction order does not depend on M).  Synchronises `stream` before returning; calls are serialised inside the library.
 */
int heal_gemm_host_act(int64_t M, int64_t N, int64_t K,
                       const void *A_host, int64_t lda,
                       const void *B, int64_t ldb,
                       void *C_host, int64_t ldc,
                       uint32_t mode, void *stream);

/*
 * heal_gemm for callers that must not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc.  Same operation and same bits as heal_gemm (split, two-product MMA, FP32 epilogue), restricted to
 * decode-sized problems, with every byte of scratch -- the hi/lo FP16 planes of A (step S) and the kernels' diagnostic words -- in
 * ONE file-scope device array of HEAL_STATIC_SCRATCH_BYTES (+ 256 B) inside the library.  Every GPU that loads the library holds
 * that array until the process exits.  The call makes no cudaMalloc / cudaFree and calls no allocating library routine, also when
 * it is the first call into the library; it launches the split kernel and the small-M GEMM kernel on `stream` and returns.
 *   A, B, C, lda, ldb, ldc, stream: as for heal_gemm (DEVICE pointers, same alignment rules); B is FP16.
 *   mode: HEAL_MODE_1P or HEAL_MODE_2P, optionally | HEAL_B_NK | HEAL_B_STATIC; anything else: HEAL_ERR_UNSUPPORTED_MODE.
 *   Limits: M <= HEAL_STATIC_MAX_M and 2 * roundup(M * roundup(K, 8) * 2, 256) <= HEAL_STATIC_SCRATCH_BYTES (every M <= 64 up to
 *   K = 32768); beyond either, and for the few shapes the small-M kernel leaves to the large-M kernels, HEAL_ERR_WORKSPACE and
 *   nothing is launched.
 *   Sharing: all calls, on all streams, use the same array.  Calls that overlap on the GPU (different streams without an ordering
 *   between them, or graphs replayed concurrently) RACE on the planes and give wrong results; calls on one stream, or otherwise
 *   ordered, are safe.  The array keeps the previous call's planes; nothing in it needs clearing between calls (each call rewrites
 *   the part it reads; the diagnostic words are zero from module load and change only when a kernel traps).
 */
#define HEAL_STATIC_SCRATCH_BYTES (8u << 20)
#define HEAL_STATIC_MAX_M 64
int heal_gemm_static(int64_t M, int64_t N, int64_t K,
                     const void *A, int64_t lda,
                     const void *B, int64_t ldb,
                     void *C, int64_t ldc,
                     uint32_t mode, void *stream);

/* Bytes of workspace heal_gemm needs for this problem (hi/lo planes of A, and of B in 3P/4P). */
size_t heal_workspace_size(int64_t M, int64_t N, int64_t K, uint32_t mode);

/*
 * Hand the library a caller-owned device workspace (256-byte aligned) so that heal_gemm never
 * allocates; it must stay valid until replaced.  (NULL, 0) returns to the library-owned,
 * lazily-grown workspace.  heal_gemm returns HEAL_ERR_WORKSPACE if a supplied one is too small.
 */
int heal_set_workspace(void *ptr, size_t bytes);

/* Number of kernels heal_* calls have launched in this process (split + GEMM), for accounting. */
uint64_t heal_launch_count(void);

/*
 * Debug hook: force the kernel family regardless of shape.  0 = automatic (default), 1 = large-M kernels
 * even for M <= 64, 2 = small-M kernel whenever M <= 64 (the default rule), 3 = single-CTA large-M kernel
 * instead of CTA pairs.  Results are bit-identical whichever kernel runs; only speed changes.
 */
int heal_debug_force_kernel(int which);

/* Name (static string) of the GEMM kernel instantiation the calling thread's most recent heal_gemm* call launched, e.g.
 * "heal_gemm_umma2_kernel<256,2P,KxN,cta_group::2>"; "none" before the first launch.  For reports (bench.py). */
const char *heal_last_kernel(void);

/* Library version: major * 10000 + minor * 100 + patch. */
int heal_version(void);

/* The cudaError_t (as int) of the most recent failing CUDA call made by this library, 0 if none. */
int heal_last_cuda_error(void);

/* Static, NUL-terminated description of a heal_status. */
const char *heal_status_string(int status);

#ifdef __cplusplus
}
#endif
#endif /* HEAL_H_ */
