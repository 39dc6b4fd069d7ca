// heal_epilogue.cuh -- step E: what the GEMM kernels do with a finished FP32 sum.
//   * FP32 output ("keep GEMM outputs in FP32");
//   * optional exact power-of-two output scale 2^-p, the inverse of the per-weight-matrix 2^p pre-scale
//     the paper applies before the GEMM;
//   * optional chained output: the hi/lo FP16 planes of the (scaled) result, i.e. step S of the NEXT
//     compensated GEMM done in this epilogue instead of a separate pass over C.
// The planes are exactly heal_split() of the FP32 value this epilogue would store (same split2 code).
#pragma once
#include <cuda_fp16.h>
#include <stdint.h>

#include "heal_split.cuh"

namespace heal {

struct OutArgs {
    float *C;             // FP32 M x N, pitch ldc (elements); may be null when the planes are written
    int64_t ldc;
    __half *hi, *lo;      // FP16 M x N planes, pitch ld16 (elements, % 8 == 0); null = not requested
    int64_t ld16;
    float scale;          // 2^-p, exactly representable; 1.0f = none
    int accumulate;       // C += scaled result (needs C): the residual add "A_i + GEMM(...)" of Algorithm 1 with
                          // C holding A_i (HEAL_EPI_ACCUMULATE)
    int silu;             // HEAL_EPI_SILU_MUL: the GEMM's columns are (gate, up) pairs -- column 2j = g_j, 2j+1 = u_j -- and the
                          // outputs (C and/or planes, N/2 columns wide) receive SiLU(g_j) * u_j
};

// The output mode is uniform for the launch.  The store loops of the kernels are fully unrolled, run once per CTA (cold
// instruction cache) and sit on the latency-critical tail, so their code size matters: the common case -- FP32 output
// only, no accumulate -- is a compile-time FAST path of one multiply and one store per element; everything else
// (chained planes, planes only, the accumulating second launch of the scaled-lo variant) goes through one out-of-line
// function per element.  Measured on a 64-row small-M epilogue: 4.1 us with per-element mode tests, 2.3 us with three
// inlined variants, see DESIGN.md for the current figure.
template <bool V>
struct EmitTag {
    static constexpr bool value = V;
};
// The fields are pinned in registers first: read in place, the compiler re-loads them from the constant bank for every
// element.
__device__ __forceinline__ OutArgs pin_out(const OutArgs &o)
{
    OutArgs r = o;
    asm volatile("" : "+l"(r.C), "+l"(r.ldc), "+l"(r.hi), "+l"(r.lo), "+l"(r.ld16), "+f"(r.scale), "+r"(r.accumulate), "+r"(r.silu));
    return r;
}
// f(out, fast): `fast` is EmitTag<true> when only the FP32 matrix is written and nothing is accumulated
template <class F>
__device__ __forceinline__ void emit_dispatch(const OutArgs &o_, F &&f)
{
    const OutArgs o = pin_out(o_);
    if (o.hi == nullptr && o.accumulate == 0 && o.silu == 0) f(o, EmitTag<true>{});
    else f(o, EmitTag<false>{});
}

// general forms, out of line, arguments by value (the caller's OutArgs stays in registers); v is already scaled
// SiLU(g) * u in FP32: g / (1 + exp(-g)) * u with IEEE division (expf: <= 2 ulp; the parity tests bound the result
// against the FP64 definition oracle/heal_fusions.c F2)
__device__ __forceinline__ float silu_mul(float g, float u)
{
    return __fmul_rn(__fdiv_rn(g, __fadd_rn(1.0f, expf(-g))), u);
}

// two output columns col2, col2+1 (col2 even) of one row, N2 output columns in all: FP32 and/or hi/lo planes
__device__ __forceinline__ void emit2_out(float *C, int64_t ldc, __half *hi, __half *lo, int64_t ld16, int accumulate,
                                          int64_t row, int col2, float a, float b, int N2)
{
    const bool full = col2 + 1 < N2;
    if (col2 >= N2) return;
    if (C) {
        float *c = C + row * ldc + col2;
        if (accumulate) {
            a = __fadd_rn(c[0], a);
            if (full) b = __fadd_rn(c[1], b);
        }
        if (full) *reinterpret_cast<float2 *>(c) = make_float2(a, b);
        else c[0] = a;
    }
    if (hi) {
        uint32_t h, l;
        split2(a, b, h, l);
        __half *ph = hi + row * ld16 + col2, *pl = lo + row * ld16 + col2;
        if (full) {
            *reinterpret_cast<uint32_t *>(ph) = h;
            *reinterpret_cast<uint32_t *>(pl) = l;
        } else {
            *reinterpret_cast<uint16_t *>(ph) = static_cast<uint16_t>(h);
            *reinterpret_cast<uint16_t *>(pl) = static_cast<uint16_t>(l);
        }
    }
}

// general forms, out of line, arguments by value (the caller's OutArgs stays in registers); v is already scaled
__device__ __noinline__ void emit4_any(float *C, int64_t ldc, __half *hi, __half *lo, int64_t ld16, int accumulate, int silu,
                                       int64_t row, int col, float4 v, int N)
{
    if (silu) {                                  // columns col..col+3 = (g, u, g, u) -> output columns col/2, col/2 + 1
        emit2_out(C, ldc, hi, lo, ld16, accumulate, row, col >> 1, silu_mul(v.x, v.y), silu_mul(v.z, v.w), N >> 1);
        return;
    }
    const bool full = col + 3 < N;
    if (C) {
        float *c = C + row * ldc + col;
        if (accumulate) {
            if (full) {
                const float4 old = *reinterpret_cast<const float4 *>(c);
                v.x = __fadd_rn(old.x, v.x); v.y = __fadd_rn(old.y, v.y); v.z = __fadd_rn(old.z, v.z); v.w = __fadd_rn(old.w, v.w);
            } else {
                if (col < N) v.x = __fadd_rn(c[0], v.x);
                if (col + 1 < N) v.y = __fadd_rn(c[1], v.y);
                if (col + 2 < N) v.z = __fadd_rn(c[2], v.z);
            }
        }
        if (full) {
            *reinterpret_cast<float4 *>(c) = v;
        } else {
            if (col < N) c[0] = v.x;
            if (col + 1 < N) c[1] = v.y;
            if (col + 2 < N) c[2] = v.z;
        }
    }
    if (hi) {
        uint2 h, l;
        split2(v.x, v.y, h.x, l.x);
        split2(v.z, v.w, h.y, l.y);
        __half *ph = hi + row * ld16 + col, *pl = lo + row * ld16 + col;
        if (full) {
            *reinterpret_cast<uint2 *>(ph) = h;
            *reinterpret_cast<uint2 *>(pl) = l;
        } else {
            const uint16_t hs[4] = {static_cast<uint16_t>(h.x), static_cast<uint16_t>(h.x >> 16),
                                    static_cast<uint16_t>(h.y), static_cast<uint16_t>(h.y >> 16)};
            const uint16_t ls[4] = {static_cast<uint16_t>(l.x), static_cast<uint16_t>(l.x >> 16),
                                    static_cast<uint16_t>(l.y), static_cast<uint16_t>(l.y >> 16)};
#pragma unroll
            for (int i = 0; i < 3; ++i)
                if (col + i < N) {
                    reinterpret_cast<uint16_t *>(ph)[i] = hs[i];
                    reinterpret_cast<uint16_t *>(pl)[i] = ls[i];
                }
        }
    }
}
__device__ __noinline__ void emit1_any(float *C, int64_t ldc, __half *hi, __half *lo, int64_t ld16, int accumulate, int silu,
                                       int64_t row, int col, float v)
{
    if (silu) {
        // small-M kernel: a warp's lanes are consecutive columns of one token, so the (gate, up) pair of output column col/2
        // sits in lanes 2j, 2j+1 (panels start at even columns, N is even: both lanes of a pair are always active together)
        const float other = __shfl_xor_sync(__activemask(), v, 1);
        if (col & 1) return;
        v = silu_mul(v, other);
        col >>= 1;
    }
    if (C) {
        float *c = C + row * ldc + col;
        if (accumulate) v = __fadd_rn(*c, v);
        *c = v;
    }
    if (hi) {
        const __half h = __float2half_rn(v);
        hi[row * ld16 + col] = h;
        lo[row * ld16 + col] = __float2half_rn(__fsub_rn(v, __half2float(h)));
    }
}

// plain FP32 store of four columns (no scale): the kernels' default instantiation
__device__ __forceinline__ void emit4_plain(float *crow, int col, float4 v, int N)
{
    if (col + 3 < N) {
        *reinterpret_cast<float4 *>(crow + col) = v;
    } else {
        if (col < N) crow[col] = v.x;
        if (col + 1 < N) crow[col + 1] = v.y;
        if (col + 2 < N) crow[col + 2] = v.z;
    }
}

// four consecutive columns col..col+3 of one row (col % 4 == 0); columns >= N are not written
template <bool FAST>
__device__ __forceinline__ void emit4(const OutArgs &o, int64_t row, int col, float4 v, int N)
{
    v.x *= o.scale; v.y *= o.scale; v.z *= o.scale; v.w *= o.scale;
    if (FAST) {
        float *c = o.C + row * o.ldc + col;
        if (col + 3 < N) {
            *reinterpret_cast<float4 *>(c) = v;
        } else {
            if (col < N) c[0] = v.x;
            if (col + 1 < N) c[1] = v.y;
            if (col + 2 < N) c[2] = v.z;
        }
    } else {
        emit4_any(o.C, o.ldc, o.hi, o.lo, o.ld16, o.accumulate, o.silu, row, col, v, N);
    }
}

// one element (the small-M kernel: a warp's lanes are consecutive columns of one row)
template <bool FAST>
__device__ __forceinline__ void emit1(const OutArgs &o, int64_t row, int col, float v)
{
    v *= o.scale;
    if (FAST) o.C[row * o.ldc + col] = v;
    else emit1_any(o.C, o.ldc, o.hi, o.lo, o.ld16, o.accumulate, o.silu, row, col, v);
}

}  // namespace heal
