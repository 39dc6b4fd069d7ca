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
    int accumulate;       // C += scaled result (needs C): second launch of the scaled-lo variant, which forms
                          // C = 2^-10 (lo'.W) + hi.W as the paper's two GEMMs summed into one FP32 output
};

// The output mode is uniform for the launch: pick it ONCE per store loop (a per-element test costs a dependent
// constant load + uniform branch, ~100 cycles each -- measured 4 us on a 64-token epilogue) and run the loop body
// with compile-time flags.  f(out, has_c, has_planes) receives the pinned OutArgs and std::integral_constant-like tags.
template <bool V>
struct EmitTag {
    static constexpr bool value = V;
};
// The fields are pinned in registers first: read in place, the compiler re-loads them from the constant bank for every
// element (LDCU -> dependent address math, ~70 cycles per store on a 64-row epilogue, measured).
__device__ __forceinline__ OutArgs pin_out(const OutArgs &o)
{
    OutArgs r = o;
    asm volatile("" : "+l"(r.C), "+l"(r.ldc), "+l"(r.hi), "+l"(r.lo), "+l"(r.ld16), "+f"(r.scale), "+r"(r.accumulate));
    return r;
}
template <class F>
__device__ __forceinline__ void emit_dispatch(const OutArgs &o_, F &&f)
{
    const OutArgs o = pin_out(o_);
    if (o.hi == nullptr) f(o, EmitTag<true>{}, EmitTag<false>{});
    else if (o.C == nullptr) f(o, EmitTag<false>{}, EmitTag<true>{});
    else f(o, EmitTag<true>{}, EmitTag<true>{});
}

// four consecutive columns col..col+3 of one row (col % 4 == 0); columns >= N are not written
template <bool HAS_C, bool HAS_P>
__device__ __forceinline__ void emit4(const OutArgs &o, int64_t row, int col, float4 v, int N)
{
    v.x *= o.scale; v.y *= o.scale; v.z *= o.scale; v.w *= o.scale;
    const bool full = col + 3 < N;
    if (HAS_C) {
        float *c = o.C + row * o.ldc + col;
        if (o.accumulate) {
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
    if (HAS_P) {
        uint2 h, l;
        split2(v.x, v.y, h.x, l.x);
        split2(v.z, v.w, h.y, l.y);
        __half *ph = o.hi + row * o.ld16 + col, *pl = o.lo + row * o.ld16 + col;
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

// one element (the small-M kernel: a warp's lanes are consecutive columns of one row)
template <bool HAS_C, bool HAS_P>
__device__ __forceinline__ void emit1(const OutArgs &o, int64_t row, int col, float v)
{
    v *= o.scale;
    if (HAS_C) {
        if (o.accumulate) v = __fadd_rn(o.C[row * o.ldc + col], v);
        o.C[row * o.ldc + col] = v;
    }
    if (HAS_P) {
        const __half h = __float2half_rn(v);
        o.hi[row * o.ld16 + col] = h;
        o.lo[row * o.ld16 + col] = __float2half_rn(__fsub_rn(v, __half2float(h)));
    }
}

}  // namespace heal
