// heal_split.cuh -- step S of the HEAL compensated GEMM: FP32 -> (hi, lo) FP16 planes,
//     hi = r16(x),  lo = r16(x - hi)          (s = 0 reading, A1)
// r16 = cvt.rn.f16.f32 (round-to-nearest-even, subnormals kept).  x - float(hi) is
// exact in FP32.  HBM-bound: 4 B read + 4 B written per element; 128-bit loads and stores.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace heal {

// Two elements at a time with the packed conversion (cvt.rn.f16x2.f32 = one F2FP.PACK_AB instead of two F2F: the single
// conversions run on the slow conversion unit and made the in-GEMM converters the bottleneck).  Same IEEE round-to-nearest-
// even, subnormals and overflow to Inf as the scalar form -- the exhaustive-range split test covers it.
__device__ __forceinline__ uint32_t pack_f16x2_rn(float lo_elem, float hi_elem)
{
    uint32_t r;
    asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi_elem), "f"(lo_elem));
    return r;
}
__device__ __forceinline__ void split2(float x0, float x1, uint32_t &hi, uint32_t &lo)
{
    hi = pack_f16x2_rn(x0, x1);
    const float2 hf = __half22float2(*reinterpret_cast<const __half2 *>(&hi));
    lo = pack_f16x2_rn(__fsub_rn(x0, hf.x), __fsub_rn(x1, hf.y));
}

// scaled residual (the paper's h = h_hi + h_lo / 2^s): lo = r16((x - hi) * 2^s); the product is exact
__device__ __forceinline__ void split2s(float x0, float x1, uint32_t &hi, uint32_t &lo, float lo_scale)
{
    hi = pack_f16x2_rn(x0, x1);
    const float2 hf = __half22float2(*reinterpret_cast<const __half2 *>(&hi));
    lo = pack_f16x2_rn(__fmul_rn(__fsub_rn(x0, hf.x), lo_scale), __fmul_rn(__fsub_rn(x1, hf.y), lo_scale));
}

// One thread handles 8 consecutive elements of a row (2 x float4 in, 2 x uint4 out); `cols8` =
// ceil(cols / 8) vectors per row; a ragged last vector is handled element-wise.
// Grid-stride over rows * cols8 vectors.
__global__ void __launch_bounds__(256)
heal_split_kernel(const float *__restrict__ X, int64_t ldx, int64_t rows, int64_t cols,
                  __half *__restrict__ hi, __half *__restrict__ lo, int64_t ld, float lo_scale)
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int64_t cols8 = (cols + 7) >> 3;
    const int64_t total = rows * cols8;
    for (int64_t v = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x; v < total;
         v += static_cast<int64_t>(gridDim.x) * blockDim.x) {
        const int64_t r = v / cols8;
        const int64_t c = (v - r * cols8) << 3;
        const float *src = X + r * ldx + c;
        __half *dh = hi + r * ld + c;
        __half *dl = lo + r * ld + c;
        if (c + 8 <= cols) {
            const float4 a = __ldg(reinterpret_cast<const float4 *>(src));
            const float4 b = __ldg(reinterpret_cast<const float4 *>(src) + 1);
            uint4 h, l;
            if (lo_scale == 1.0f) {
                split2(a.x, a.y, h.x, l.x);
                split2(a.z, a.w, h.y, l.y);
                split2(b.x, b.y, h.z, l.z);
                split2(b.z, b.w, h.w, l.w);
            } else {
                split2s(a.x, a.y, h.x, l.x, lo_scale);
                split2s(a.z, a.w, h.y, l.y, lo_scale);
                split2s(b.x, b.y, h.z, l.z, lo_scale);
                split2s(b.z, b.w, h.w, l.w, lo_scale);
            }
            *reinterpret_cast<uint4 *>(dh) = h;
            *reinterpret_cast<uint4 *>(dl) = l;
        } else {
            for (int64_t i = 0; c + i < cols; ++i) {
                const float x = src[i];
                const __half h = __float2half_rn(x);
                dh[i] = h;
                dl[i] = __float2half_rn(__fmul_rn(__fsub_rn(x, __half2float(h)), lo_scale));
            }
        }
    }
}

}  // namespace heal

namespace heal {

// Norm -> step S in one pass ("g, u <- GEMM(Norm(A_i), W_gate_up)"; normalization inputs and
// outputs stay FP32): RMSNorm of every FP32 row,
//     y[k] = (x[k] * rstd) * gamma[k],     rstd = 1 / sqrt(mean_k x[k]^2 + eps)           (all FP32, round-to-nearest),
// followed by the hi/lo split of y -- the FP32 normalised activations never travel to HBM unless the caller
// asks for them (Y != nullptr).  One CTA per row; the sum of squares has a fixed order (thread t accumulates the 8-element
// groups t, t+256, ... in ascending order with FMAs, then a fixed shuffle / shared-memory tree), so the result does not
// depend on M, the grid or the run.  HBM-bound like the split kernel: 4 B read + 4 B written per element (the second
// read of the row hits L1/L2).
__global__ void __launch_bounds__(256)
heal_rmsnorm_split_kernel(const float *__restrict__ X, int64_t ldx, int64_t rows, int64_t cols, const float *__restrict__ gamma,
                          float eps, __half *__restrict__ hi, __half *__restrict__ lo, int64_t ld, float *__restrict__ Y, int64_t ldy)
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    __shared__ float warp_ss[8];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t cols8 = (cols + 7) >> 3;
    for (int64_t r = blockIdx.x; r < rows; r += gridDim.x) {
        const float *src = X + r * ldx;
        float ss = 0.0f;
        for (int64_t v = tid; v < cols8; v += 256) {
            const int64_t c = v << 3;
            if (c + 8 <= cols) {
                const float4 a = __ldg(reinterpret_cast<const float4 *>(src + c));
                const float4 b = __ldg(reinterpret_cast<const float4 *>(src + c) + 1);
                ss = __fmaf_rn(a.x, a.x, ss); ss = __fmaf_rn(a.y, a.y, ss); ss = __fmaf_rn(a.z, a.z, ss); ss = __fmaf_rn(a.w, a.w, ss);
                ss = __fmaf_rn(b.x, b.x, ss); ss = __fmaf_rn(b.y, b.y, ss); ss = __fmaf_rn(b.z, b.z, ss); ss = __fmaf_rn(b.w, b.w, ss);
            } else {
                for (int64_t i = 0; c + i < cols; ++i) ss = __fmaf_rn(src[c + i], src[c + i], ss);
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) ss = __fadd_rn(ss, __shfl_xor_sync(0xffffffffu, ss, o));
        __syncthreads();                                   // warp_ss of the previous row has been read
        if (lane == 0) warp_ss[warp] = ss;
        __syncthreads();
        float tot = warp_ss[0];
#pragma unroll
        for (int w = 1; w < 8; ++w) tot = __fadd_rn(tot, warp_ss[w]);
        const float rstd = __fdiv_rn(1.0f, __fsqrt_rn(__fadd_rn(__fdiv_rn(tot, static_cast<float>(cols)), eps)));
        __half *dh = hi + r * ld, *dl = lo + r * ld;
        float *dy = Y ? Y + r * ldy : nullptr;
        for (int64_t v = tid; v < cols8; v += 256) {
            const int64_t c = v << 3;
            if (c + 8 <= cols) {
                float4 a = __ldg(reinterpret_cast<const float4 *>(src + c));
                float4 b = __ldg(reinterpret_cast<const float4 *>(src + c) + 1);
                float4 ga = make_float4(1.f, 1.f, 1.f, 1.f), gb = ga;
                if (gamma) {
                    ga = __ldg(reinterpret_cast<const float4 *>(gamma + c));
                    gb = __ldg(reinterpret_cast<const float4 *>(gamma + c) + 1);
                }
                a.x = __fmul_rn(__fmul_rn(a.x, rstd), ga.x); a.y = __fmul_rn(__fmul_rn(a.y, rstd), ga.y);
                a.z = __fmul_rn(__fmul_rn(a.z, rstd), ga.z); a.w = __fmul_rn(__fmul_rn(a.w, rstd), ga.w);
                b.x = __fmul_rn(__fmul_rn(b.x, rstd), gb.x); b.y = __fmul_rn(__fmul_rn(b.y, rstd), gb.y);
                b.z = __fmul_rn(__fmul_rn(b.z, rstd), gb.z); b.w = __fmul_rn(__fmul_rn(b.w, rstd), gb.w);
                uint4 h, l;
                split2(a.x, a.y, h.x, l.x);
                split2(a.z, a.w, h.y, l.y);
                split2(b.x, b.y, h.z, l.z);
                split2(b.z, b.w, h.w, l.w);
                *reinterpret_cast<uint4 *>(dh + c) = h;
                *reinterpret_cast<uint4 *>(dl + c) = l;
                if (dy) {
                    *reinterpret_cast<float4 *>(dy + c) = a;
                    *(reinterpret_cast<float4 *>(dy + c) + 1) = b;
                }
            } else {
                for (int64_t i = 0; c + i < cols; ++i) {
                    const float y = __fmul_rn(__fmul_rn(src[c + i], rstd), gamma ? gamma[c + i] : 1.0f);
                    const __half h = __float2half_rn(y);
                    dh[c + i] = h;
                    dl[c + i] = __float2half_rn(__fsub_rn(y, __half2float(h)));
                    if (dy) dy[c + i] = y;
                }
            }
        }
    }
}

}  // namespace heal
