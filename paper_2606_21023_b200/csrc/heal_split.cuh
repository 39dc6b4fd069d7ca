// heal_split.cuh -- step S of the HEAL compensated GEMM: FP32 -> (hi, lo) FP16 planes,
//     hi = r16(x),  lo = r16(x - hi)          (s = 0 reading, A1)
// r16 = cvt.rn.f16.f32 (round-to-nearest-even, subnormals kept).  x - float(hi) is
// exact in FP32.  HBM-bound: 4 B read + 4 B written per element; 128-bit loads and stores.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace heal {

__device__ __forceinline__ void split2(float x0, float x1, uint32_t &hi, uint32_t &lo)
{
    const __half h0 = __float2half_rn(x0), h1 = __float2half_rn(x1);
    const __half l0 = __float2half_rn(__fsub_rn(x0, __half2float(h0)));
    const __half l1 = __float2half_rn(__fsub_rn(x1, __half2float(h1)));
    hi = static_cast<uint32_t>(__half_as_ushort(h0)) | (static_cast<uint32_t>(__half_as_ushort(h1)) << 16);
    lo = static_cast<uint32_t>(__half_as_ushort(l0)) | (static_cast<uint32_t>(__half_as_ushort(l1)) << 16);
}

// scaled residual (the paper's h = h_hi + h_lo / 2^s): lo = r16((x - hi) * 2^s); the product is exact
__device__ __forceinline__ void split2s(float x0, float x1, uint32_t &hi, uint32_t &lo, float lo_scale)
{
    const __half h0 = __float2half_rn(x0), h1 = __float2half_rn(x1);
    const __half l0 = __float2half_rn(__fmul_rn(__fsub_rn(x0, __half2float(h0)), lo_scale));
    const __half l1 = __float2half_rn(__fmul_rn(__fsub_rn(x1, __half2float(h1)), lo_scale));
    hi = static_cast<uint32_t>(__half_as_ushort(h0)) | (static_cast<uint32_t>(__half_as_ushort(h1)) << 16);
    lo = static_cast<uint32_t>(__half_as_ushort(l0)) | (static_cast<uint32_t>(__half_as_ushort(l1)) << 16);
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
