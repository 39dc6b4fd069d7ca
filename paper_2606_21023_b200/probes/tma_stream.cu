// tma_stream.cu -- measurement probe (not part of libheal.so): HBM -> shared-memory streaming rate through TMA.
//   part 1: one long stream (268 MB) as a function of grid size and pipeline stages;
//   part 2: "decode-like": 33.5 MB (one 4096 x 4096 FP16 matrix) per launch, 24 launches over 8 matrices in a CUDA graph
//           with programmatic dependent launch -- once with griddepcontrol.wait before the stream (a kernel that depends
//           on its predecessor: the floor for a decode GEMM of this size) and once without (independent launches overlap).
// Built and run by `python -m paper_2606_21023_b200.probes`; results quoted in DESIGN.md section 7.
#include <cuda.h>
#include <cudaTypedefs.h>
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <cstdio>
#include <cstdlib>
#include <vector>
#include "../csrc/heal_ptx.cuh"
using namespace heal;

// W: K x N fp16 row-major (N contiguous), N = 4096.  Each CTA streams `tiles` tiles of (64 k x 128 cols) = 2 boxes of 64x64
__global__ void __launch_bounds__(128) stream_kernel(const __grid_constant__ CUtensorMap tm, int tiles_per_cta, int stages, int K, int N, int mode, int kbase, int pdl_early,
                                                     const uint4 *raw)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar = base + stages * 16384;
    if (threadIdx.x == 0) {
        for (int s = 0; s < stages; ++s) { mbar_init(bar + 8 * s, 1); mbar_init(bar + 128 + 8 * s, 1); }
        fence_mbar_init();
    }
    __syncthreads();
    if (!pdl_early) pdl_wait();
    pdl_launch_dependents();
    const int panels = N / 128;
    // CTA b: panel = b % panels, k-chunk = b / panels
    const int panel = blockIdx.x % panels, kc = blockIdx.x / panels;
    if (threadIdx.x == 0) {
        int stage = 0; uint32_t phase = 0;
        for (int t = 0; t < tiles_per_cta; ++t) {
            mbar_wait(bar + 128 + 8 * stage, phase ^ 1u, nullptr, 0);
            mbar_arrive_expect_tx(bar + 8 * stage, 16384);
            const int k0 = kbase + (kc * tiles_per_cta + t) * 64;
            if (mode == 0) {
                tma_load_2d(base + stage * 16384, &tm, bar + 8 * stage, panel * 128, k0);
                tma_load_2d(base + stage * 16384 + 8192, &tm, bar + 8 * stage, panel * 128 + 64, k0);
            } else {
                // 1-D bulk copy of 16 KB contiguous
                const char *src = reinterpret_cast<const char *>(raw) + (static_cast<size_t>(blockIdx.x) * tiles_per_cta + t) * 16384;
                asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                             ::"r"(base + stage * 16384), "l"(src), "r"(16384), "r"(bar + 8 * stage) : "memory");
            }
            if (++stage == stages) { stage = 0; phase ^= 1u; }
        }
    } else if (threadIdx.x == 32) {
        int stage = 0; uint32_t phase = 0;
        for (int t = 0; t < tiles_per_cta; ++t) {
            mbar_wait(bar + 8 * stage, phase, nullptr, 0);
            mbar_arrive(bar + 128 + 8 * stage);
            if (++stage == stages) { stage = 0; phase ^= 1u; }
        }
    }
}

int main()
{
    const int K = 4096 * 8, N = 4096;      // 268 MB: 8 distinct 4096x4096 matrices stacked along K
    __half *W; cudaMalloc(&W, (size_t)K * N * 2); cudaMemset(W, 1, (size_t)K * N * 2);
    void *fn; cudaDriverEntryPointQueryResult q;
    cudaGetDriverEntryPointByVersion("cuTensorMapEncodeTiled", &fn, 12000, cudaEnableDefault, &q);
    auto enc = (PFN_cuTensorMapEncodeTiled_v12000)fn;
    CUtensorMap tm;
    cuuint64_t dims[2] = {(cuuint64_t)N, (cuuint64_t)K}; cuuint64_t strides[1] = {(cuuint64_t)N * 2};
    cuuint32_t box[2] = {64, 64}; cuuint32_t es[2] = {1, 1};
    enc(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, W, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
        CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    cudaFuncSetAttribute(stream_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    // total bytes fixed = 4096 x 4096 x 2 x 8 = 268 MB per launch: grid * tiles_per_cta * 16 KB
    const size_t total_tiles = (size_t)K * N * 2 / 16384;   // 16384 tiles
    for (int mode = 0; mode < 1; ++mode)
        for (int grid : {128, 256, 512, 1024, 2048}) {
            for (int stages : {2, 3, 4, 6, 8, 12}) {
                if (total_tiles % grid) continue;
                const int tpc = (int)(total_tiles / grid);
                const size_t smem = 1024 + stages * 16384 + 512;
                if (smem > 200 * 1024) continue;
                float best = 1e9;
                for (int rep = 0; rep < 4; ++rep) {
                    cudaEventRecord(e0);
                    stream_kernel<<<grid, 128, smem>>>(tm, tpc, stages, K, N, mode, 0, 1, reinterpret_cast<const uint4 *>(W));
                    cudaEventRecord(e1); cudaEventSynchronize(e1);
                    float ms; cudaEventElapsedTime(&ms, e0, e1); if (ms < best) best = ms;
                }
                cudaError_t err = cudaGetLastError();
                printf("mode %d grid %4d stages %2d smem %3zu KB: %7.1f us  %6.0f GB/s %s\n", mode, grid, stages, smem / 1024, best * 1e3,
                       (double)K * N * 2 / best / 1e6, err == cudaSuccess ? "" : cudaGetErrorString(err));
            }
        }
    // decode-like: 33.5 MB per launch (one 4096x4096 matrix), 24 launches over 8 matrices in a graph with PDL
    cudaStream_t st; cudaStreamCreate(&st);
    for (int pdl_early = 0; pdl_early < 2; ++pdl_early)
    for (int grid : {128, 256}) for (int stages : {3, 4, 5, 6}) {
        const int tpc = (int)(total_tiles / 8 / grid);
        const size_t smem = 1024 + stages * 16384 + 512;
        cudaGraph_t g; cudaGraphExec_t ge;
        cudaStreamBeginCapture(st, cudaStreamCaptureModeGlobal);
        for (int i = 0; i < 24; ++i) {
            cudaLaunchConfig_t cfg = {}; cfg.gridDim = dim3(grid); cfg.blockDim = dim3(128); cfg.dynamicSmemBytes = smem; cfg.stream = st;
            cudaLaunchAttribute at[1]; at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[0].val.programmaticStreamSerializationAllowed = 1;
            cfg.attrs = at; cfg.numAttrs = 1;
            cudaLaunchKernelEx(&cfg, stream_kernel, tm, tpc, stages, K, N, 0, (i % 8) * 4096, pdl_early, reinterpret_cast<const uint4 *>(W));
        }
        cudaStreamEndCapture(st, &g); cudaGraphInstantiate(&ge, g, 0);
        float best = 1e9;
        for (int rep = 0; rep < 5; ++rep) {
            cudaEventRecord(e0, st); cudaGraphLaunch(ge, st); cudaEventRecord(e1, st); cudaEventSynchronize(e1);
            float ms; cudaEventElapsedTime(&ms, e0, e1); if (ms < best) best = ms;
        }
        printf("decode-like pdl_early %d grid %d stages %d: %.2f us per 33.5 MB launch (%.0f GB/s) %s\n", pdl_early, grid, stages, best * 1e3 / 24,
               33.554432 / (best / 24) , cudaGetErrorString(cudaGetLastError()));
    }
    return 0;
}
