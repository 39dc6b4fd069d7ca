// mc_delivery.cu -- measurement probe (not part of libheal.so): L2 -> SM operand delivery rate with L2-resident data,
// every CTA loading its own tiles (unicast) versus clusters of 2 / 4 CTAs sharing each tile through TMA multicast.
// "delivered" counts the bytes that land in shared memory, summed over the SMs.  Built and run by
// `python -m paper_2606_21023_b200.probes`; results quoted in DESIGN.md section 7.
#include <cuda.h>
#include <cudaTypedefs.h>
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <cstdio>
#include "../csrc/heal_ptx.cuh"
using namespace heal;

__device__ __forceinline__ void tma_load_2d_mc(uint32_t smem_dst, const CUtensorMap *m, uint32_t bar, int x, int y, uint16_t mask)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1, {%3, %4}], [%2], %5;"
        ::"r"(smem_dst), "l"(reinterpret_cast<uint64_t>(m)), "r"(bar), "r"(x), "r"(y), "h"(mask) : "memory");
}

// tile = 128 rows (k) x 64 cols fp16 = 16 KB as `cs` boxes of (128/cs) rows.  W: rows x 64-col panels.
__global__ void __launch_bounds__(128) k(const __grid_constant__ CUtensorMap tm_full, const __grid_constant__ CUtensorMap tm_part,
                                          int tiles, int stages, int mc, int rows_total, int npanels)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar = base + stages * 16384;
    const uint32_t cs = cluster_nctarank(), rank = cluster_ctarank();
    if (threadIdx.x == 0) {
        for (int s = 0; s < stages; ++s) { mbar_init(bar + 8 * s, 1); mbar_init(bar + 128 + 8 * s, mc ? cs : 1); }
        fence_mbar_init();
    }
    __syncthreads();
    if (cs > 1) cluster_sync_all();
    const int cluster_id = blockIdx.x / cs;
    const int stream_id = mc ? cluster_id : blockIdx.x;           // unicast: every CTA its own stream; mc: one per cluster
    const int panel = stream_id % npanels;
    int row = (stream_id / npanels) * 128 * 7;
    if (threadIdx.x == 0) {
        int stage = 0; uint32_t phase = 0;
        for (int t = 0; t < tiles; ++t) {
            mbar_wait(bar + 128 + 8 * stage, phase ^ 1u, nullptr, 0);
            mbar_arrive_expect_tx(bar + 8 * stage, 16384);
            const int r0 = (row + t * 128) % rows_total;
            if (!mc) {
                tma_load_2d(base + stage * 16384, &tm_full, bar + 8 * stage, panel * 64, r0);
            } else {
                const int pr = 128 / cs;
                tma_load_2d_mc(base + stage * 16384 + rank * pr * 128, &tm_part, bar + 8 * stage, panel * 64, r0 + rank * pr, (uint16_t)((1u << cs) - 1));
            }
            if (++stage == stages) { stage = 0; phase ^= 1u; }
        }
    } else if (threadIdx.x == 32) {
        int stage = 0; uint32_t phase = 0;
        for (int t = 0; t < tiles; ++t) {
            mbar_wait(bar + 8 * stage, phase, nullptr, 0);
            if (!mc) mbar_arrive(bar + 128 + 8 * stage);
            else for (uint32_t r = 0; r < cs; ++r) asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(map_to_cta(bar + 128 + 8 * stage, r)) : "memory");
            if (++stage == stages) { stage = 0; phase ^= 1u; }
        }
    }
    __syncthreads();
    if (cs > 1) cluster_sync_all();
}

int main()
{
    const int ROWS = 8192, COLS = 2048;      // 32 MB fp16: L2 resident
    __half *W; cudaMalloc(&W, (size_t)ROWS * COLS * 2); cudaMemset(W, 1, (size_t)ROWS * COLS * 2);
    void *fn; cudaDriverEntryPointQueryResult q;
    cudaGetDriverEntryPointByVersion("cuTensorMapEncodeTiled", &fn, 12000, cudaEnableDefault, &q);
    auto enc = (PFN_cuTensorMapEncodeTiled_v12000)fn;
    auto mk = [&](CUtensorMap *tm, int box_rows) {
        cuuint64_t dims[2] = {(cuuint64_t)COLS, (cuuint64_t)ROWS}; cuuint64_t strides[1] = {(cuuint64_t)COLS * 2};
        cuuint32_t box[2] = {64, (cuuint32_t)box_rows}; cuuint32_t es[2] = {1, 1};
        enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, W, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    };
    cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int tiles = 4096;                    // 64 MB delivered per CTA
    for (int cs : {1, 2, 4}) for (int mc = 0; mc < 2; ++mc) {
        if (cs == 1 && mc) continue;
        CUtensorMap tf, tp; mk(&tf, 128); mk(&tp, 128 / cs);
        for (int stages : {4, 8}) {
            const size_t smem = 1024 + stages * 16384 + 512;
            cudaLaunchConfig_t cfg = {}; cfg.gridDim = dim3(148); cfg.blockDim = dim3(128); cfg.dynamicSmemBytes = smem;
            cudaLaunchAttribute at[1]; at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
            cfg.attrs = at; cfg.numAttrs = 1;
            float best = 1e9;
            for (int rep = 0; rep < 3; ++rep) {
                cudaEventRecord(e0);
                cudaLaunchKernelEx(&cfg, k, tf, tp, tiles, stages, mc, ROWS, COLS / 64);
                cudaEventRecord(e1); cudaEventSynchronize(e1);
                float ms; cudaEventElapsedTime(&ms, e0, e1); if (ms < best) best = ms;
            }
            printf("cluster %d %s stages %d: %.1f us, delivered %.0f GB/s (per SM %.1f GB/s) %s\n", cs, mc ? "multicast" : "unicast  ", stages, best * 1e3,
                   148.0 * tiles * 16384 / best / 1e6, tiles * 16384.0 / best / 1e6, cudaGetErrorString(cudaGetLastError()));
        }
    }
    return 0;
}
