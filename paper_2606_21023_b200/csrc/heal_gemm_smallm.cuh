// heal_gemm_smallm.cuh -- steps G + E for small M (decode / LM-head shapes, M <= 64): the weight
// matrix is streamed once from HBM and is the tensor core's 128-row operand ("swap-AB"), the few
// token rows are the UMMA N side (16/32/64), and the K segments of one 128-column weight panel are
// spread over the CTAs of a thread-block cluster so that enough CTAs stream HBM.
//
// Same reduction order as heal_gemm_umma.cuh (include/heal.h): inside a 512-long K segment the tensor
// core accumulates k16 slices in ascending k, products hi.hi, hi.lo, lo.hi, lo.lo; the segment partial
// sums are then added in ascending segment order in FP32 RN -- here by a distributed reduction over
// the cluster's shared memory (DSMEM), no atomics.  Results are bit-identical to the large-M kernel.
//
// Cluster of CS CTAs = one 128-column panel; CTA rank r owns segments r, r+CS, r+2CS, ... (local slot
// j = s / CS lives in TMEM columns j*MPAD..).  Roles per CTA (192 threads): warp 0 TMA producer,
// warp 1 MMA issuer + TMEM allocator, warps 2-5 epilogue (warp w owns TMEM lanes 32*(w%4)..+31).
#pragma once
#include "heal_ptx.cuh"

namespace heal {

constexpr int kSmallThreads = 192;
constexpr int kSmallBNW = 128;          // weight columns per panel (UMMA M)

__device__ __forceinline__ uint32_t map_to_cta(uint32_t saddr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
__device__ __forceinline__ float ld_dsmem_f32(uint32_t addr)
{
    float v;
    asm volatile("ld.shared::cluster.f32 %0, [%1];" : "=f"(v) : "r"(addr) : "memory");
    return v;
}

template <int MPAD_, int NPROD_, bool B_MN_>
struct SmallCfg {
    static constexpr int MPAD = MPAD_;                  // UMMA N: padded token count
    static constexpr int NPROD = NPROD_;
    static constexpr bool B_MN = B_MN_;                 // weights stored K x N (N contiguous)
    static constexpr int A_PLANES = NPROD >= 2 ? 2 : 1; // activation planes
    static constexpr int B_PLANES = NPROD >= 3 ? 2 : 1; // weight planes
    static constexpr int W_TILE = kSmallBNW * kBK * 2;  // 16 KB
    static constexpr int X_TILE = MPAD * kBK * 2;
    static constexpr int X_TILE_AL = (X_TILE + 1023) / 1024 * 1024;
    static constexpr int STAGE_BYTES = B_PLANES * W_TILE + A_PLANES * X_TILE_AL;
    static constexpr int STAGES = (96 * 1024 / STAGE_BYTES) < 2 ? 2 : (96 * 1024 / STAGE_BYTES) > 8 ? 8 : (96 * 1024 / STAGE_BYTES);
    static constexpr int BAR_BYTES = 256;
    static_assert(MPAD % 16 == 0 && MPAD >= 16 && MPAD <= 64, "MPAD");
};

struct SmallArgs {
    float *C;
    int64_t ldc;
    int M, N, K;
    int n_seg;            // ceil(K / 512)
    int max_local;        // ceil(n_seg / CS)
    int tmem_cols;        // power of two >= max(32, max_local * MPAD)
    int *diag;
};

template <class Cfg>
__global__ void __launch_bounds__(kSmallThreads)
heal_gemm_smallm_kernel(const __grid_constant__ CUtensorMap tm_x_hi, const __grid_constant__ CUtensorMap tm_x_lo,
                        const __grid_constant__ CUtensorMap tm_w_hi, const __grid_constant__ CUtensorMap tm_w_lo,
                        const SmallArgs args)
{
    constexpr int MPAD = Cfg::MPAD, NPROD = Cfg::NPROD, STAGES = Cfg::STAGES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    // layout: [pipeline stages | aliased after the main loop by the segment staging area][barriers]
    const uint32_t pipe_bytes = STAGES * Cfg::STAGE_BYTES;
    const uint32_t cs = cluster_nctarank();
    const uint32_t rank = cluster_ctarank();
    const uint32_t stage_area = cs > 1 ? static_cast<uint32_t>(args.max_local) * MPAD * kSmallBNW * 4 : 0u;
    const uint32_t bar_base = smem_base + (pipe_bytes > stage_area ? pipe_bytes : stage_area);
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
    const uint32_t done_bar = bar_base + 8u * (2 * STAGES);
    const uint32_t tmem_slot = bar_base + 8u * (2 * STAGES + 1);
    volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int panel = blockIdx.x / cs;
    const int n0 = panel * kSmallBNW;
    const int k_tiles = (args.K + kBK - 1) / kBK;
    const int n_local = (args.n_seg > static_cast<int>(rank)) ? (args.n_seg - 1 - static_cast<int>(rank)) / static_cast<int>(cs) + 1 : 0;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tm_x_hi);
        if (Cfg::A_PLANES == 2) tma_prefetch_desc(&tm_x_lo);
        tma_prefetch_desc(&tm_w_hi);
        if (Cfg::B_PLANES == 2) tma_prefetch_desc(&tm_w_lo);
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(full_bar(s), 1);
            mbar_init(empty_bar(s), 1);
        }
        mbar_init(done_bar, 1);
        fence_mbar_init();
    }
    if (warp == 1) {
        tmem_alloc(tmem_slot, static_cast<uint32_t>(args.tmem_cols));
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;
    pdl_wait();                       // everything above overlapped the previous kernel's tail
    pdl_launch_dependents();

    if (warp == 0) {
        // ================================ TMA producer ================================
        if (lane == 0) {
            const uint64_t pol_w = l2_policy_evict_first();      // weights are streamed once
            int stage = 0;
            uint32_t phase = 0;
            for (int j = 0; j < n_local; ++j) {
                const int seg = static_cast<int>(rank) + j * static_cast<int>(cs);
                const int kt_end = min(k_tiles, (seg + 1) * kTilesPerSeg);
                for (int kt = seg * kTilesPerSeg; kt < kt_end; ++kt) {
                    mbar_wait(empty_bar(stage), phase ^ 1u, args.diag, 500 + stage);
                    const uint32_t sb = smem_base + stage * Cfg::STAGE_BYTES;
                    const uint32_t fb = full_bar(stage);
                    mbar_arrive_expect_tx(fb, Cfg::B_PLANES * Cfg::W_TILE + Cfg::A_PLANES * Cfg::X_TILE);
                    const int k0 = kt * kBK;
                    if (Cfg::B_MN) {
#pragma unroll
                        for (int c = 0; c < 2; ++c) {
                            tma_load_2d_hint(sb + c * 8192, &tm_w_hi, fb, n0 + c * 64, k0, pol_w);
                            if (Cfg::B_PLANES == 2)
                                tma_load_2d_hint(sb + Cfg::W_TILE + c * 8192, &tm_w_lo, fb, n0 + c * 64, k0, pol_w);
                        }
                    } else {
                        tma_load_2d_hint(sb, &tm_w_hi, fb, k0, n0, pol_w);
                        if (Cfg::B_PLANES == 2) tma_load_2d_hint(sb + Cfg::W_TILE, &tm_w_lo, fb, k0, n0, pol_w);
                    }
                    const uint32_t sx = sb + Cfg::B_PLANES * Cfg::W_TILE;
                    tma_load_2d(sx, &tm_x_hi, fb, k0, 0);
                    if (Cfg::A_PLANES == 2) tma_load_2d(sx + Cfg::X_TILE_AL, &tm_x_lo, fb, k0, 0);
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ================================ MMA issuer ==================================
        if (lane == 0) {
            // D[n][m] = sum_k W[k][n] * X[m][k]: UMMA A = weights (128 rows), UMMA B = tokens (N = MPAD)
            constexpr uint32_t idesc = umma_idesc_f16_f32(kSmallBNW, MPAD, Cfg::B_MN ? 1u : 0u, 0u);
            constexpr uint64_t kdesc0 = umma_smem_desc_sw128(0, 16, 1024);                 // K-major SW128
            constexpr uint64_t wdesc0 = Cfg::B_MN ? umma_smem_desc_sw128(0, kBK * 128, 1024) : kdesc0;
            constexpr uint32_t w_step = (Cfg::B_MN ? 16 * 128 : 32) >> 4;
            constexpr uint32_t x_step = 32 >> 4;
            int stage = 0;
            uint32_t phase = 0;
            for (int j = 0; j < n_local; ++j) {
                const int seg = static_cast<int>(rank) + j * static_cast<int>(cs);
                const int kt_end = min(k_tiles, (seg + 1) * kTilesPerSeg);
                const uint32_t d_tmem = tmem_base + static_cast<uint32_t>(j * MPAD);
                uint32_t accumulate = 0;
                for (int kt = seg * kTilesPerSeg; kt < kt_end; ++kt) {
                    mbar_wait(full_bar(stage), phase, args.diag, 600 + stage);
                    tc_fence_after();
                    const uint32_t sb = smem_base + stage * Cfg::STAGE_BYTES;
                    const uint64_t w_hi = wdesc0 | desc_addr(sb);
                    const uint64_t w_lo = wdesc0 | desc_addr(sb + Cfg::W_TILE);
                    const uint32_t sx = sb + Cfg::B_PLANES * Cfg::W_TILE;
                    const uint64_t x_hi = kdesc0 | desc_addr(sx);
                    const uint64_t x_lo = kdesc0 | ((sx + Cfg::X_TILE_AL) >> 4);
#pragma unroll
                    for (int q = 0; q < kBK / 16; ++q) {
                        const uint64_t wo = static_cast<uint64_t>(q * w_step), xo = static_cast<uint64_t>(q * x_step);
                        // product order as in the large-M kernel: a_hi.b_hi, a_hi.b_lo, a_lo.b_hi, a_lo.b_lo
                        umma_f16(d_tmem, w_hi + wo, x_hi + xo, idesc, accumulate);
                        accumulate = 1;
                        if (NPROD == 2) umma_f16(d_tmem, w_hi + wo, x_lo + xo, idesc, 1);
                        if (NPROD >= 3) {
                            umma_f16(d_tmem, w_lo + wo, x_hi + xo, idesc, 1);
                            umma_f16(d_tmem, w_hi + wo, x_lo + xo, idesc, 1);
                        }
                        if (NPROD == 4) umma_f16(d_tmem, w_lo + wo, x_lo + xo, idesc, 1);
                    }
                    umma_commit(empty_bar(stage));
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
            }
            umma_commit(done_bar);                         // all local segments complete in TMEM
        }
    } else {
        // ================================ epilogue: TMEM -> staging ======================
        const int quad = warp & 3;
        const int nl = quad * 32 + lane;                   // weight column within the panel = TMEM lane
        mbar_wait(done_bar, 0, args.diag, 700);
        tc_fence_after();
        if (cs == 1) {
            // single-CTA panel: all segments are local slots; sum them in ascending order in registers
            const int col = n0 + nl;
#pragma unroll
            for (int c = 0; c < MPAD / 16; ++c) {
                if (c * 16 < args.M) {
                    const uint32_t taddr = tmem_base + (static_cast<uint32_t>(quad * 32) << 16) + static_cast<uint32_t>(c * 16);
                    uint32_t v[16];
                    float acc[16];
                    tmem_ld_32x32b_x16(taddr, v);
                    tmem_ld_wait();
#pragma unroll
                    for (int i = 0; i < 16; ++i) acc[i] = __uint_as_float(v[i]);
                    for (int j = 1; j < n_local; ++j) {
                        tmem_ld_32x32b_x16(taddr + static_cast<uint32_t>(j * MPAD), v);
                        tmem_ld_wait();
#pragma unroll
                        for (int i = 0; i < 16; ++i) acc[i] = __fadd_rn(acc[i], __uint_as_float(v[i]));
                    }
                    if (col < args.N) {
#pragma unroll
                        for (int i = 0; i < 16; ++i)
                            if (c * 16 + i < args.M) args.C[static_cast<int64_t>(c * 16 + i) * args.ldc + col] = acc[i];
                    }
                }
            }
        } else {
            // the pipeline buffers are dead now (every TMA load has been consumed by a completed MMA)
            for (int j = 0; j < n_local; ++j) {
#pragma unroll
                for (int c = 0; c < MPAD / 16; ++c) {
                    uint32_t v[16];
                    tmem_ld_32x32b_x16(tmem_base + (static_cast<uint32_t>(quad * 32) << 16) + static_cast<uint32_t>(j * MPAD + c * 16), v);
                    tmem_ld_wait();
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        const uint32_t off = (static_cast<uint32_t>(j * MPAD + c * 16 + i) * kSmallBNW + nl) * 4u;
                        asm volatile("st.shared.b32 [%0], %1;" ::"r"(smem_base + off), "r"(v[i]) : "memory");
                    }
                }
            }
        }
        tc_fence_before();
    }

    if (cs > 1) {
        // ---- every CTA's segment partials are staged: reduce over the cluster in ascending segment order
        __syncwarp();
        cluster_sync_all();
        if (warp >= 2) {
            const int nl = (warp & 3) * 32 + lane;
            const int col = n0 + nl;
            for (int m = static_cast<int>(rank); m < args.M; m += static_cast<int>(cs)) {
                float acc = 0.f;
#pragma unroll 8
                for (int s = 0; s < args.n_seg; ++s) {
                    const uint32_t src = static_cast<uint32_t>(s) % cs, slot = static_cast<uint32_t>(s) / cs;
                    const uint32_t off = ((slot * MPAD + static_cast<uint32_t>(m)) * kSmallBNW + nl) * 4u;
                    const float v = ld_dsmem_f32(map_to_cta(smem_base + off, src));
                    acc = (s == 0) ? v : __fadd_rn(acc, v);
                }
                if (col < args.N) args.C[static_cast<int64_t>(m) * args.ldc + col] = acc;
            }
        }
        __syncwarp();
        cluster_sync_all();                                 // nobody leaves while its smem is being read
    } else {
        __syncthreads();
    }
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tmem_base, static_cast<uint32_t>(args.tmem_cols));
    }
}

}  // namespace heal
