// heal_gemm_umma.cuh -- steps G + E of the HEAL compensated GEMM (Eq. 10; Eq. 9
// PAPER.md:195) for sm_100a: TMA-fed shared-memory stages, mbarrier pipeline, all compensation
// products of a k-slice issued as tcgen05.mma into ONE FP32 accumulator in TMEM, K-segment
// partial sums promoted to an FP32 (RN) register accumulation, FP32 epilogue.
//
// Roles (384 threads, one persistent CTA per SM):
//   warp 0      TMA producer          (one lane)
//   warp 1      MMA issuer            (one lane)
//   warp 2      TMEM allocator
//   warp 3      idle
//   warps 4-11  epilogue: warp w owns TMEM lanes 32*(w%4)..+31 and column half (w-4)/4
//
// Reduction order per output element (see include/heal.h): K segments of 512; inside a segment the
// tensor core accumulates k16 slices in ascending k, products in the order hi.hi, hi.lo, lo.hi,
// lo.lo (those the mode keeps); segments are added in ascending order in FP32 RN.  Nothing here
// depends on M, on the tile an element falls in, or on the SM that computes it.
#pragma once
#include "heal_ptx.cuh"

namespace heal {

constexpr int kBM = 128;          // UMMA M (rows of A per tile)
constexpr int kGemmThreads = 384;

template <int BN_, int NPROD_, bool B_MN_>
struct GemmCfg {
    static constexpr int BN = BN_;
    static constexpr int NPROD = NPROD_;
    static constexpr bool B_MN = B_MN_;                 // B stored K x N (N contiguous): MN-major operand
    static constexpr int A_PLANES = NPROD >= 2 ? 2 : 1;
    static constexpr int B_PLANES = NPROD >= 3 ? 2 : 1;
    static constexpr int A_TILE = kBM * kBK * 2;
    static constexpr int B_TILE = BN * kBK * 2;
    static constexpr int STAGE_BYTES = A_PLANES * A_TILE + B_PLANES * B_TILE;
    static constexpr int BAR_BYTES = 256;
    static constexpr int STAGES_RAW = (kSmemLimit - 1024 - BAR_BYTES) / STAGE_BYTES;
    static constexpr int STAGES = STAGES_RAW > 8 ? 8 : STAGES_RAW;
    static constexpr int SMEM_BYTES = 1024 + STAGES * STAGE_BYTES + BAR_BYTES;
    static constexpr int TMEM_COLS = (2 * BN <= 32) ? 32 : (2 * BN <= 64) ? 64 : (2 * BN <= 128) ? 128 : (2 * BN <= 256) ? 256 : 512;
    static constexpr int COLS_PER_WARP = BN / 2;
    static_assert(BN % 32 == 0 && BN >= 32 && BN <= 256, "BN");
    static_assert(!B_MN || BN % 64 == 0, "MN-major B tiles are built from 64-column swizzle atoms");
    static_assert(STAGES >= 2, "need at least two stages");
};

struct GemmArgs {
    float *C;
    int64_t ldc;
    int M, N, K;
    int tiles_m, tiles_n;
    int *diag;
};

template <class Cfg>
__global__ void __launch_bounds__(kGemmThreads, 1)
heal_gemm_umma_kernel(const __grid_constant__ CUtensorMap tm_a_hi, const __grid_constant__ CUtensorMap tm_a_lo,
                      const __grid_constant__ CUtensorMap tm_b_hi, const __grid_constant__ CUtensorMap tm_b_lo,
                      const GemmArgs args)
{
    constexpr int BN = Cfg::BN, NPROD = Cfg::NPROD, STAGES = Cfg::STAGES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;      // SWIZZLE_128B: 1024-byte aligned stages
    const uint32_t bar_base = smem_base + STAGES * Cfg::STAGE_BYTES;
    // barrier map (8 bytes each): full[STAGES], empty[STAGES], tmem_full[2], tmem_empty[2]; then tmem ptr
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
    auto tfull_bar = [&](int b) { return bar_base + 8u * (2 * STAGES + b); };
    auto tempty_bar = [&](int b) { return bar_base + 8u * (2 * STAGES + 2 + b); };
    const uint32_t tmem_slot = bar_base + 8u * (2 * STAGES + 4);
    volatile uint32_t *tmem_slot_ptr =
        reinterpret_cast<volatile uint32_t *>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int num_tiles = args.tiles_m * args.tiles_n;
    const int k_tiles = (args.K + kBK - 1) / kBK;
    const int n_seg = (k_tiles + kTilesPerSeg - 1) / kTilesPerSeg;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tm_a_hi);
        if (Cfg::A_PLANES == 2) tma_prefetch_desc(&tm_a_lo);
        tma_prefetch_desc(&tm_b_hi);
        if (Cfg::B_PLANES == 2) tma_prefetch_desc(&tm_b_lo);
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(full_bar(s), 1);
            mbar_init(empty_bar(s), 1);
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(tfull_bar(b), 1);
            mbar_init(tempty_bar(b), 8);          // one arrival per epilogue warp
        }
        fence_mbar_init();
    }
    if (warp == 2) {
        tmem_alloc(tmem_slot, Cfg::TMEM_COLS);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    if (warp == 0) {
        // ================================ TMA producer ================================
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
                const int m0 = (tile % args.tiles_m) * kBM;
                const int n0 = (tile / args.tiles_m) * BN;
                for (int kt = 0; kt < k_tiles; ++kt) {
                    mbar_wait(empty_bar(stage), phase ^ 1u, args.diag, 100 + stage);
                    const uint32_t sb = smem_base + stage * Cfg::STAGE_BYTES;
                    const uint32_t fb = full_bar(stage);
                    mbar_arrive_expect_tx(fb, Cfg::STAGE_BYTES);
                    const int k0 = kt * kBK;
                    tma_load_2d(sb, &tm_a_hi, fb, k0, m0);
                    if (Cfg::A_PLANES == 2) tma_load_2d(sb + Cfg::A_TILE, &tm_a_lo, fb, k0, m0);
                    const uint32_t sbB = sb + Cfg::A_PLANES * Cfg::A_TILE;
                    if (Cfg::B_MN) {
#pragma unroll
                        for (int c = 0; c < BN / 64; ++c) {
                            tma_load_2d(sbB + c * (64 * kBK * 2), &tm_b_hi, fb, n0 + c * 64, k0);
                            if (Cfg::B_PLANES == 2)
                                tma_load_2d(sbB + Cfg::B_TILE + c * (64 * kBK * 2), &tm_b_lo, fb, n0 + c * 64, k0);
                        }
                    } else {
                        tma_load_2d(sbB, &tm_b_hi, fb, k0, n0);
                        if (Cfg::B_PLANES == 2) tma_load_2d(sbB + Cfg::B_TILE, &tm_b_lo, fb, k0, n0);
                    }
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ================================ MMA issuer ==================================
        if (lane == 0) {
            constexpr uint32_t idesc = umma_idesc_f16_f32(kBM, BN, 0u, Cfg::B_MN ? 1u : 0u);
            // K-major SW128 (A, and B when stored N x K): 8-row groups 1024 B apart; LBO unused (1).
            constexpr uint64_t adesc0 = umma_smem_desc_sw128(0, 16, 1024);
            // MN-major SW128 (B stored K x N): 64-column atoms of kBK rows -> LBO = kBK*128 B between
            // atoms along N, SBO = 1024 B between 8-row groups along K.
            constexpr uint64_t bdesc0 = Cfg::B_MN ? umma_smem_desc_sw128(0, kBK * 128, 1024) : adesc0;
            constexpr uint32_t a_step = 32 >> 4;                               // +16 k = +32 bytes
            constexpr uint32_t b_step = (Cfg::B_MN ? 16 * 128 : 32) >> 4;      // +16 k = +16 rows of 128 B
            int stage = 0;
            uint32_t phase = 0;
            int buf = 0;
            uint32_t tphase = 0;                                // bit b = phase of TMEM buffer b
            for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
                for (int seg = 0; seg < n_seg; ++seg) {
                    mbar_wait(tempty_bar(buf), ((tphase >> buf) & 1u) ^ 1u, args.diag, 300 + buf);
                    tc_fence_after();
                    const uint32_t d_tmem = tmem_base + static_cast<uint32_t>(buf * BN);
                    const int kt_end = min(k_tiles, (seg + 1) * kTilesPerSeg);
                    uint32_t accumulate = 0;
                    for (int kt = seg * kTilesPerSeg; kt < kt_end; ++kt) {
                        mbar_wait(full_bar(stage), phase, args.diag, 200 + stage);
                        tc_fence_after();
                        const uint32_t sb = smem_base + stage * Cfg::STAGE_BYTES;
                        const uint64_t a_hi = adesc0 | desc_addr(sb);
                        const uint64_t a_lo = adesc0 | desc_addr(sb + Cfg::A_TILE);
                        const uint64_t b_hi = bdesc0 | desc_addr(sb + Cfg::A_PLANES * Cfg::A_TILE);
                        const uint64_t b_lo = bdesc0 | desc_addr(sb + Cfg::A_PLANES * Cfg::A_TILE + Cfg::B_TILE);
#pragma unroll
                        for (int j = 0; j < kBK / 16; ++j) {
                            const uint64_t ao = static_cast<uint64_t>(j * a_step), bo = static_cast<uint64_t>(j * b_step);
                            umma_f16(d_tmem, a_hi + ao, b_hi + bo, idesc, accumulate);
                            accumulate = 1;
                            if (NPROD == 2) umma_f16(d_tmem, a_lo + ao, b_hi + bo, idesc, 1);
                            if (NPROD >= 3) {
                                umma_f16(d_tmem, a_hi + ao, b_lo + bo, idesc, 1);
                                umma_f16(d_tmem, a_lo + ao, b_hi + bo, idesc, 1);
                            }
                            if (NPROD == 4) umma_f16(d_tmem, a_lo + ao, b_lo + bo, idesc, 1);
                        }
                        umma_commit(empty_bar(stage));          // smem slot free once these MMAs retire
                        if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                    }
                    umma_commit(tfull_bar(buf));                // segment partial sum complete in TMEM
                    tphase ^= 1u << buf;
                    buf ^= 1;
                }
            }
        }
    } else if (warp >= 4) {
        // ================================ epilogue ====================================
        constexpr int CPW = Cfg::COLS_PER_WARP;
        const int quad = warp & 3;
        const int chalf = (warp - 4) >> 2;
        float run[CPW];
        int buf = 0;
        uint32_t tphase = 0;
        for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
            const int m0 = (tile % args.tiles_m) * kBM;
            const int n0 = (tile / args.tiles_m) * BN;
            for (int seg = 0; seg < n_seg; ++seg) {
                mbar_wait(tfull_bar(buf), (tphase >> buf) & 1u, args.diag, 400 + buf);
                tc_fence_after();
                const uint32_t taddr = tmem_base + (static_cast<uint32_t>(quad * 32) << 16) +
                                       static_cast<uint32_t>(buf * BN + chalf * CPW);
#pragma unroll
                for (int c = 0; c < CPW / 16; ++c) {
                    uint32_t v[16];
                    tmem_ld_32x32b_x16(taddr + c * 16, v);
                    tmem_ld_wait();
                    if (seg == 0) {
#pragma unroll
                        for (int i = 0; i < 16; ++i) run[c * 16 + i] = __uint_as_float(v[i]);
                    } else {
#pragma unroll
                        for (int i = 0; i < 16; ++i) run[c * 16 + i] = __fadd_rn(run[c * 16 + i], __uint_as_float(v[i]));
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(tempty_bar(buf));
                tphase ^= 1u << buf;
                buf ^= 1;
            }
            // ---- store: thread owns row m0 + quad*32 + lane, CPW consecutive columns
            const int row = m0 + quad * 32 + lane;
            const int col0 = n0 + chalf * CPW;
            if (row < args.M) {
                float *crow = args.C + static_cast<int64_t>(row) * args.ldc;
#pragma unroll
                for (int c = 0; c < CPW; c += 4) {
                    const int col = col0 + c;
                    if (col + 3 < args.N) {
                        *reinterpret_cast<float4 *>(crow + col) = make_float4(run[c], run[c + 1], run[c + 2], run[c + 3]);
                    } else {
#pragma unroll
                        for (int i = 0; i < 4; ++i)
                            if (col + i < args.N) crow[col + i] = run[c + i];
                    }
                }
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 2) {
        tc_fence_after();
        tmem_dealloc(tmem_base, Cfg::TMEM_COLS);
    }
}

}  // namespace heal
