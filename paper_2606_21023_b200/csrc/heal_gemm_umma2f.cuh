// heal_gemm_umma2f.cuh -- steps S + G + E in ONE kernel for prefill shapes: the
// CTA-pair kernel of heal_gemm_umma2.cuh with the activation split done on the fly in shared memory.  The FP32 activation
// tile travels by TMA (128 rows x 64 k x 4 B = 32 KB, exactly the bytes of the hi + lo FP16 tiles it replaces), four
// converter warps turn it IN PLACE into the two 128B-swizzled FP16 operand tiles (hi = r16(x), lo = r16(x - hi): the
// split kernel's own split2), and the tensor core consumes them as before.  No hi/lo planes in HBM, no split launch:
// 8 B per activation element of HBM traffic and one launch less than split + GEMM.  Weights: FP16 as given (2P), or the
// pre-split planes of FP32 weights (3P).
//
// In-place layout trick.  The FP32 tile is fetched as two TMA boxes of 32 k each (128-byte rows, no swizzle): k 0..31
// of row m land at byte m*128 of the stage's first 16 KB, k 32..63 at byte m*128 of the second 16 KB.  The K-major
// SWIZZLE_128B operand tiles the MMA wants put row m of `hi` at byte m*128 of the first 16 KB (its eight 16-byte chunks
// permuted by m % 8) and row m of `lo` at byte m*128 of the second 16 KB.  So the 256 input bytes and the 256 output
// bytes of a row are the SAME bytes: eight lanes of one warp own a row, read it completely, __syncwarp, write it back
// converted -- no second buffer, no CTA-wide barrier, and the pipeline keeps its full depth.
//
// Roles (512 threads, one persistent CTA per SM, clusters of 2): warp 0 TMA producer, warp 1 MMA issuer (leader),
// warp 2 TMEM allocator, warp 3 idle, warps 4-11 epilogue, warps 12-15 converters.  Register file: setmaxnreg gives the
// epilogue warps (128-float running sums) 184 registers, the control warps 56, the converters 88 (56 + 2 * 184 + 88 = 512 = 4 * 128).
// The shrunk warps must not call out-of-line functions (ptxas cannot fit a callee's ABI register budget into them), hence the
// inline mbarrier waits in those roles.
//
// Barriers per stage: afull (local: this CTA's FP32 tile has landed), full (leader: both CTAs' weight tiles), conv (leader:
// 8 arrivals = 4 converter warps x 2 CTAs, after fence.proxy.async), empty (both CTAs, multicast tcgen05.commit).
//
// Same numerical contract as every other kernel of the library (K segments of 512, k16 slices ascending, products
// hi.hi, hi.lo, lo.hi, lo.lo, segments added in FP32 RN ascending); the planes the converters build are bit-identical to
// heal_split's, so heal_gemm gives the same bits whichever path runs (tested).
#pragma once
#include "heal_gemm_umma2.cuh"

namespace heal {

constexpr int kFusedThreads = 512;

template <int NPROD_, bool B_MN_, bool FULL_ = false>
struct Gemm2FCfg {
    static constexpr bool FULL = FULL_;
    static constexpr int BN = 256;
    static constexpr int NPROD = NPROD_;
    static constexpr bool B_MN = B_MN_;
    static constexpr int B_PLANES = NPROD >= 3 ? 2 : 1;
    static constexpr int A_TILE = kBM * kBK * 2;            // one FP16 operand tile = half of the FP32 tile
    static constexpr int A_BYTES = 2 * A_TILE;              // FP32 tile = hi tile + lo tile
    static constexpr int BH = BN / 2;
    static constexpr int B_TILE = BH * kBK * 2;
    static constexpr int B_BYTES = B_PLANES * B_TILE;
    static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
    static constexpr int BAR_BYTES = 512;
    static constexpr int STAGES_RAW = (kSmemLimit - 1024 - BAR_BYTES) / STAGE_BYTES;
    static constexpr int STAGES = STAGES_RAW > 8 ? 8 : STAGES_RAW;
    static constexpr int TMEM_COLS = 512;
    // TMEM rule (heal_gemm_umma.cuh): this kernel takes all 512 columns, so no other TMEM-allocating CTA may share its SM.  Its stages fill
    // 193-225 KB of shared memory, and its CTA takes the whole register file (384 x 168 or 512 x 128 registers), so nothing co-resides at all;
    // padding the shared memory to the full 227 KB on top of that measured 1 % slower on the headline GEMM and is not done.
    static constexpr int SMEM_BYTES = 1024 + STAGES * STAGE_BYTES + BAR_BYTES;
    static constexpr int COLS_PER_WARP = BN / 2;
    static_assert(NPROD >= 2 && NPROD <= 4, "the lo plane is what the fused split is for");
    static_assert(STAGES >= 2, "need at least two stages");
};

template <class Cfg>
__global__ void __launch_bounds__(kFusedThreads, 1)
heal_gemm_umma2f_kernel(const __grid_constant__ CUtensorMap tm_a32, const __grid_constant__ CUtensorMap tm_b_hi,
                        const __grid_constant__ CUtensorMap tm_b_lo, const GemmArgs args)
{
    constexpr int BN = Cfg::BN, NPROD = Cfg::NPROD, STAGES = Cfg::STAGES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_base = smem_base + STAGES * Cfg::STAGE_BYTES;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
    auto afull_bar = [&](int s) { return bar_base + 8u * (2 * STAGES + s); };
    auto conv_bar = [&](int s) { return bar_base + 8u * (3 * STAGES + s); };
    auto tfull_bar = [&](int b) { return bar_base + 8u * (4 * STAGES + b); };
    auto tempty_bar = [&](int b) { return bar_base + 8u * (4 * STAGES + 2 + b); };
    const uint32_t tmem_slot = bar_base + 8u * (4 * STAGES + 4);
    volatile uint32_t *tmem_slot_ptr =
        reinterpret_cast<volatile uint32_t *>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int rank = static_cast<int>(cluster_ctarank());          // 0 = leader
    const int k_tiles = (args.K + kBK - 1) / kBK;
    const int n_seg = (k_tiles + kTilesPerSeg - 1) / kTilesPerSeg;
    TileSched sched;
    sched.init(args.tiles_m * args.tiles_n, args.balance, args.dp_tiles, n_seg, static_cast<int>(blockIdx.x >> 1), static_cast<int>(gridDim.x >> 1));

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tm_a32);
        tma_prefetch_desc(&tm_b_hi);
        if (Cfg::B_PLANES == 2) tma_prefetch_desc(&tm_b_lo);
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(full_bar(s), 2);            // one arrive.expect_tx from each CTA's producer
            mbar_init(empty_bar(s), 1);
            mbar_init(afull_bar(s), 1);
            mbar_init(conv_bar(s), 8);            // 4 converter warps of each CTA
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(tfull_bar(b), 1);
            mbar_init(tempty_bar(b), 16);         // 8 epilogue warps of each CTA
        }
        fence_mbar_init();
    }
    if (warp == 2) {
        tmem_alloc_2cta(tmem_slot, Cfg::TMEM_COLS);
        tmem_relinquish_2cta();
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();                            // peer barriers initialised before any remote arrive
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;
    pdl_wait();
    pdl_launch_dependents();

    if (warp < 4) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        if (warp == 0) {
            // ================================ TMA producer (both CTAs) =====================
            if (lane == 0) {
                int stage = 0;
                uint32_t phase = 0;
                for (int ci = 0; ci < sched.n_chunks; ++ci) {
                    int tile, sb_seg, se_seg;
                    sched.get(ci, tile, sb_seg, se_seg);
                    int tm, tn;
                    tile_coords(tile, args.tiles_m, args.tiles_n, tm, tn, args.group_m);
                    const int m0 = tm * (2 * kBM) + rank * kBM;
                    const int n0 = tn * BN + rank * Cfg::BH;
                    const int kt_hi = min(k_tiles, se_seg * kTilesPerSeg);
                    for (int kt = sb_seg * kTilesPerSeg; kt < kt_hi; ++kt) {
                        mbar_wait(empty_bar(stage), phase ^ 1u, args.diag, 100 + stage);
                        const uint32_t sb = smem_base + stage * Cfg::STAGE_BYTES;
                        const int k0 = kt * kBK;
                        // activations first: the converters start as soon as they land
                        const uint32_t ab = afull_bar(stage);
                        mbar_arrive_expect_tx(ab, Cfg::A_BYTES);
                        tma_load_2d(sb, &tm_a32, ab, k0, m0);
                        tma_load_2d(sb + Cfg::A_TILE, &tm_a32, ab, k0 + 32, m0);
                        const uint32_t fb = leader_addr(full_bar(stage));
                        mbar_arrive_expect_tx_cluster(fb, Cfg::B_BYTES);
                        const uint32_t sbB = sb + Cfg::A_BYTES;
                        if (Cfg::B_MN) {
#pragma unroll
                            for (int c = 0; c < Cfg::BH / 64; ++c) {
                                tma_load_2d_2cta(sbB + c * (64 * kBK * 2), &tm_b_hi, fb, n0 + c * 64, k0);
                                if (Cfg::B_PLANES == 2)
                                    tma_load_2d_2cta(sbB + Cfg::B_TILE + c * (64 * kBK * 2), &tm_b_lo, fb, n0 + c * 64, k0);
                            }
                        } else {
                            tma_load_2d_2cta(sbB, &tm_b_hi, fb, k0, n0);
                            if (Cfg::B_PLANES == 2) tma_load_2d_2cta(sbB + Cfg::B_TILE, &tm_b_lo, fb, k0, n0);
                        }
                        if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                    }
                }
            }
        } else if (warp == 1) {
            // ================================ MMA issuer (leader only) =====================
            if (lane == 0 && rank == 0) {
                constexpr uint32_t idesc = umma_idesc_f16_f32(2 * kBM, BN, 0u, Cfg::B_MN ? 1u : 0u);
                constexpr uint64_t adesc0 = umma_smem_desc_sw128(0, 16, 1024);
                constexpr uint64_t bdesc0 = Cfg::B_MN ? umma_smem_desc_sw128(0, kBK * 128, 1024) : adesc0;
                constexpr uint32_t a_step = 32 >> 4;
                constexpr uint32_t b_step = (Cfg::B_MN ? 16 * 128 : 32) >> 4;
                int stage = 0;
                uint32_t phase = 0;
                int buf = 0;
                uint32_t tphase = 0;
                for (int ci = 0; ci < sched.n_chunks; ++ci) {
                    int tile, sb_seg, se_seg;
                    sched.get(ci, tile, sb_seg, se_seg);
                    for (int seg = sb_seg; seg < se_seg; ++seg) {
                        mbar_wait(tempty_bar(buf), ((tphase >> buf) & 1u) ^ 1u, args.diag, 300 + buf);
                        tc_fence_after();
                        const uint32_t d_tmem = tmem_base + static_cast<uint32_t>(buf * BN);
                        const int kt_end = min(k_tiles, (seg + 1) * kTilesPerSeg);
                        uint32_t accumulate = 0;
                        for (int kt = seg * kTilesPerSeg; kt < kt_end; ++kt) {
                            mbar_wait(full_bar(stage), phase, args.diag, 200 + stage);
                            mbar_wait_cluster_inl(conv_bar(stage), phase, args.diag, 250 + stage);     // acquire.cluster: the peer's converters arrive remotely
                            tc_fence_after();
                            const uint32_t sb = smem_base + stage * Cfg::STAGE_BYTES;
                            const uint64_t a_hi = adesc0 | desc_addr(sb);
                            const uint64_t a_lo = adesc0 | desc_addr(sb + Cfg::A_TILE);
                            const uint64_t b_hi = bdesc0 | desc_addr(sb + Cfg::A_BYTES);
                            const uint64_t b_lo = bdesc0 | desc_addr(sb + Cfg::A_BYTES + Cfg::B_TILE);
#pragma unroll
                            for (int j = 0; j < kBK / 16; ++j) {
                                const uint64_t ao = static_cast<uint64_t>(j * a_step), bo = static_cast<uint64_t>(j * b_step);
                                umma_f16_2cta(d_tmem, a_hi + ao, b_hi + bo, idesc, accumulate);
                                accumulate = 1;
                                if (NPROD == 2) umma_f16_2cta(d_tmem, a_lo + ao, b_hi + bo, idesc, 1);
                                if (NPROD >= 3) {
                                    umma_f16_2cta(d_tmem, a_hi + ao, b_lo + bo, idesc, 1);
                                    umma_f16_2cta(d_tmem, a_lo + ao, b_hi + bo, idesc, 1);
                                }
                                if (NPROD == 4) umma_f16_2cta(d_tmem, a_lo + ao, b_lo + bo, idesc, 1);
                            }
                            umma_commit_2cta(empty_bar(stage), 3);      // slot free in both CTAs
                            if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                        }
                        umma_commit_2cta(tfull_bar(buf), 3);            // segment partial complete in both TMEMs
                        tphase ^= 1u << buf;
                        buf ^= 1;
                    }
                }
            }
        }
    } else if (warp >= 12) {
        // ================================ converters: step S in shared memory (both CTAs) =================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 88;");
        const int cw = warp - 12;                           // rows 32*cw .. 32*cw + 31 of the tile
        const int j = lane & 7, rq = lane >> 3;             // 16-byte output chunk (k = 8j..8j+7), row within a group of 4
        // input: k 8j..8j+3 and 8j+4..8j+7 are 16-byte chunks 2(j%4), 2(j%4)+1 of the row in the first (j < 4) or second
        // (j >= 4) half of the FP32 tile; lanes j >= 4 fetch the odd chunk first, so that the eight lanes of a row touch
        // eight different bank groups in each of the two loads
        const uint32_t in_half = (j >= 4) ? static_cast<uint32_t>(Cfg::A_TILE) : 0u;
        const uint32_t c_even = static_cast<uint32_t>((2 * (j & 3)) << 4), c_odd = c_even + 16u;
        const uint32_t first = (j >= 4) ? c_odd : c_even, second = (j >= 4) ? c_even : c_odd;
        const uint32_t conv_leader = leader_addr(conv_bar(0));
        int stage = 0;
        uint32_t phase = 0;
        for (int ci = 0; ci < sched.n_chunks; ++ci) {
            int tile, sb_seg, se_seg;
            sched.get(ci, tile, sb_seg, se_seg);
            const int kt_hi = min(k_tiles, se_seg * kTilesPerSeg);
            for (int kt = sb_seg * kTilesPerSeg; kt < kt_hi; ++kt) {
                mbar_wait(afull_bar(stage), phase, args.diag, 150 + stage);
                const uint32_t sa = smem_base + stage * Cfg::STAGE_BYTES;
#pragma unroll
                for (int it = 0; it < 8; it += 2) {
                    float4 x[2][2];
                    uint32_t row_off[2];
#pragma unroll
                    for (int u = 0; u < 2; ++u) {
                        const int m = cw * 32 + (it + u) * 4 + rq;
                        row_off[u] = static_cast<uint32_t>(m) * 128u;
                        const uint32_t src = sa + in_half + row_off[u];
                        asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                                     : "=f"(x[u][0].x), "=f"(x[u][0].y), "=f"(x[u][0].z), "=f"(x[u][0].w) : "r"(src + first) : "memory");
                        asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                                     : "=f"(x[u][1].x), "=f"(x[u][1].y), "=f"(x[u][1].z), "=f"(x[u][1].w) : "r"(src + second) : "memory");
                    }
                    __syncwarp();                            // every lane of a row has read it before anyone overwrites it
#pragma unroll
                    for (int u = 0; u < 2; ++u) {
                        const float4 lo4 = (j >= 4) ? x[u][1] : x[u][0];        // k 8j..8j+3
                        const float4 hi4 = (j >= 4) ? x[u][0] : x[u][1];        // k 8j+4..8j+7
                        uint4 h, l;
                        split2(lo4.x, lo4.y, h.x, l.x);
                        split2(lo4.z, lo4.w, h.y, l.y);
                        split2(hi4.x, hi4.y, h.z, l.z);
                        split2(hi4.z, hi4.w, h.w, l.w);
                        const int m7 = ((it + u) * 4 + rq) & 7;                  // (cw * 32 is a multiple of 8)
                        const uint32_t dst = sa + row_off[u] + (static_cast<uint32_t>(j ^ m7) << 4);
                        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(dst), "r"(h.x), "r"(h.y), "r"(h.z), "r"(h.w) : "memory");
                        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(dst + Cfg::A_TILE), "r"(l.x), "r"(l.y), "r"(l.z), "r"(l.w) : "memory");
                    }
                }
                // generic-proxy writes -> visible to this SM's tensor core (the consumer of this CTA's activation rows); then a
                // RELAXED remote arrive: a cluster-scope release costs ~0.5 us per arrive on this part (measured), which would
                // make the converters the bottleneck, and nothing but the local async proxy -- ordered by the fence -- reads
                // these bytes; the leader's MMA reaches this SM's tensor core only after it has seen the arrive
                fence_proxy_async_smem();
                __syncwarp();
                if (lane == 0) mbar_arrive_relaxed_cluster(conv_leader + 8u * stage);
                if (++stage == STAGES) { stage = 0; phase ^= 1u; }
            }
        }
    } else {
        // ================================ epilogue (both CTAs) =========================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 184;");
        constexpr int CPW = Cfg::COLS_PER_WARP;
        const int quad = warp & 3;
        const int chalf = (warp - 4) >> 2;
        const int etid = threadIdx.x - 128;
        float run[CPW];
        int buf = 0;
        uint32_t tphase = 0;
        for (int ci = 0; ci < sched.n_chunks; ++ci) {
            int tile, sb_seg, se_seg;
            sched.get(ci, tile, sb_seg, se_seg);
            int tm, tn;
            tile_coords(tile, args.tiles_m, args.tiles_n, tm, tn, args.group_m);
            const int m0 = tm * (2 * kBM) + rank * kBM;
            const int n0 = tn * BN;
            if constexpr (Cfg::FULL) {
                if (args.sk) {
                    for (int seg = sb_seg; seg < se_seg; ++seg) {
                        mbar_wait_ool(tfull_bar(buf), (tphase >> buf) & 1u, args.diag, 400 + buf);
                        tc_fence_after();
                        const uint32_t taddr = tmem_base + (static_cast<uint32_t>(quad * 32) << 16) +
                                               static_cast<uint32_t>(buf * BN + chalf * CPW);
                        sk_store_partial<CPW>(args.part + ((static_cast<size_t>(tile) * 2 + rank) * n_seg + seg) * (kBM * BN), taddr, etid);
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive_cluster(leader_addr(tempty_bar(buf)));
                        tphase ^= 1u << buf;
                        buf ^= 1;
                    }
                    continue;
                }
            }
            if (sb_seg > 0)
                epi_take_prefix<CPW>(args.xfer + static_cast<size_t>(blockIdx.x - 2) * (kBM * 256), args.flags + (blockIdx.x - 2), run, etid, args.diag);
            for (int seg = sb_seg; seg < se_seg; ++seg) {
                mbar_wait_ool(tfull_bar(buf), (tphase >> buf) & 1u, args.diag, 400 + buf);
                tc_fence_after();
                const uint32_t taddr = tmem_base + (static_cast<uint32_t>(quad * 32) << 16) +
                                       static_cast<uint32_t>(buf * BN + chalf * CPW);
                epi_add_segment<CPW>(taddr, run, seg == 0);
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(leader_addr(tempty_bar(buf)));
                tphase ^= 1u << buf;
                buf ^= 1;
            }
            if (se_seg < n_seg) {
                epi_hand_on<CPW>(args.xfer + static_cast<size_t>(blockIdx.x) * (kBM * 256), args.flags + blockIdx.x, run, etid);
                continue;
            }
            epi_store<CPW, Cfg::FULL>(args.out, m0 + quad * 32 + lane, n0 + chalf * CPW, run, args.M, args.N);
        }
    }

    tc_fence_before();
    __syncthreads();
    cluster_sync_all();                            // the peer may still be reading this CTA's smem / signalling its barriers
    if (warp == 2) {
        tc_fence_after();
        tmem_dealloc_2cta(tmem_base, Cfg::TMEM_COLS);
    }
}

}  // namespace heal
