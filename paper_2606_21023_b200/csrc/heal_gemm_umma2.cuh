// heal_gemm_umma2.cuh -- steps G + E with CTA pairs (tcgen05 cta_group::2): the two CTAs of a cluster
// share one 256 x BN output tile.  Each CTA loads its own 128 rows of the A planes and HALF of the B
// tile (BN/2 columns); the leader's single thread issues 256 x BN x 16 MMAs that read both CTAs' shared
// memory and write each CTA's 128 rows of the accumulator into its own TMEM.  Per CTA and k-tile this
// moves 48 KB (2P) / 64 KB (3P) from L2 instead of 64 / 96 KB for single-CTA tiles -- the L2 -> SM fabric,
// not the tensor pipe, is what bounds the single-CTA kernel.
//
// Same numerical contract as heal_gemm_umma.cuh (K segments of 512, k16 slices ascending, products
// hi.hi, hi.lo, lo.hi, lo.lo, segments added in FP32 RN ascending): bit-identical results.
//
// Barriers: full[stage] lives in the leader (2 producer arrivals + both CTAs' TMA bytes); empty[stage],
// tmem_full[buf] are signalled in both CTAs by multicast tcgen05.commit; tmem_empty[buf] lives in the
// leader (16 arrivals: 8 epilogue warps of each CTA).
#pragma once
#include "heal_gemm_umma.cuh"

namespace heal {

#ifdef HEAL_TRACE
// trace builds only (python -m paper_2606_21023_b200.build --trace; the product library compiles all of this out): per CTA pair,
// cycles the MMA thread waited for operands / for a free accumulator / in total, and cycles one epilogue warp of the leader
// waited for a finished segment / drained TMEM / stored C / in total.  Read back with heal_debug_read_pair_trace().
__device__ unsigned long long g_pair_trace[512 * 8];
#define HEAL_TCLK() clock64()
#else
#define HEAL_TCLK() 0ll
#endif

template <int BN_, int NPROD_, bool B_MN_, bool FULL_ = false>
struct Gemm2Cfg {
    static constexpr bool FULL = FULL_;                 // with the extended epilogue (2^-p scale, chained planes, accumulate) and the
                                                        // ordered split-K schedule; the default instantiation has neither, so the
                                                        // headline path carries no extra registers or code (measured: 2.5 % otherwise)
    static constexpr int BN = BN_;                       // pair-tile width; each CTA stages BN/2 columns of B
    static constexpr bool SCALED = NPROD_ == kScaledLo;  // HEAL_LO_SCALED in one kernel (see heal_gemm_umma.cuh): two passes per K segment
    static constexpr int NPROD = SCALED ? 2 : NPROD_;
    static constexpr bool B_MN = B_MN_;
    static constexpr int A_PLANES = NPROD >= 2 ? 2 : 1;
    static constexpr int B_PLANES = NPROD >= 3 ? 2 : 1;
    static constexpr int A_TILE = kBM * kBK * 2;
    static constexpr int BH = BN / 2;
    static constexpr int B_TILE = BH * kBK * 2;
    static constexpr int A_SLOTS = SCALED ? 1 : A_PLANES;   // SCALED: one activation plane per pass shares the slot
    static constexpr int STAGE_BYTES = A_SLOTS * A_TILE + B_PLANES * B_TILE;
    static constexpr int BAR_BYTES = 256;
    static constexpr int STAGES_RAW = (kSmemLimit - 1024 - BAR_BYTES) / STAGE_BYTES;
    static constexpr int STAGES = STAGES_RAW > 8 ? 8 : STAGES_RAW;
    static constexpr int TMEM_COLS = 512;
    // TMEM rule (heal_gemm_umma.cuh): this kernel takes all 512 columns, so no other TMEM-allocating CTA may share its SM.  Its stages fill
    // 193-225 KB of shared memory, and its CTA takes the whole register file (384 x 168 or 512 x 128 registers), so nothing co-resides at all;
    // padding the shared memory to the full 227 KB on top of that measured 1 % slower on the headline GEMM and is not done.
    static constexpr int SMEM_BYTES = 1024 + STAGES * STAGE_BYTES + BAR_BYTES;
    static constexpr int COLS_PER_WARP = BN / 2;
    static_assert(BN == 256 || BN == 128, "BN");
    static_assert(STAGES >= 2, "need at least two stages");
};

template <class Cfg>
__global__ void __launch_bounds__(kGemmThreads, 1)
heal_gemm_umma2_kernel(const __grid_constant__ CUtensorMap tm_a_hi, const __grid_constant__ CUtensorMap tm_a_lo,
                       const __grid_constant__ CUtensorMap tm_b_hi, const __grid_constant__ CUtensorMap tm_b_lo,
                       const GemmArgs args)
{
    constexpr int BN = Cfg::BN, NPROD = Cfg::NPROD, STAGES = Cfg::STAGES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_base = smem_base + STAGES * Cfg::STAGE_BYTES;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
    auto tfull_bar = [&](int b) { return bar_base + 8u * (2 * STAGES + b); };
    auto tempty_bar = [&](int b) { return bar_base + 8u * (2 * STAGES + 2 + b); };
    const uint32_t tmem_slot = bar_base + 8u * (2 * STAGES + 4);
    volatile uint32_t *tmem_slot_ptr =
        reinterpret_cast<volatile uint32_t *>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int rank = static_cast<int>(cluster_ctarank());          // 0 = leader
    const int k_tiles = (args.K + kBK - 1) / kBK;
    const int n_seg = (k_tiles + kTilesPerSeg - 1) / kTilesPerSeg;
    TileSched sched;
    sched.init(args.tiles_m * args.tiles_n, args.balance, args.dp_tiles, n_seg, static_cast<int>(blockIdx.x >> 1), static_cast<int>(gridDim.x >> 1));

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tm_a_hi);
        if (Cfg::A_PLANES == 2) tma_prefetch_desc(&tm_a_lo);
        tma_prefetch_desc(&tm_b_hi);
        if (Cfg::B_PLANES == 2) tma_prefetch_desc(&tm_b_lo);
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(full_bar(s), 2);            // one arrive.expect_tx from each CTA's producer
            mbar_init(empty_bar(s), 1);
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
                // SCALED: every K segment is walked twice -- first the scaled residual plane, then the hi plane (each with the weight tile)
                const int n_steps = Cfg::SCALED ? 2 * (kt_hi - sb_seg * kTilesPerSeg) : kt_hi - sb_seg * kTilesPerSeg;
                for (int step = 0; step < n_steps; ++step) {
                    int kt = sb_seg * kTilesPerSeg + step;
                    bool lo_pass = false;
                    if (Cfg::SCALED) {
                        const int seg = sb_seg + step / (2 * kTilesPerSeg), r = step % (2 * kTilesPerSeg);
                        const int len = min(k_tiles, (seg + 1) * kTilesPerSeg) - seg * kTilesPerSeg;     // (only the last segment of K is short,
                        lo_pass = r < len;                                                                //  and it is the last one of the chunk)
                        kt = seg * kTilesPerSeg + (lo_pass ? r : r - len);
                    }
                    mbar_wait_ool(empty_bar(stage), phase ^ 1u, args.diag, 100 + stage);
                    const uint32_t sb = smem_base + stage * Cfg::STAGE_BYTES;
                    const uint32_t fb = leader_addr(full_bar(stage));
                    mbar_arrive_expect_tx_cluster(fb, Cfg::STAGE_BYTES);
                    const int k0 = kt * kBK;
                    if (Cfg::SCALED) {
                        tma_load_2d_2cta(sb, lo_pass ? &tm_a_lo : &tm_a_hi, fb, k0, m0);
                    } else {
                        tma_load_2d_2cta(sb, &tm_a_hi, fb, k0, m0);
                        if (Cfg::A_PLANES == 2) tma_load_2d_2cta(sb + Cfg::A_TILE, &tm_a_lo, fb, k0, m0);
                    }
                    const uint32_t sbB = sb + Cfg::A_SLOTS * Cfg::A_TILE;
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
            long long w_full = 0, w_tempty = 0;
            const long long t_begin = HEAL_TCLK();
            for (int ci = 0; ci < sched.n_chunks; ++ci) {
                int tile, sb_seg, se_seg;
                sched.get(ci, tile, sb_seg, se_seg);
                for (int seg = sb_seg; seg < se_seg; ++seg) {
                    const long long t0 = HEAL_TCLK();
                    mbar_wait_ool(tempty_bar(buf), ((tphase >> buf) & 1u) ^ 1u, args.diag, 300 + buf);
                    w_tempty += HEAL_TCLK() - t0;
                    tc_fence_after();
                    const uint32_t d_tmem = tmem_base + static_cast<uint32_t>(buf * BN);
                    const int kt_end = min(k_tiles, (seg + 1) * kTilesPerSeg);
                    uint32_t accumulate = 0;
                    if constexpr (Cfg::SCALED) {
                        // D = sum_k lo'_k . W_k (k ascending), then D = hi_0 . W_0 + D * 2^-10, then D += hi_k . W_k: Eq. 10 as printed
                        // in one accumulator -- the tensor core scales the residual sum by an exact power of two
                        // before the first hi product is added (scale_input_d)
                        for (int pass = 0; pass < 2; ++pass)
                            for (int kt = seg * kTilesPerSeg; kt < kt_end; ++kt) {
                                mbar_wait_ool(full_bar(stage), phase, args.diag, 200 + stage);
                                tc_fence_after();
                                const uint32_t sb = smem_base + stage * Cfg::STAGE_BYTES;
                                const uint64_t a_d = adesc0 | desc_addr(sb);
                                const uint64_t b_d = bdesc0 | desc_addr(sb + Cfg::A_TILE);
#pragma unroll
                                for (int j = 0; j < kBK / 16; ++j) {
                                    const uint64_t ao = static_cast<uint64_t>(j * a_step), bo = static_cast<uint64_t>(j * b_step);
                                    if (pass == 1 && kt == seg * kTilesPerSeg && j == 0)
                                        umma_f16_2cta_scale_d<kLoShift>(d_tmem, a_d + ao, b_d + bo, idesc);
                                    else
                                        umma_f16_2cta(d_tmem, a_d + ao, b_d + bo, idesc, accumulate);
                                    accumulate = 1;
                                }
                                umma_commit_2cta(empty_bar(stage), 3);
                                if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                            }
                    } else
                    for (int kt = seg * kTilesPerSeg; kt < kt_end; ++kt) {
                        const long long t1 = HEAL_TCLK();
                        mbar_wait_ool(full_bar(stage), phase, args.diag, 200 + stage);
                        w_full += HEAL_TCLK() - t1;
                        tc_fence_after();
                        const uint32_t sb = smem_base + stage * Cfg::STAGE_BYTES;
                        const uint64_t a_hi = adesc0 | desc_addr(sb);
                        const uint64_t a_lo = adesc0 | desc_addr(sb + Cfg::A_TILE);
                        const uint64_t b_hi = bdesc0 | desc_addr(sb + Cfg::A_PLANES * Cfg::A_TILE);
                        const uint64_t b_lo = bdesc0 | desc_addr(sb + Cfg::A_PLANES * Cfg::A_TILE + Cfg::B_TILE);
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
#ifdef HEAL_TRACE
            if ((blockIdx.x >> 1) < 512) {
                unsigned long long *tr = g_pair_trace + (blockIdx.x >> 1) * 8;
                tr[0] = static_cast<unsigned long long>(w_full);
                tr[1] = static_cast<unsigned long long>(w_tempty);
                tr[2] = static_cast<unsigned long long>(HEAL_TCLK() - t_begin);
            }
#endif
            (void)w_full; (void)w_tempty; (void)t_begin;
        }
    } else if (warp >= 4) {
        // ================================ epilogue (both CTAs) =========================
        constexpr int CPW = Cfg::COLS_PER_WARP;
        const int quad = warp & 3;
        const int chalf = (warp - 4) >> 2;
        const int etid = threadIdx.x - 128;
        float run[CPW];
        int buf = 0;
        uint32_t tphase = 0;
        long long e_wait = 0, e_drain = 0, e_store = 0, e_segs = 0;
        const long long e_begin = HEAL_TCLK();
        for (int ci = 0; ci < sched.n_chunks; ++ci) {
            int tile, sb_seg, se_seg;
            sched.get(ci, tile, sb_seg, se_seg);
            int tm, tn;
            tile_coords(tile, args.tiles_m, args.tiles_n, tm, tn, args.group_m);
            const int m0 = tm * (2 * kBM) + rank * kBM;
            const int n0 = tn * BN;
            if constexpr (Cfg::FULL) {
                if (args.sk) {
                    // ordered split-K (see heal_gemm_umma.cuh): park every segment partial of this CTA's 128 rows
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
            if (sb_seg > 0)        // same rank of the previous pair
                epi_take_prefix<CPW>(args.xfer + static_cast<size_t>(blockIdx.x - 2) * (kBM * 256), args.flags + (blockIdx.x - 2), run, etid, args.diag);
            for (int seg = sb_seg; seg < se_seg; ++seg) {
                const long long t0 = HEAL_TCLK();
                mbar_wait_ool(tfull_bar(buf), (tphase >> buf) & 1u, args.diag, 400 + buf);
                const long long t1 = HEAL_TCLK();
                tc_fence_after();
                const uint32_t taddr = tmem_base + (static_cast<uint32_t>(quad * 32) << 16) +
                                       static_cast<uint32_t>(buf * BN + chalf * CPW);
                epi_add_segment<CPW>(taddr, run, seg == 0);
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(leader_addr(tempty_bar(buf)));
                e_wait += t1 - t0;
                e_drain += HEAL_TCLK() - t1;
                ++e_segs;
                tphase ^= 1u << buf;
                buf ^= 1;
            }
            if (se_seg < n_seg) {
                epi_hand_on<CPW>(args.xfer + static_cast<size_t>(blockIdx.x) * (kBM * 256), args.flags + blockIdx.x, run, etid);
                continue;
            }
            const long long t2 = HEAL_TCLK();
            epi_store<CPW, Cfg::FULL>(args.out, m0 + quad * 32 + lane, n0 + chalf * CPW, run, args.M, args.N);
            e_store += HEAL_TCLK() - t2;
        }
#ifdef HEAL_TRACE
        if (etid == 0 && rank == 0 && (blockIdx.x >> 1) < 512) {
            unsigned long long *tr = g_pair_trace + (blockIdx.x >> 1) * 8;
            tr[3] = static_cast<unsigned long long>(e_wait);
            tr[4] = static_cast<unsigned long long>(e_drain);
            tr[5] = static_cast<unsigned long long>(e_store);
            tr[6] = static_cast<unsigned long long>(HEAL_TCLK() - e_begin);
            tr[7] = static_cast<unsigned long long>(e_segs);
        }
#endif
        (void)e_wait; (void)e_drain; (void)e_store; (void)e_begin; (void)e_segs;
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
