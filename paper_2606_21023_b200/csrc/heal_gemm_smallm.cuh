// heal_gemm_smallm.cuh -- steps (S +) G + E for small M (decode / LM-head shapes, M <= 64): the weight
// matrix is streamed once from HBM and is the tensor core's 128-row operand ("swap-AB"), the few
// token rows are the UMMA N side (16/32/64), and the K segments of one 128-column weight panel are
// spread over the CTAs of a thread-block cluster so that enough CTAs stream HBM.
//
// Same reduction order as heal_gemm_umma.cuh (include/heal.h): inside a 512-long K segment the tensor
// core accumulates k16 slices in ascending k, products hi.hi, hi.lo, lo.hi, lo.lo; the segment partial
// sums are then added in ascending segment order in FP32 RN.  Results are bit-identical to the
// large-M kernels.
//
// Cluster of CS CTAs = one 128-column panel; CTA rank r owns segments r, r+CS, r+2CS, ... (local slot
// j = s / CS lives in TMEM columns j*MPAD..).  Token rows are dealt to the ranks in contiguous blocks: every rank
// PUSHES its segment partials of those rows straight from its TMEM registers into the owner's shared
// memory -- with st.async when a thread has few values to send (the bytes are counted on the owner's
// mbarrier: no fence, no arrive), else with plain st.shared::cluster plus one fence and one relaxed
// remote arrive per warp; the owner adds the n_seg partials in ascending segment order and stores C.
// No atomics, no cluster-wide barrier after the main loop.
//
// FUSED variant (heal_gemm, B already FP16): step S runs inside the kernel -- the four epilogue warps
// convert the FP32 activations of each k-tile to hi/lo FP16 (same arithmetic as
// heal_split.cuh) directly into the swizzled shared-memory operand tiles while the TMA producer streams W;
// no hi/lo planes in HBM, no split launch.
//
// Static weights (HEAL_B_STATIC): the producer starts streaming W before griddepcontrol.wait, i.e. while
// the previous kernel on the stream is still in its tail; everything that touches activations or C waits.
//
// PAIR variant (M > 32, large N, one CTA per panel): two adjacent panels form a CTA pair under one cta_group::2 MMA
// (UMMA M = 256), each CTA staging its own weight panel and HALF of the token tile; barriers as in heal_gemm_umma2.cuh
// (full in the leader, empty / slot-full / done by multicast commit, slot-empty in the leader).
//
// Roles per CTA (192 threads): warp 0 TMA producer, warp 1 MMA issuer + TMEM allocator, warps 2-5
// converter (FUSED) and epilogue (warp w owns TMEM lanes 32*(w%4)..+31).
#pragma once
#include "heal_epilogue.cuh"
#include "heal_ptx.cuh"

namespace heal {

constexpr int kSmallThreads = 192;
constexpr int kSmallBNW = 128;          // weight columns per panel (UMMA M)
constexpr int kSmallMaxStages = 8;

template <int MPAD_, int NPROD_, bool B_MN_, bool FUSED_, bool PAIR_ = false>
struct SmallCfg {
    static constexpr int MPAD = MPAD_;                  // UMMA N: padded token count
    // NPROD_ == kScaledLo (HEAL_LO_SCALED, Eq. 10 as printed): as in heal_gemm_umma.cuh every local K segment is walked twice,
    // first the lo'.W products, then the hi.W products whose first MMA scales the accumulator by 2^-10 (scale_input_d); one
    // activation plane per step shares the stage's X slot, the weight tile of the second pass comes out of L2
    static constexpr bool SCALED = NPROD_ == kScaledLo;
    static constexpr int NPROD = SCALED ? 2 : NPROD_;
    static constexpr bool B_MN = B_MN_;                 // weights stored K x N (N contiguous)
    static constexpr bool FUSED = FUSED_;               // split the FP32 activations in the kernel
    static constexpr bool PAIR = PAIR_;                 // large N, no K split, many tokens: two adjacent panels share one
                                                        // cta_group::2 MMA and each CTA stages only HALF of the token tile
                                                        // (at MPAD = 64 the token tile is as large as the weight tile and
                                                        // the L2 -> SM delivery cap, not HBM, bounds the unpaired kernel)
    static constexpr int XROWS = PAIR ? MPAD / 2 : MPAD;// token rows this CTA stages per k-tile
    static constexpr int A_PLANES = NPROD >= 2 ? 2 : 1; // activation planes
    static constexpr int B_PLANES = NPROD >= 3 ? 2 : 1; // weight planes
    static constexpr int W_TILE = kSmallBNW * kBK * 2;  // 16 KB
    static constexpr int X_TILE = XROWS * kBK * 2;
    static constexpr int X_TILE_AL = (X_TILE + 1023) / 1024 * 1024;
    static constexpr int X_SLOTS = SCALED ? 1 : A_PLANES;
    static constexpr int STAGE_BYTES = B_PLANES * W_TILE + X_SLOTS * X_TILE_AL;
    static constexpr int W_BYTES = B_PLANES * W_TILE;
    static constexpr int TX_BYTES = W_BYTES + (FUSED ? 0 : X_SLOTS * X_TILE);
    static constexpr int BAR_BYTES = 512;
    static constexpr int TASKS = MPAD / 16;             // FUSED: 8-float chunks per converter thread per k-tile
    static constexpr int PF = MPAD <= 32 ? 4 : 2;       // FUSED: k-tiles of activations kept in flight in registers
    static_assert(MPAD % 16 == 0 && MPAD >= 16 && MPAD <= 64, "MPAD");
    static_assert(!FUSED || NPROD <= 2, "the fused split needs FP16 weights");
    static_assert(!FUSED || !SCALED, "scaled residual: planes only");
    static_assert(!PAIR || (!FUSED && MPAD >= 32), "pairs: planes only, UMMA N >= 32 across the pair");
};

// One pipeline step of a rank: which local segment (TMEM slot) and k-tile of it, and whether the step opens / closes the
// segment.  Plain: step t -> segment t / 8, k-tile t % 8.  SCALED: a segment of len k-tiles takes 2 len steps, the residual
// pass first.  Only a rank's last local segment can be short (len < 8).
struct SmallStep {
    int seg_j, kk;
    bool lo_pass, first, last;
};
template <bool SCALED>
__device__ __forceinline__ SmallStep small_step(int s, int n_t, int n_local)
{
    SmallStep r;
    if (SCALED) {
        r.seg_j = s / (2 * kTilesPerSeg);
        const int q = s % (2 * kTilesPerSeg);
        const int len = r.seg_j == n_local - 1 ? n_t - (n_local - 1) * kTilesPerSeg : kTilesPerSeg;
        r.lo_pass = q < len;
        r.kk = r.lo_pass ? q : q - len;
        r.first = q == 0;
        r.last = q == 2 * len - 1;
    } else {
        r.seg_j = s >> 3;
        r.kk = s & 7;
        r.lo_pass = false;
        r.first = r.kk == 0;
        r.last = r.kk == 7 || s == n_t - 1;
    }
    return r;
}

struct SmallArgs {
    OutArgs out;          // step E: FP32 C and/or hi/lo planes, optional 2^-p scale
    const float *A;       // FUSED: FP32 activations, row pitch lda (elements)
    int64_t lda;
    int M, N, K;
    int n_seg;            // ceil(K / 512)
    int max_local;        // ceil(n_seg / CS)
    int tmem_cols;        // power of two >= max(32, max_local * MPAD)
    int stages;           // pipeline depth (2..8)
    int rows_per_rank;    // ceil(M / CS): token rows finished by one rank (CS > 1)
    int red_bytes;        // CS > 1: n_seg * rows_per_rank * 128 floats of partial sums pushed by the cluster
    int red_async;        // few pushes per thread: st.async (completion counted in bytes on the owner's mbarrier, no fence,
                          // no arrive); many: plain remote stores + one fence and arrive per warp (higher throughput)
    int red_alias;        // the pushed partial sums reuse the pipeline stages (large M * K): needs a second cluster
                          // barrier ("every rank's main loop is over") before anybody pushes
    int early_push;       // CS > 1, dedicated partial-sum area, several local segments: every finished segment is committed on its own
                          // barrier and pushed while the next ones still stream
    int ring;             // CS == 1, planes: number of TMEM slots the segments cycle through (0 = every local
                          // segment keeps its own slot until the end)
    int b_static;         // HEAL_B_STATIC: W may be read before the stream predecessor has completed
    int *diag;
    unsigned long long *trace;   // phase stamps (HEAL_TRACE builds only), else unused
};

template <class Cfg>
__global__ void __launch_bounds__(kSmallThreads, Cfg::MPAD >= 32 ? 3 : 0)
heal_gemm_smallm_kernel(const __grid_constant__ CUtensorMap tm_x_hi, const __grid_constant__ CUtensorMap tm_x_lo,
                        const __grid_constant__ CUtensorMap tm_w_hi, const __grid_constant__ CUtensorMap tm_w_lo,
                        const SmallArgs args)
{
    constexpr int MPAD = Cfg::MPAD, NPROD = Cfg::NPROD;
    constexpr bool FUSED = Cfg::FUSED;
    // 128B-swizzled tiles need a 1024-byte aligned base.  The dynamic shared memory window of a kernel without static
    // shared memory starts 1024-aligned; the host therefore reserves no slack (which keeps two of the largest CTAs on
    // one SM: M = 64, K = 14336 decode 79 -> 51 us), and a launch that ever got a misaligned base fails loudly.
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t smem_base = smem_u32(smem_raw);
    if ((smem_base & 1023u) != 0u) {
        if (threadIdx.x == 0 && args.diag) {
            args.diag[0] = 900;
            args.diag[1] = static_cast<int>(smem_base);
        }
        __trap();
    }
    // layout: [pipeline stages][partial sums pushed by the cluster][barriers]; with red_alias the partial sums
    // overlay the pipeline stages instead
    const int STAGES = args.stages;
    constexpr bool PAIR = Cfg::PAIR;
    // cluster = the CS ranks that split K of one panel, or (PAIR) the two panels of one cta_group::2 MMA
    const uint32_t cs = PAIR ? 1u : cluster_nctarank();
    const uint32_t rank = PAIR ? 0u : cluster_ctarank();
    const uint32_t prank = PAIR ? cluster_ctarank() : 0u;          // 0 = leader of the pair
    const uint32_t pipe_bytes = static_cast<uint32_t>(STAGES) * Cfg::STAGE_BYTES;
    const uint32_t red_base = args.red_alias ? smem_base : smem_base + pipe_bytes;
    const uint32_t bar_base = args.red_alias ? smem_base + max(pipe_bytes, static_cast<uint32_t>(args.red_bytes))
                                             : red_base + static_cast<uint32_t>(args.red_bytes);
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 64u + 8u * s; };
    auto xfull_bar = [&](int s) { return bar_base + 128u + 8u * s; };
    const uint32_t done_bar = bar_base + 192u;
    const uint32_t red_bar = bar_base + 200u;
    const uint32_t tmem_slot = bar_base + 208u;
    auto tfull_bar = [&](int j) { return bar_base + 256u + 8u * j; };      // ring: slot j holds a finished segment
    auto tempty_bar = [&](int j) { return bar_base + 384u + 8u * j; };     // ring: slot j has been drained (4 warps)
    const int ring = args.ring;
    volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) HEAL_STAMP(args.trace, 0);
    const int panel = PAIR ? static_cast<int>(blockIdx.x) : static_cast<int>(blockIdx.x / cs);
    const int n0 = panel * kSmallBNW;
    const int k_tiles = (args.K + kBK - 1) / kBK;
    const int n_local = (args.n_seg > static_cast<int>(rank)) ? (args.n_seg - 1 - static_cast<int>(rank)) / static_cast<int>(cs) + 1 : 0;
    // local k-tiles, flattened: t -> slot j = t / 8, k-tile (rank + j*cs) * 8 + t % 8; only the last segment
    // of K can be short, and it is the last slot of the rank that owns it
    int n_t = 0;
    if (n_local > 0) {
        const int last_seg = static_cast<int>(rank) + (n_local - 1) * static_cast<int>(cs);
        n_t = (n_local - 1) * kTilesPerSeg + (min(k_tiles, (last_seg + 1) * kTilesPerSeg) - last_seg * kTilesPerSeg);
    }
    const int n_steps = Cfg::SCALED ? 2 * n_t : n_t;     // pipeline steps (SCALED: every k-tile of W travels twice)
    // ranks that finish at least one token row (rank r owns rows [r * rows_per_rank, (r + 1) * rows_per_rank))
    const int owners = cs > 1 ? (args.M + args.rows_per_rank - 1) / args.rows_per_rank : 1;

    if (warp == 0 && lane == 0) {
        if (!FUSED) {
            tma_prefetch_desc(&tm_x_hi);
            if (Cfg::A_PLANES == 2) tma_prefetch_desc(&tm_x_lo);
        }
        tma_prefetch_desc(&tm_w_hi);
        if (Cfg::B_PLANES == 2) tma_prefetch_desc(&tm_w_lo);
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(full_bar(s), PAIR ? 2 : 1);        // PAIR: lives in the leader, one arrive.expect_tx per producer
            mbar_init(empty_bar(s), 1);
            mbar_init(xfull_bar(s), 4);                  // one arrival per converter warp
        }
        mbar_init(done_bar, 1);
        mbar_init(red_bar, args.red_async ? 1 : cs * 4); // async: completes when every pushed byte has landed;
                                                         // else one arrival per epilogue warp of every rank
        if (args.early_push)                                   // (no ring in a cluster: the slots' barriers are free)
            for (int j = 0; j < args.max_local; ++j) mbar_init(tfull_bar(j), 1);
        for (int j = 0; j < ring; ++j) {
            mbar_init(tfull_bar(j), 1);
            mbar_init(tempty_bar(j), PAIR ? 8 : 4);      // PAIR: lives in the leader, 4 epilogue warps of each CTA
        }
        fence_mbar_init();
        if (cs > 1 && args.red_async && static_cast<int>(rank) < owners) {
            // this rank finishes rows [rank * rpr, ...): every rank pushes, per segment and column, one vector per started
            // group of VW owned rows (VW = 4 / 2 / 1 by the divisibility of rpr)
            const int rpr = args.rows_per_rank;
            const int rows = min(rpr, args.M - static_cast<int>(rank) * rpr);
            const int vw = (rpr & 3) == 0 ? 4 : ((rpr & 1) == 0 ? 2 : 1);
            mbar_arrive_expect_tx(red_bar, static_cast<uint32_t>(args.n_seg) * kSmallBNW * static_cast<uint32_t>((rows + vw - 1) / vw * vw) * 4u);
        }
    }
    if (warp == 1) {
        if (PAIR) {
            tmem_alloc_2cta(tmem_slot, static_cast<uint32_t>(args.tmem_cols));
            tmem_relinquish_2cta();
        } else {
            tmem_alloc(tmem_slot, static_cast<uint32_t>(args.tmem_cols));
            tmem_relinquish();
        }
        if (lane == 0) HEAL_STAMP(args.trace, 13);
    }
    if (FUSED) {
        // token rows >= M of the operand tiles are never written by the converters: zero them once
        for (int s = 0; s < STAGES; ++s) {
            const uint32_t sx = smem_base + s * Cfg::STAGE_BYTES + Cfg::W_BYTES;
            for (int o = threadIdx.x * 16; o < Cfg::A_PLANES * Cfg::X_TILE_AL; o += kSmallThreads * 16)
                asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(sx + o), "r"(0u) : "memory");
        }
        fence_proxy_async_smem();
    }
    tc_fence_before();
    __syncthreads();
    if (threadIdx.x == 0) HEAL_STAMP(args.trace, 12);
    if (PAIR) cluster_sync_all();                        // the peer's barriers exist before any remote arrive / commit
    if (cs > 1) cluster_arrive_relaxed();                // matched by cluster_wait() before the first remote access
                                                         // (the barrier inits were published by fence.mbarrier_init)
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;
    if (threadIdx.x == 0) HEAL_STAMP(args.trace, 1);
    const bool early_w = args.b_static != 0 && warp == 0;
    if (!early_w) {
        pdl_wait();                   // everything above overlapped the previous kernel's tail
        pdl_launch_dependents();      // the next kernel may start its prologue (and, with static weights, its W stream)
    }
    if (threadIdx.x == 32) HEAL_STAMP(args.trace, 2);

    if (warp == 0) {
        // ================================ TMA producer ================================
        if (lane == 0) {
            const uint64_t pol_w = l2_policy_evict_first();      // weights are streamed once
            // one TMA box; PAIR: the completion barrier is the leader's (cta_group::2 form of the copy)
            auto ld_w = [&](uint32_t dst, const CUtensorMap *m, uint32_t fb, int x, int y) {
                if (PAIR) tma_load_2d_2cta_hint(dst, m, fb, x, y, pol_w);
                else      tma_load_2d_hint(dst, m, fb, x, y, pol_w);
            };
            auto ld_x = [&](uint32_t dst, const CUtensorMap *m, uint32_t fb, int x, int y) {
                if (PAIR) tma_load_2d_2cta(dst, m, fb, x, y);
                else      tma_load_2d(dst, m, fb, x, y);
            };
            auto expect = [&](uint32_t fb) {
                if (PAIR) mbar_arrive_expect_tx_cluster(fb, Cfg::TX_BYTES);
                else      mbar_arrive_expect_tx(fb, Cfg::TX_BYTES);
            };
            auto fbar = [&](int st) { return PAIR ? leader_addr(full_bar(st)) : full_bar(st); };
            auto load_w = [&](int t, uint32_t sb, uint32_t fb) {
                const SmallStep sp = small_step<Cfg::SCALED>(t, n_t, n_local);
                const int k0 = ((static_cast<int>(rank) + sp.seg_j * static_cast<int>(cs)) * kTilesPerSeg + sp.kk) * kBK;
                if (Cfg::B_MN) {
#pragma unroll
                    for (int c = 0; c < 2; ++c) {
                        ld_w(sb + c * 8192, &tm_w_hi, fb, n0 + c * 64, k0);
                        if (Cfg::B_PLANES == 2) ld_w(sb + Cfg::W_TILE + c * 8192, &tm_w_lo, fb, n0 + c * 64, k0);
                    }
                } else {
                    ld_w(sb, &tm_w_hi, fb, k0, n0);
                    if (Cfg::B_PLANES == 2) ld_w(sb + Cfg::W_TILE, &tm_w_lo, fb, k0, n0);
                }
            };
            auto load_x = [&](int t, uint32_t sb, uint32_t fb) {
                const SmallStep sp = small_step<Cfg::SCALED>(t, n_t, n_local);
                const int k0 = ((static_cast<int>(rank) + sp.seg_j * static_cast<int>(cs)) * kTilesPerSeg + sp.kk) * kBK;
                const uint32_t sx = sb + Cfg::W_BYTES;
                const int m_first = static_cast<int>(prank) * Cfg::XROWS;          // PAIR: this CTA's half of the tokens
                if (Cfg::SCALED) {
                    ld_x(sx, sp.lo_pass ? &tm_x_lo : &tm_x_hi, fb, k0, m_first);
                } else {
                    ld_x(sx, &tm_x_hi, fb, k0, m_first);
                    if (Cfg::A_PLANES == 2) ld_x(sx + Cfg::X_TILE_AL, &tm_x_lo, fb, k0, m_first);
                }
            };
            int stage = 0, t = 0;
            uint32_t phase = 0;
            if (early_w && !FUSED) {
                // static weights: fill the pipeline with W tiles now, add the activation tiles once the
                // stream predecessor (which may have produced them) has completed
                const int pre = min(STAGES, n_steps);
                for (int s = 0; s < pre; ++s) {
                    expect(fbar(s));
                    load_w(s, smem_base + s * Cfg::STAGE_BYTES, fbar(s));
                }
                HEAL_STAMP(args.trace, 3);
                pdl_wait();
                for (int s = 0; s < pre; ++s) load_x(s, smem_base + s * Cfg::STAGE_BYTES, fbar(s));
                t = pre;
                if (pre == STAGES) phase = 1u; else stage = pre;
            }
            for (; t < n_steps; ++t) {
                mbar_wait_ool(empty_bar(stage), phase ^ 1u, args.diag, 500 + stage);
                const uint32_t sb = smem_base + stage * Cfg::STAGE_BYTES;
                const uint32_t fb = fbar(stage);
                expect(fb);
                load_w(t, sb, fb);
                if (!FUSED) load_x(t, sb, fb);
                if (t == 0) HEAL_STAMP(args.trace, 3);
                if (++stage == STAGES) { stage = 0; phase ^= 1u; }
            }
        }
        if (cs > 1 && args.red_alias) {
            __syncwarp();
            mbar_wait_ool(done_bar, 0, args.diag, 701);
            cluster_wait();
            cluster_arrive_relaxed();          // "my pipeline is dead": observed through done_bar, no data to publish
        }
    } else if (warp == 1) {
        // ================================ MMA issuer ==================================
        if (lane == 0 && prank == 0) {
            // D[n][m] = sum_k W[k][n] * X[m][k]: UMMA A = weights (128 rows per CTA), UMMA B = tokens (N = MPAD;
            // PAIR: 256 weight rows over the two CTAs, each holding half of the token rows)
            constexpr uint32_t idesc = umma_idesc_f16_f32(PAIR ? 2 * kSmallBNW : kSmallBNW, MPAD, Cfg::B_MN ? 1u : 0u, 0u);
            auto mma = [&](uint32_t d, uint64_t a, uint64_t b, uint32_t acc) {
                if (PAIR) umma_f16_2cta(d, a, b, idesc, acc);
                else      umma_f16(d, a, b, idesc, acc);
            };
            auto mma_scale_d = [&](uint32_t d, uint64_t a, uint64_t b) {      // D = a.b + D * 2^-kLoShift
                if (PAIR) umma_f16_2cta_scale_d<kLoShift>(d, a, b, idesc);
                else      umma_f16_scale_d<kLoShift>(d, a, b, idesc);
            };
            auto commit = [&](uint32_t bar) {                  // PAIR: the barrier at this offset in both CTAs
                if (PAIR) umma_commit_2cta(bar, 3);
                else      umma_commit(bar);
            };
            constexpr uint64_t kdesc0 = umma_smem_desc_sw128(0, 16, 1024);                 // K-major SW128
            constexpr uint64_t wdesc0 = Cfg::B_MN ? umma_smem_desc_sw128(0, kBK * 128, 1024) : kdesc0;
            constexpr uint32_t w_step = (Cfg::B_MN ? 16 * 128 : 32) >> 4;
            constexpr uint32_t x_step = 32 >> 4;
            int stage = 0;
            uint32_t phase = 0;
            uint32_t accumulate = 0;
            const int seg_commit = ring | args.early_push;        // (early push: at most 16 local segments, slot = local segment)
            for (int t = 0; t < n_steps; ++t) {
                const SmallStep sp = small_step<Cfg::SCALED>(t, n_t, n_local);
                const int seg_j = sp.seg_j;
                const int slot = ring ? seg_j % ring : seg_j;
                if (sp.first) {                                   // new segment -> next TMEM slot
                    accumulate = 0;
                    if (ring && seg_j >= ring) {                  // the slot's previous segment must have been drained
                        mbar_wait_ool(tempty_bar(slot), static_cast<uint32_t>((seg_j / ring - 1) & 1), args.diag, 640 + slot);
                        tc_fence_after();
                    }
                }
                const uint32_t d_tmem = tmem_base + static_cast<uint32_t>(slot * MPAD);
                mbar_wait_ool(full_bar(stage), phase, args.diag, 600 + stage);
                if (FUSED) mbar_wait_ool(xfull_bar(stage), phase, args.diag, 620 + stage);
                tc_fence_after();
                if (t == 0) HEAL_STAMP(args.trace, 4);
                if (t == n_steps - 1) HEAL_STAMP(args.trace, 5);
                const uint32_t sb = smem_base + stage * Cfg::STAGE_BYTES;
                const uint64_t w_hi = wdesc0 | desc_addr(sb);
                const uint64_t w_lo = wdesc0 | desc_addr(sb + Cfg::W_TILE);
                const uint32_t sx = sb + Cfg::W_BYTES;
                const uint64_t x_hi = kdesc0 | desc_addr(sx);
                const uint64_t x_lo = kdesc0 | desc_addr(sx + Cfg::X_TILE_AL);
#pragma unroll
                for (int q = 0; q < kBK / 16; ++q) {
                    const uint64_t wo = static_cast<uint64_t>(q * w_step), xo = static_cast<uint64_t>(q * x_step);
                    if (Cfg::SCALED) {                     // x_hi is the step's plane: the residual in the first pass
                        if (!sp.lo_pass && sp.kk == 0 && q == 0) mma_scale_d(d_tmem, w_hi + wo, x_hi + xo);
                        else                                     mma(d_tmem, w_hi + wo, x_hi + xo, accumulate);
                        accumulate = 1;
                        continue;
                    }
                    // product order as in the large-M kernel: a_hi.b_hi, a_hi.b_lo, a_lo.b_hi, a_lo.b_lo
                    mma(d_tmem, w_hi + wo, x_hi + xo, accumulate);
                    accumulate = 1;
                    if (NPROD == 2) mma(d_tmem, w_hi + wo, x_lo + xo, 1);
                    if (NPROD >= 3) {
                        mma(d_tmem, w_lo + wo, x_hi + xo, 1);
                        mma(d_tmem, w_hi + wo, x_lo + xo, 1);
                    }
                    if (NPROD == 4) mma(d_tmem, w_lo + wo, x_lo + xo, 1);
                }
                commit(empty_bar(stage));
                if (seg_commit && sp.last) commit(tfull_bar(slot));                            // segment complete (ring / early push)
                if (++stage == STAGES) { stage = 0; phase ^= 1u; }
            }
            commit(done_bar);                              // all local segments complete in TMEM
        }
        if (cs > 1 && args.red_alias) {
            __syncwarp();
            mbar_wait_ool(done_bar, 0, args.diag, 702);
            cluster_wait();
            cluster_arrive_relaxed();          // "my pipeline is dead": observed through done_bar, no data to publish
        }
    } else {
        const int et = threadIdx.x - 64;                   // 0..127 among the converter / epilogue threads
        if (FUSED) {
            // ============================ step S: FP32 activations -> hi/lo operand tiles ==========
            // Thread `et` owns 16-byte chunk c = et % 8 (k = 8c..8c+7 of the k-tile) of token rows
            // et/8, et/8 + 16, ...; K-major 128B-swizzled tile: row m at (m/8)*1024 + (m%8)*128, chunk c
            // stored at position c ^ (m%8).
            constexpr int TASKS = Cfg::TASKS, PF = Cfg::PF;
            const int c = et & 7, r0 = et >> 3;
            float4 buf[PF][TASKS][2];
            auto fetch = [&](int t, float4 (&dst)[TASKS][2]) {
                const int k = ((static_cast<int>(rank) + (t >> 3) * static_cast<int>(cs)) * kTilesPerSeg + (t & 7)) * kBK + c * 8;
#pragma unroll
                for (int q = 0; q < TASKS; ++q) {
                    const int m = r0 + q * 16;
                    dst[q][0] = dst[q][1] = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (m < args.M) {
                        const float *src = args.A + static_cast<int64_t>(m) * args.lda + k;
                        if (k + 8 <= args.K) {
                            dst[q][0] = __ldg(reinterpret_cast<const float4 *>(src));
                            dst[q][1] = __ldg(reinterpret_cast<const float4 *>(src) + 1);
                        } else {
                            float v[8];
#pragma unroll
                            for (int i = 0; i < 8; ++i) v[i] = (k + i < args.K) ? __ldg(src + i) : 0.f;
                            dst[q][0] = make_float4(v[0], v[1], v[2], v[3]);
                            dst[q][1] = make_float4(v[4], v[5], v[6], v[7]);
                        }
                    }
                }
            };
#pragma unroll
            for (int p = 0; p < PF; ++p)
                if (p < n_t) fetch(p, buf[p]);
            int stage = 0;
            uint32_t phase = 0;
            for (int t0 = 0; t0 < n_t; t0 += PF) {
#pragma unroll
                for (int p = 0; p < PF; ++p) {
                    const int t = t0 + p;
                    if (t < n_t) {
                        mbar_wait_ool(empty_bar(stage), phase ^ 1u, args.diag, 540 + stage);
                        const uint32_t sx = smem_base + stage * Cfg::STAGE_BYTES + Cfg::W_BYTES;
#pragma unroll
                        for (int q = 0; q < TASKS; ++q) {
                            const int m = r0 + q * 16;
                            if (m < args.M) {
                                uint4 h, l;
                                split2(buf[p][q][0].x, buf[p][q][0].y, h.x, l.x);
                                split2(buf[p][q][0].z, buf[p][q][0].w, h.y, l.y);
                                split2(buf[p][q][1].x, buf[p][q][1].y, h.z, l.z);
                                split2(buf[p][q][1].z, buf[p][q][1].w, h.w, l.w);
                                const uint32_t off = static_cast<uint32_t>((m >> 3) * 1024 + (m & 7) * 128 + ((c ^ (m & 7)) << 4));
                                asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(sx + off), "r"(h.x), "r"(h.y), "r"(h.z), "r"(h.w) : "memory");
                                if (Cfg::A_PLANES == 2)
                                    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(sx + Cfg::X_TILE_AL + off), "r"(l.x), "r"(l.y), "r"(l.z), "r"(l.w) : "memory");
                            }
                        }
                        if (r0 < args.M) fence_proxy_async_smem();   // generic-proxy writes -> visible to the tensor core (writers only)
                        __syncwarp();
                        if (lane == 0) mbar_arrive(xfull_bar(stage));
                        if (t + PF < n_t) fetch(t + PF, buf[p]);
                        if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                    }
                }
            }
        }
        // ================================ epilogue ====================================
        const int quad = warp & 3;
        const int nl = quad * 32 + lane;                   // weight column within the panel = TMEM lane
        const int col = n0 + nl;
        int Mr = args.M;                                   // kept in a register: the unrolled loops test it per element
        asm volatile("" : "+r"(Mr));
        if (cs == 1 && ring) {
            // single-CTA panel, ring of TMEM slots: drain each finished segment into the ascending FP32 RN running sum
            // while the tensor core fills the next slot
            float acc[MPAD / 16][16];
            for (int j = 0; j < n_local; ++j) {
                const int slot = j % ring;
                mbar_wait_ool(tfull_bar(slot), static_cast<uint32_t>((j / ring) & 1), args.diag, 660 + slot);
                tc_fence_after();
#pragma unroll
                for (int c = 0; c < MPAD / 16; ++c) {
                    if (c * 16 < Mr) {
                        uint32_t v[16];
                        tmem_ld_32x32b_x16(tmem_base + (static_cast<uint32_t>(quad * 32) << 16) + static_cast<uint32_t>(slot * MPAD + c * 16), v);
                        tmem_ld_wait();
                        if (j == 0) {
#pragma unroll
                            for (int i = 0; i < 16; ++i) acc[c][i] = __uint_as_float(v[i]);
                        } else {
#pragma unroll
                            for (int i = 0; i < 16; ++i) acc[c][i] = __fadd_rn(acc[c][i], __uint_as_float(v[i]));
                        }
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) {
                    if (PAIR) mbar_arrive_cluster(leader_addr(tempty_bar(slot)));
                    else      mbar_arrive(tempty_bar(slot));
                }
            }
            if (et == 0) HEAL_STAMP(args.trace, 6);
            if (col < args.N) {
                emit_dispatch(args.out, [&](const OutArgs &po, auto fast) {
#pragma unroll
                    for (int c = 0; c < MPAD / 16; ++c)
#pragma unroll
                        for (int i = 0; i < 16; ++i)
                            if (c * 16 + i < Mr) emit1<decltype(fast)::value>(po, c * 16 + i, col, acc[c][i]);
                });
            }
            if (et == 0) HEAL_STAMP(args.trace, 7);
            mbar_wait_ool(done_bar, 0, args.diag, 700);        // every MMA (and its commits) has retired before the CTA leaves
            tc_fence_after();
            tc_fence_before();
            if (et == 0) HEAL_STAMP(args.trace, 8);
        } else {
        // the cluster barrier of the prologue ("every rank's red_bar is initialised") is collected here, while the tensor core
        // is still busy, instead of between the last commit and the first push (barrier.cluster.wait.acquire costs ~0.2 us)
        if (cs > 1) cluster_wait();
        if (!args.early_push) {
            mbar_wait_ool(done_bar, 0, args.diag, 700);
            tc_fence_after();
        }
        if (et == 0) HEAL_STAMP(args.trace, 6);
        if (cs == 1) {
            // single-CTA panel: all segments are local slots; sum them in ascending order in registers
#pragma unroll
            for (int c = 0; c < MPAD / 16; ++c) {
                if (c * 16 < Mr) {
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
                        emit_dispatch(args.out, [&](const OutArgs &po, auto fast) {
#pragma unroll
                            for (int i = 0; i < 16; ++i)
                                if (c * 16 + i < Mr) emit1<decltype(fast)::value>(po, c * 16 + i, col, acc[i]);
                        });
                    }
                }
            }
            tc_fence_before();
        } else {
            if (args.red_alias) {                          // every rank's pipeline buffers are dead
                cluster_arrive_relaxed();
                cluster_wait();
            }
            // push this rank's partials: token m -> rank m / rpr; its red area holds, per segment, [nl][rpr] floats, or for
            // rpr % 4 == 0 [rpr / 4][nl] 16-byte vectors of four consecutive rows
            const int rpr = args.rows_per_rank;
            for (int j = 0; j < n_local; ++j) {
                if (args.early_push) {                     // this segment's MMAs have retired (the later ones may still be running)
                    mbar_wait_ool(tfull_bar(j), 0, args.diag, 730);
                    tc_fence_after();
                }
                const int seg = static_cast<int>(rank) + j * static_cast<int>(cs);
                const uint32_t row_off = static_cast<uint32_t>((seg * kSmallBNW + nl) * rpr) * 4u;
#pragma unroll
                for (int c = 0; c < MPAD / 16; ++c) {
                    if (c * 16 < Mr) {
                        uint32_t v[16];
                        tmem_ld_32x32b_x16(tmem_base + (static_cast<uint32_t>(quad * 32) << 16) + static_cast<uint32_t>(j * MPAD + c * 16), v);
                        tmem_ld_wait();
                        const bool async = args.red_async != 0;
                        // rows_per_rank is 1, 2 or a multiple of 4 (host): the owner rank and the row inside its block follow from
                        // shifts, or are stepped along from one division per chunk.  Past the last token the 16-token kernels leave the
                        // loop; the 32- and 64-token ones skip the iteration (leaving costs them 30-70 registers, i.e. a CTA per SM).
                        // This code runs once, on the latency-critical tail, with one warp per scheduler: 16 iterations that each stepped the
                        // owner with a data-dependent loop cost 1100 cycles per segment at M = 1 (clock stamps), this form about 100.
#define HEAL_PAST_LAST_TOKEN if constexpr (MPAD == 16) break; else continue
                        if ((rpr & 3) == 0) {
                            uint32_t dst = static_cast<uint32_t>((c * 16) / rpr), ml = static_cast<uint32_t>((c * 16) % rpr);
#pragma unroll
                            for (int i = 0; i < 16; i += 4) {
                                if (c * 16 + i >= Mr) { HEAL_PAST_LAST_TOKEN; }      // rows m..m+3 have one owner (rows >= M: unused zeros)
                                // groups of four rows are the slow index: a warp's vector stores land on 512 contiguous bytes
                                const uint32_t a = map_to_cta(red_base + ((static_cast<uint32_t>(seg * (rpr >> 2)) + (ml >> 2)) * kSmallBNW + nl) * 16u, dst);
                                if (async) st_async_v4(a, v[i], v[i + 1], v[i + 2], v[i + 3], map_to_cta(red_bar, dst));
                                else       st_dsmem_v4(a, v[i], v[i + 1], v[i + 2], v[i + 3]);
                                ml += 4;
                                if (ml == static_cast<uint32_t>(rpr)) { ml = 0; ++dst; }
                            }
                        } else if (rpr == 2 && async) {
#pragma unroll
                            for (int i = 0; i < 16; i += 2) {
                                if (c * 16 + i >= Mr) { HEAL_PAST_LAST_TOKEN; }
                                const uint32_t dst = static_cast<uint32_t>(c * 16 + i) >> 1;
                                st_async_v2(map_to_cta(red_base + row_off, dst), v[i], v[i + 1], map_to_cta(red_bar, dst));
                            }
                        } else {                                  // one row per rank (or two, plain stores)
                            const uint32_t sh = static_cast<uint32_t>(rpr) - 1u;            // 0 or 1
#pragma unroll
                            for (int i = 0; i < 16; ++i) {
                                if (c * 16 + i >= Mr) { HEAL_PAST_LAST_TOKEN; }
                                const uint32_t m = static_cast<uint32_t>(c * 16 + i), dst = m >> sh, ml = m & sh;
                                const uint32_t a = map_to_cta(red_base + row_off + ml * 4u, dst);
                                if (async) st_async_b32(a, v[i], map_to_cta(red_bar, dst));
                                else       st_dsmem_b32(a, v[i]);
                            }
                        }
                    }
                }
            }
#undef HEAL_PAST_LAST_TOKEN
            if (args.early_push) mbar_wait_ool(done_bar, 0, args.diag, 731);       // every MMA (and its commits) has retired
            tc_fence_before();
            if (!args.red_async) {
                __syncwarp();
                // one fence per signalling lane (cumulative over the warp's pushes, ordered by the __syncwarp) and a
                // relaxed remote arrive: a cluster-scope release costs ~0.5 us each on this part (measured), so pay it once
                if (lane < owners) {
                    fence_acq_rel_cluster();
                    mbar_arrive_relaxed_cluster(map_to_cta(red_bar, static_cast<uint32_t>(lane)));
                }
            }
            tc_fence_before();
            if (et == 0) HEAL_STAMP(args.trace, 7);
            if (static_cast<int>(rank) < owners) {
                if (args.red_async) mbar_wait_ool(red_bar, 0, args.diag, 710);       // every byte has landed
                else                mbar_wait_cluster(red_bar, 0, args.diag, 710);
                if (et == 0) HEAL_STAMP(args.trace, 8);
                // this rank finishes rows [rank * rpr, min(M, (rank + 1) * rpr)): ascending segment order, FP32 RN
                const float *red = reinterpret_cast<const float *>(smem_raw + (red_base - smem_u32(smem_raw)));
                const int m_lo = static_cast<int>(rank) * rpr;
                const int rows = min(rpr, args.M - m_lo);
                const int seg_stride = kSmallBNW * rpr;
                if ((rpr & 3) == 0) {
                    for (int r4 = 0; r4 < rows; r4 += 4) {
                        const float4 *src = reinterpret_cast<const float4 *>(red) + (r4 >> 2) * kSmallBNW + nl;
                        float4 acc = src[0];
#pragma unroll 4
                        for (int s = 1; s < args.n_seg; ++s) {
                            const float4 v = src[static_cast<size_t>(s) * (seg_stride / 4)];
                            acc.x = __fadd_rn(acc.x, v.x); acc.y = __fadd_rn(acc.y, v.y);
                            acc.z = __fadd_rn(acc.z, v.z); acc.w = __fadd_rn(acc.w, v.w);
                        }
                        if (col < args.N) {
                            emit_dispatch(args.out, [&](const OutArgs &po, auto fast) {
                                constexpr bool kf = decltype(fast)::value;
                                emit1<kf>(po, m_lo + r4, col, acc.x);
                                if (r4 + 1 < rows) emit1<kf>(po, m_lo + r4 + 1, col, acc.y);
                                if (r4 + 2 < rows) emit1<kf>(po, m_lo + r4 + 2, col, acc.z);
                                if (r4 + 3 < rows) emit1<kf>(po, m_lo + r4 + 3, col, acc.w);
                            });
                        }
                    }
                } else {
                    for (int r = 0; r < rows; ++r) {
                        const float *src = red + nl * rpr + r;
                        float acc = src[0];
#pragma unroll 4
                        for (int s = 1; s < args.n_seg; ++s) acc = __fadd_rn(acc, src[static_cast<size_t>(s) * seg_stride]);
                        if (col < args.N) {
                            emit_dispatch(args.out, [&](const OutArgs &po, auto fast) {
                                emit1<decltype(fast)::value>(po, m_lo + r, col, acc);
                            });
                        }
                    }
                }
                if (et == 0) HEAL_STAMP(args.trace, 9);
            }
        }
        }
    }

    __syncthreads();
    if (PAIR) cluster_sync_all();                          // the peer may still read this CTA's smem / signal its barriers
    if (threadIdx.x == 64) HEAL_STAMP(args.trace, 9);
    if (warp == 1) {
        tc_fence_after();
        if (PAIR) tmem_dealloc_2cta(tmem_base, static_cast<uint32_t>(args.tmem_cols));
        else      tmem_dealloc(tmem_base, static_cast<uint32_t>(args.tmem_cols));
        if (lane == 0) HEAL_STAMP(args.trace, 11);
    }
}

}  // namespace heal
