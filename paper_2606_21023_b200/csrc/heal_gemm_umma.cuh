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
#include "heal_epilogue.cuh"
#include "heal_ptx.cuh"
#include "heal_sched.h"

namespace heal {

constexpr int kBM = 128;          // UMMA M (rows of A per tile)
constexpr int kGemmThreads = 384;

template <int BN_, int NPROD_, bool B_MN_, bool FULL_ = false>
struct GemmCfg {
    static constexpr bool FULL = FULL_;                 // with the extended epilogue (2^-p scale, chained planes, accumulate) and the
                                                        // ordered split-K schedule; the default instantiation has neither, so the
                                                        // headline path carries no extra registers or code (measured: 2.5 % otherwise)
    static constexpr int BN = BN_;
    // NPROD_ == kScaledLo: the paper's scaled residual (HEAL_LO_SCALED, Eq. 10 as printed) in ONE kernel and ONE
    // accumulator.  Every K segment is walked twice: first all lo'.W products (lo' = r16((x - hi) 2^10)), then the hi.W products, the
    // first of which is issued with scale_input_d = 10, i.e. D = hi_0.W_0 + D * 2^-10 inside the tensor core (an exact power-of-two
    // scaling of the residual sum).  Segment sums are then added in FP32 RN as always.  The weight tile travels twice (64 instead of
    // 48 KB per k-tile and product pair), which is why this is a variant and not the default (measured 1.08x on the MLP
    // GEMMs; round 1 formed it from two one-product launches at 1.55x).
    static constexpr bool SCALED = NPROD_ == kScaledLo;
    static constexpr int NPROD = SCALED ? 2 : NPROD_;
    static constexpr bool B_MN = B_MN_;                 // B stored K x N (N contiguous): MN-major operand
    static constexpr int A_PLANES = NPROD >= 2 ? 2 : 1;
    static constexpr int B_PLANES = NPROD >= 3 ? 2 : 1;
    static constexpr int A_TILE = kBM * kBK * 2;
    static constexpr int B_TILE = BN * kBK * 2;
    static constexpr int A_SLOTS = SCALED ? 1 : A_PLANES;   // SCALED: one activation plane per pass shares the slot
    static constexpr int STAGE_BYTES = A_SLOTS * A_TILE + B_PLANES * B_TILE;
    static constexpr int BAR_BYTES = 256;
    static constexpr int STAGES_RAW = (kSmemLimit - 1024 - BAR_BYTES) / STAGE_BYTES;
    static constexpr int STAGES = STAGES_RAW > 8 ? 8 : STAGES_RAW;
    static constexpr int TMEM_COLS = (2 * BN <= 32) ? 32 : (2 * BN <= 64) ? 64 : (2 * BN <= 128) ? 128 : (2 * BN <= 256) ? 256 : 512;
    // TMEM can never be oversubscribed: a kernel takes at least the same fraction of an SM's shared memory (228 KB, 1 KB
    // reserved per CTA) as of its 512 TMEM columns, so whatever mix of the library's CTAs fits an SM's shared memory also fits its TMEM --
    // a CTA blocked in tcgen05.alloc while cluster peers hold TMEM elsewhere could otherwise close a wait cycle across streams.
    static constexpr int SMEM_USED = 1024 + STAGES * STAGE_BYTES + BAR_BYTES;
    static constexpr int SMEM_TMEM = TMEM_COLS * (228 * 1024 / 512) - 1024;
    static constexpr int SMEM_BYTES = SMEM_USED > SMEM_TMEM ? SMEM_USED : SMEM_TMEM;
    static constexpr int COLS_PER_WARP = BN / 2;
    static_assert(BN % 32 == 0 && BN >= 32 && BN <= 256, "BN");
    static_assert(!B_MN || BN % 64 == 0, "MN-major B tiles are built from 64-column swizzle atoms");
    static_assert(STAGES >= 2, "need at least two stages");
};

struct GemmArgs {
    OutArgs out;            // step E: FP32 C and/or hi/lo planes, optional 2^-p scale
    int M, N, K;
    int tiles_m, tiles_n;
    int group_m;            // row tiles per rasterisation group (heal_sched.h tile_coords)
    int *diag;
    // segment-granular load balancing (0 = plain tile round-robin)
    int balance;
    int dp_tiles;           // tiles dealt whole, round-robin (multiple of the grid size)
    float *xfer;            // per-CTA hand-off slot: kBM * BN floats each
    uint32_t *flags;        // per-CTA flag: 1 once the slot is written, reset to 0 by its consumer
    // ordered split-K (few tiles, many CTAs): every (tile, segment) partial goes to `part`; heal_splitk_reduce_kernel,
    // launched right behind, adds them in ascending segment order and runs the epilogue
    int sk;
    float *part;            // [(tile * R + rank) * n_seg + seg] x (kBM * BN) floats, R = CTAs per tile
};

// ---- epilogue building blocks shared by the single-CTA and the CTA-pair kernel (256 epilogue threads, etid = 0..255;
// a thread owns accumulator row quad*32+lane and CPW consecutive columns, kept as the FP32 running sum run[CPW]) -------

// one finished K segment: TMEM -> registers, FP32 RN add into the running sum (the first segment initialises it)
template <int CPW>
__device__ __forceinline__ void epi_add_segment(uint32_t taddr, float (&run)[CPW], bool first)
{
#pragma unroll
    for (int c = 0; c < CPW / 16; ++c) {
        uint32_t v[16];
        tmem_ld_32x32b_x16(taddr + c * 16, v);
        tmem_ld_wait();
        if (first) {
#pragma unroll
            for (int i = 0; i < 16; ++i) run[c * 16 + i] = __uint_as_float(v[i]);
        } else {
#pragma unroll
            for (int i = 0; i < 16; ++i) run[c * 16 + i] = __fadd_rn(run[c * 16 + i], __uint_as_float(v[i]));
        }
    }
}

// Balanced schedule, tail of a shared tile: start from the running sum (segments 0..sb-1) that the neighbouring CTA
// (or CTA pair) parked in `slot`, once its `flag` is up; the flag is re-armed for the next launch (launches on a stream
// are serialised, and 0/1 flags -- unlike launch counters -- stay correct when a captured graph is replayed).
// Progress: the producer is the CTA with the next lower index (same rank of the previous pair), which runs this tile's
// head FIRST and never waits before it has parked the sum; it is resident whenever this CTA is, because the grid has at
// most one CTA per SM and the launch is cooperative (all CTAs co-resident, see launch_gemm*_cfg) -- and even without
// that guarantee blocks are dispatched in index order, so a lower-indexed block is never scheduled later.
template <int CPW>
__device__ __forceinline__ void epi_take_prefix(const float *slot, uint32_t *flag, float (&run)[CPW], int etid, int *diag)
{
    if (etid == 0) {
        const uint64_t t0 = globaltimer_ns();
        uint32_t f;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(f) : "l"(flag) : "memory");
            if (f == 0u && globaltimer_ns() - t0 > 4000000000ull) {
                diag[0] = 800;
                diag[1] = static_cast<int>(blockIdx.x);
                __trap();
            }
        } while (f == 0u);
    }
    asm volatile("bar.sync 1, 256;" ::: "memory");
    const float4 *src = reinterpret_cast<const float4 *>(slot);
#pragma unroll
    for (int c = 0; c < CPW / 4; ++c) {
        float4 v;
        asm volatile("ld.global.cg.v4.f32 {%0, %1, %2, %3}, [%4];"
                     : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(src + c * 256 + etid) : "memory");
        run[c * 4] = v.x; run[c * 4 + 1] = v.y; run[c * 4 + 2] = v.z; run[c * 4 + 3] = v.w;
    }
    asm volatile("bar.sync 1, 256;" ::: "memory");
    if (etid == 0) asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(flag), "r"(0u) : "memory");
}
// Balanced schedule, head of a shared tile: hand the running sum to the next CTA (pair)
template <int CPW>
__device__ __forceinline__ void epi_hand_on(float *slot, uint32_t *flag, const float (&run)[CPW], int etid)
{
    float4 *dst = reinterpret_cast<float4 *>(slot);
#pragma unroll
    for (int c = 0; c < CPW / 4; ++c)
        dst[c * 256 + etid] = make_float4(run[c * 4], run[c * 4 + 1], run[c * 4 + 2], run[c * 4 + 3]);
    __threadfence();
    asm volatile("bar.sync 1, 256;" ::: "memory");
    if (etid == 0) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(flag), "r"(1u) : "memory");
}
// final store of a thread's row segment: plain FP32 (lean instantiation) or the extended epilogue
template <int CPW, bool FULL>
__device__ __forceinline__ void epi_store(const OutArgs &out, int row, int col0, const float (&run)[CPW], int M, int N)
{
    if (row >= M) return;
    if constexpr (FULL) {
        emit_dispatch(out, [&](const OutArgs &po, auto fast) {
#pragma unroll
            for (int c = 0; c < CPW; c += 4)
                emit4<decltype(fast)::value>(po, row, col0 + c, make_float4(run[c], run[c + 1], run[c + 2], run[c + 3]), N);
        });
    } else {
        float *crow = out.C + static_cast<int64_t>(row) * out.ldc;
#pragma unroll
        for (int c = 0; c < CPW; c += 4) emit4_plain(crow, col0 + c, make_float4(run[c], run[c + 1], run[c + 2], run[c + 3]), N);
    }
}

// ---- ordered split-K (few tiles, many SMs) -------------------------------------------------------------------------
// The (tile, K segment) units are dealt to more CTAs than there are tiles; every segment partial is parked in global
// memory by the GEMM kernel and a second, dependent kernel (heal_splitk_reduce_kernel, programmatic dependent launch)
// adds the n_seg partials of every element in ascending segment order in FP32 RN and runs the epilogue.  No CTA ever
// waits for another one: nothing depends on which CTAs are resident, and no counters have to be re-armed.
// Partial layout: float4 index c4 * 256 + etid, c4 = 0..CPW/4-1 (the thread's columns 4*c4..4*c4+3): coalesced for the
// writer and for the reducer, which use the same thread mapping.
template <int CPW>
__device__ __forceinline__ void sk_store_partial(float *part, uint32_t taddr, int etid)
{
    float4 *dst = reinterpret_cast<float4 *>(part);
#pragma unroll
    for (int c = 0; c < CPW / 16; ++c) {
        uint32_t v[16];
        tmem_ld_32x32b_x16(taddr + c * 16, v);
        tmem_ld_wait();
#pragma unroll
        for (int q = 0; q < 4; ++q)
            dst[(c * 4 + q) * 256 + etid] = make_float4(__uint_as_float(v[4 * q]), __uint_as_float(v[4 * q + 1]),
                                                        __uint_as_float(v[4 * q + 2]), __uint_as_float(v[4 * q + 3]));
    }
}

// grid = units * shares CTAs of 256 threads; unit = tile * R + rank (R = CTAs per tile: 1, or 2 for CTA pairs); CTA
// `share` finishes float4 chunks [share*NC/shares, (share+1)*NC/shares) of every row of the unit's 128 x BN block.
template <int BN>
__global__ void __launch_bounds__(256)
heal_splitk_reduce_kernel(const float *__restrict__ part, int n_seg, int R, int tiles_m, int tiles_n, int group_m, int shares, const OutArgs out, int M, int N)
{
    pdl_wait();
    pdl_launch_dependents();
    constexpr int CPW = BN / 2, NC = CPW / 4;
    const int unit = static_cast<int>(blockIdx.x) / shares, share = static_cast<int>(blockIdx.x) % shares;
    const int tile = unit / R, rank = unit % R;
    const int etid = threadIdx.x, warp = etid >> 5, lane = etid & 31, quad = warp & 3, chalf = warp >> 2;
    int tm, tn;
    tile_coords(tile, tiles_m, tiles_n, tm, tn, group_m);
    const int64_t row = static_cast<int64_t>(tm) * (R * kBM) + rank * kBM + quad * 32 + lane;
    const int col0 = tn * BN + chalf * CPW;
    const float4 *src = reinterpret_cast<const float4 *>(part + static_cast<size_t>(unit) * n_seg * (kBM * BN));
    const size_t seg_stride = static_cast<size_t>(kBM) * BN / 4;               // float4 per partial
    const int c_lo = share * NC / shares, c_hi = (share + 1) * NC / shares;
    for (int c4 = c_lo; c4 < c_hi; ++c4) {
        float4 acc;
        asm volatile("ld.global.cg.v4.f32 {%0, %1, %2, %3}, [%4];"
                     : "=f"(acc.x), "=f"(acc.y), "=f"(acc.z), "=f"(acc.w) : "l"(src + c4 * 256 + etid) : "memory");
        // (non-volatile loads, eight segments per batch: the loads of a batch are all in flight before the first add)
#pragma unroll 1
        for (int s0 = 1; s0 < n_seg; s0 += 8) {
            float4 v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u)
                if (s0 + u < n_seg)
                    asm("ld.global.cg.v4.f32 {%0, %1, %2, %3}, [%4];"
                        : "=f"(v[u].x), "=f"(v[u].y), "=f"(v[u].z), "=f"(v[u].w) : "l"(src + (s0 + u) * seg_stride + c4 * 256 + etid));
#pragma unroll
            for (int u = 0; u < 8; ++u)
                if (s0 + u < n_seg) {
                    acc.x = __fadd_rn(acc.x, v[u].x); acc.y = __fadd_rn(acc.y, v[u].y);
                    acc.z = __fadd_rn(acc.z, v[u].z); acc.w = __fadd_rn(acc.w, v[u].w);
                }
        }
        if (row < M) {
            emit_dispatch(out, [&](const OutArgs &po, auto fast) {
                emit4<decltype(fast)::value>(po, row, col0 + c4 * 4, acc, N);
            });
        }
    }
}

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
    const int k_tiles = (args.K + kBK - 1) / kBK;
    const int n_seg = (k_tiles + kTilesPerSeg - 1) / kTilesPerSeg;
    TileSched sched;
    sched.init(args.tiles_m * args.tiles_n, args.balance, args.dp_tiles, n_seg, static_cast<int>(blockIdx.x), static_cast<int>(gridDim.x));

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
    pdl_wait();
    pdl_launch_dependents();

    if (warp == 0) {
        // ================================ TMA producer ================================
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int ci = 0; ci < sched.n_chunks; ++ci) {
                int tile, sb_seg, se_seg;
                sched.get(ci, tile, sb_seg, se_seg);
                int tm, tn;
                tile_coords(tile, args.tiles_m, args.tiles_n, tm, tn, args.group_m);
                const int m0 = tm * kBM;
                const int n0 = tn * BN;
                const int kt_hi = min(k_tiles, se_seg * kTilesPerSeg);
                const int n_steps = Cfg::SCALED ? 2 * (kt_hi - sb_seg * kTilesPerSeg) : kt_hi - sb_seg * kTilesPerSeg;
                for (int step = 0; step < n_steps; ++step) {
                    int kt = sb_seg * kTilesPerSeg + step;
                    bool lo_pass = false;
                    if (Cfg::SCALED) {                       // segment by segment: the residual pass, then the hi pass
                        const int seg = sb_seg + step / (2 * kTilesPerSeg), r = step % (2 * kTilesPerSeg);
                        const int len = min(k_tiles, (seg + 1) * kTilesPerSeg) - seg * kTilesPerSeg;
                        lo_pass = r < len;
                        kt = seg * kTilesPerSeg + (lo_pass ? r : r - len);
                    }
                    mbar_wait_ool(empty_bar(stage), phase ^ 1u, args.diag, 100 + stage);
                    const uint32_t sb = smem_base + stage * Cfg::STAGE_BYTES;
                    const uint32_t fb = full_bar(stage);
                    mbar_arrive_expect_tx(fb, Cfg::STAGE_BYTES);
                    const int k0 = kt * kBK;
                    if (Cfg::SCALED) {
                        tma_load_2d(sb, lo_pass ? &tm_a_lo : &tm_a_hi, fb, k0, m0);
                    } else {
                        tma_load_2d(sb, &tm_a_hi, fb, k0, m0);
                        if (Cfg::A_PLANES == 2) tma_load_2d(sb + Cfg::A_TILE, &tm_a_lo, fb, k0, m0);
                    }
                    const uint32_t sbB = sb + Cfg::A_SLOTS * Cfg::A_TILE;
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
            for (int ci = 0; ci < sched.n_chunks; ++ci) {
                int tile, sb_seg, se_seg;
                sched.get(ci, tile, sb_seg, se_seg);
                for (int seg = sb_seg; seg < se_seg; ++seg) {
                    mbar_wait_ool(tempty_bar(buf), ((tphase >> buf) & 1u) ^ 1u, args.diag, 300 + buf);
                    tc_fence_after();
                    const uint32_t d_tmem = tmem_base + static_cast<uint32_t>(buf * BN);
                    const int kt_end = min(k_tiles, (seg + 1) * kTilesPerSeg);
                    uint32_t accumulate = 0;
                    if constexpr (Cfg::SCALED) {
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
                                        umma_f16_scale_d<kLoShift>(d_tmem, a_d + ao, b_d + bo, idesc);
                                    else
                                        umma_f16(d_tmem, a_d + ao, b_d + bo, idesc, accumulate);
                                    accumulate = 1;
                                }
                                umma_commit(empty_bar(stage));
                                if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                            }
                    } else
                    for (int kt = seg * kTilesPerSeg; kt < kt_end; ++kt) {
                        mbar_wait_ool(full_bar(stage), phase, args.diag, 200 + stage);
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
        const int etid = threadIdx.x - 128;                      // 0..255 among the epilogue threads
        for (int ci = 0; ci < sched.n_chunks; ++ci) {
            int tile, sb_seg, se_seg;
            sched.get(ci, tile, sb_seg, se_seg);
            int tm, tn;
            tile_coords(tile, args.tiles_m, args.tiles_n, tm, tn, args.group_m);
            const int m0 = tm * kBM;
            const int n0 = tn * BN;
            if constexpr (Cfg::FULL) {
                if (args.sk) {
                    // ordered split-K: park every segment partial in global memory; heal_splitk_reduce_kernel forms the sums
                    for (int seg = sb_seg; seg < se_seg; ++seg) {
                        mbar_wait_ool(tfull_bar(buf), (tphase >> buf) & 1u, args.diag, 400 + buf);
                        tc_fence_after();
                        const uint32_t taddr = tmem_base + (static_cast<uint32_t>(quad * 32) << 16) +
                                               static_cast<uint32_t>(buf * BN + chalf * CPW);
                        sk_store_partial<CPW>(args.part + (static_cast<size_t>(tile) * n_seg + seg) * (kBM * BN), taddr, etid);
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive(tempty_bar(buf));
                        tphase ^= 1u << buf;
                        buf ^= 1;
                    }
                    continue;
                }
            }
            if (sb_seg > 0)        // tail of a shared tile: start from the neighbour's running sum (segments 0..sb_seg-1)
                epi_take_prefix<CPW>(args.xfer + static_cast<size_t>(blockIdx.x - 1) * (kBM * BN), args.flags + (blockIdx.x - 1), run, etid, args.diag);
            for (int seg = sb_seg; seg < se_seg; ++seg) {
                mbar_wait_ool(tfull_bar(buf), (tphase >> buf) & 1u, args.diag, 400 + buf);
                tc_fence_after();
                const uint32_t taddr = tmem_base + (static_cast<uint32_t>(quad * 32) << 16) +
                                       static_cast<uint32_t>(buf * BN + chalf * CPW);
                epi_add_segment<CPW>(taddr, run, seg == 0);
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(tempty_bar(buf));
                tphase ^= 1u << buf;
                buf ^= 1;
            }
            if (se_seg < n_seg) {  // head of a shared tile: hand the running sum to the next CTA
                epi_hand_on<CPW>(args.xfer + static_cast<size_t>(blockIdx.x) * (kBM * BN), args.flags + blockIdx.x, run, etid);
                continue;
            }
            // ---- store: thread owns row m0 + quad*32 + lane, CPW consecutive columns
            epi_store<CPW, Cfg::FULL>(args.out, m0 + quad * 32 + lane, n0 + chalf * CPW, run, args.M, args.N);
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
