// heal_api.cu -- the C ABI of libheal.so (include/heal.h): argument validation, workspace,
// TMA tensor-map encoding, kernel dispatch.  Every step of the path runs in the kernels of
// heal_split.cuh / heal_gemm_umma.cuh; there is no CPU or library fallback.
#include "../../include/heal.h"

#include <cuda.h>
#include <cudaTypedefs.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <atomic>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <deque>
#include <mutex>
#include <string>
#include <vector>

#include "heal_gemm_smallm.cuh"
#include "heal_gemm_umma.cuh"
#include "heal_gemm_umma2.cuh"
#include "heal_gemm_umma2f.cuh"
#include "heal_split.cuh"

namespace {

using namespace heal;

thread_local const char *t_last_kernel = "none";      // heal_last_kernel(): the GEMM kernel of this thread's latest call
std::string kernel_name(const char *family, int a, int nprod, bool b_mn, const char *extra)
{
    return std::string(family) + "<" + std::to_string(a) + "," + std::to_string(nprod) + "P," + (b_mn ? "KxN" : "NxK") + extra + ">";
}
std::atomic<int> g_last_cuda_error{0};
std::atomic<uint64_t> g_launches{0};
std::mutex g_mu;
std::mutex g_xf_mu;
std::mutex g_host_mu;

struct State {
    bool init = false;
    int init_status = HEAL_OK;
    int device = -1;
    int num_sms = 0;
    int *diag = nullptr;
    // Per-stream resources: hand-off buffers of the balanced schedule, hi/lo plane workspace, split-K partial area (concurrent
    // streams must not share them).  A slot that was ever used while its stream was being captured is PINNED: its buffers may
    // be baked into a CUDA graph, so they are never freed, shrunk, moved or handed to another stream (see acquire_slot).
    struct Xfer {
        cudaStream_t stream = nullptr;
        bool used = false;
        bool pinned = false;       // used during stream capture at least once
        float *xfer = nullptr;     // per-CTA running-sum slots (128 x 256 floats each)
        uint32_t *flags = nullptr; // per-CTA flag: 1 = slot written, reset by the consumer
        uint64_t last_use = 0;     // for recycling the least recently used un-pinned slot
        void *ws = nullptr;        // library-owned hi/lo plane workspace of this stream, grown on demand
        size_t ws_bytes = 0;
        float *part = nullptr;     // ordered split-K: segment partials, grown on demand (never while capturing)
        size_t part_bytes = 0;
    };
    std::deque<Xfer> xf;           // grows when every slot is pinned or busy; addresses of elements stay valid
    std::vector<void *> retired;   // buffers replaced while their slot was pinned: kept alive for the graphs that hold them
    // workspace
    void *user_ws = nullptr;
    size_t user_ws_bytes = 0;
    // host-variant staging
    void *stage = nullptr;
    size_t stage_bytes = 0;
    cudaStream_t copy_in = nullptr, copy_out = nullptr;      // host variant: one stream per PCIe direction
    cudaEvent_t ev_in[8] = {}, ev_done[8] = {}, ev_start = nullptr;
    PFN_cuTensorMapEncodeTiled_v12000 encode = nullptr;
};
State g;

inline int cuda_fail(cudaError_t e)
{
    g_last_cuda_error.store(static_cast<int>(e));
    return HEAL_ERR_CUDA;
}
#define HEAL_CUDA(expr)                                  \
    do {                                                 \
        cudaError_t e__ = (expr);                        \
        if (e__ != cudaSuccess) return cuda_fail(e__);   \
    } while (0)

int ensure_init()
{
    std::lock_guard<std::mutex> lk(g_mu);
    if (g.init) {
        // one device per process (the launch pattern of bench.py / torchrun): buffers, SM count and tensor-map entry
        // point belong to the device of the first call
        int cur = -1;
        if (g.init_status == HEAL_OK && (cudaGetDevice(&cur) != cudaSuccess || cur != g.device)) return HEAL_ERR_UNSUPPORTED_DEVICE;
        return g.init_status;
    }
    g.init = true;
    auto fail = [&](int st) { g.init_status = st; return st; };
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(cuda_fail(e));
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) return fail(cuda_fail(e));
    if (prop.major != 10) return fail(HEAL_ERR_UNSUPPORTED_DEVICE);
    g.device = dev;
    g.num_sms = prop.multiProcessorCount;
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    e = cudaGetDriverEntryPointByVersion("cuTensorMapEncodeTiled", &fn, 12000, cudaEnableDefault, &qres);
    if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn)
        return fail(cuda_fail(e != cudaSuccess ? e : cudaErrorUnknown));
    g.encode = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(fn);
    e = cudaMalloc(&g.diag, 64);
    if (e != cudaSuccess) return fail(cuda_fail(e));
    e = cudaMemset(g.diag, 0, 64);
    if (e != cudaSuccess) return fail(cuda_fail(e));
    return HEAL_OK;
}

inline bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }

// 2-D FP16 tensor map, 128-byte swizzle, out-of-bounds elements read as zero (K/M/N tails).
//   inner/outer: extents in elements; ld: row pitch in elements; box: {inner, outer} elements.
// Encoded maps are cached (direct-mapped, keyed on everything that enters the encoding): an inference loop calls with
// the same few (pointer, shape) combinations over and over, and four driver encodes per launch are a measurable part
// of the host-side cost of a 9 us decode GEMM.  A map holds only the address and geometry, never data, so a stale
// entry for a freed-and-reused pointer is still a correct encoding of the same arguments.
struct MapKey {
    const void *base;
    int64_t inner, outer, ld;
    uint32_t box_inner, box_outer, kind;
    bool operator==(const MapKey &o) const
    {
        return base == o.base && inner == o.inner && outer == o.outer && ld == o.ld && box_inner == o.box_inner &&
               box_outer == o.box_outer && kind == o.kind;
    }
};
struct MapEntry {
    MapKey key;
    bool valid = false;
    CUtensorMap map;
};
constexpr int kMapCache = 256;
MapEntry g_maps[kMapCache];
std::mutex g_map_mu;

// kind 0: FP16, 128-byte swizzle (MMA operand tiles); kind 1: FP32, no swizzle (activation tiles the kernel converts itself)
int encode_2d(CUtensorMap *tm, const void *base, int64_t inner, int64_t outer, int64_t ld, uint32_t box_inner,
              uint32_t box_outer, uint32_t kind)
{
    const MapKey key{base, inner, outer, ld, box_inner, box_outer, kind};
    uint64_t h = reinterpret_cast<uintptr_t>(base) >> 4;
    h = (h ^ static_cast<uint64_t>(inner) * 0x9E3779B97F4A7C15ull) + static_cast<uint64_t>(outer) * 0xC2B2AE3D27D4EB4Full;
    h ^= static_cast<uint64_t>(ld) * 0x165667B19E3779F9ull + box_inner * 131u + box_outer * 31u + kind;
    h ^= h >> 29;
    MapEntry &e = g_maps[h % kMapCache];
    {
        std::lock_guard<std::mutex> lk(g_map_mu);
        if (e.valid && e.key == key) {
            *tm = e.map;
            return HEAL_OK;
        }
    }
    const size_t es = kind == 1 ? 4 : 2;
    cuuint64_t dims[2] = {static_cast<cuuint64_t>(inner), static_cast<cuuint64_t>(outer)};
    cuuint64_t strides[1] = {static_cast<cuuint64_t>(ld) * es};
    cuuint32_t box[2] = {box_inner, box_outer};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = g.encode(tm, kind == 1 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2,
                          const_cast<void *>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                          kind == 1 ? CU_TENSOR_MAP_SWIZZLE_NONE : CU_TENSOR_MAP_SWIZZLE_128B,
                          CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        g_last_cuda_error.store(static_cast<int>(cudaErrorInvalidValue));
        return HEAL_ERR_CUDA;
    }
    std::lock_guard<std::mutex> lk(g_map_mu);
    e.key = key;
    e.map = *tm;
    e.valid = true;
    return HEAL_OK;
}
inline int encode_f16_2d(CUtensorMap *tm, const void *base, int64_t inner, int64_t outer, int64_t ld, uint32_t box_inner,
                         uint32_t box_outer)
{
    return encode_2d(tm, base, inner, outer, ld, box_inner, box_outer, 0);
}

}  // namespace

namespace {

// Launch attributes: optional cluster dimension + programmatic stream serialization (PDL), which lets the
// kernel's prologue (barrier init, TMEM allocation, descriptor prefetch) overlap the previous kernel's tail;
// every kernel calls griddepcontrol.wait before its first global-memory access.
int fill_attrs(cudaLaunchAttribute *attr, unsigned cluster_x, int cooperative = 0)
{
    static const bool no_pdl = std::getenv("HEAL_NO_PDL") != nullptr;          // debug only
    int n = 0;
    if (cluster_x > 1) {
        attr[n].id = cudaLaunchAttributeClusterDimension;
        attr[n].val.clusterDim.x = cluster_x;
        attr[n].val.clusterDim.y = 1;
        attr[n].val.clusterDim.z = 1;
        ++n;
    }
    if (cooperative) {                   // all CTAs co-resident or the launch waits: see epi_take_prefix
        attr[n].id = cudaLaunchAttributeCooperative;
        attr[n].val.cooperative = 1;
        ++n;
    }
    if (!no_pdl && cooperative != 1) {
        attr[n].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[n].val.programmaticStreamSerializationAllowed = 1;
        ++n;
    }
    return n;
}

// ---- step S launch --------------------------------------------------------------------------
int launch_split(int64_t rows, int64_t cols, const float *X, int64_t ldx, __half *hi, __half *lo, int64_t ld,
                 cudaStream_t stream, int lo_shift = 0)
{
    if (rows == 0 || cols == 0) return HEAL_OK;
    const int64_t vecs = rows * ((cols + 7) / 8);
    int64_t blocks = (vecs + 255) / 256;
    const int64_t cap = static_cast<int64_t>(g.num_sms) * 16;      // grid-stride beyond 16 CTAs per SM
    if (blocks > cap) blocks = cap;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(blocks));
    cfg.blockDim = dim3(256);
    cfg.stream = stream;
    cudaLaunchAttribute attr[3];
    cfg.numAttrs = fill_attrs(attr, 1);
    cfg.attrs = attr;
    const float lo_scale = static_cast<float>(1u << lo_shift);                   // 2^s, s in [0, 16]
    HEAL_CUDA(cudaLaunchKernelEx(&cfg, heal_split_kernel, X, ldx, rows, cols, hi, lo, ld, lo_scale));
    g_launches.fetch_add(1);
    return HEAL_OK;
}

// Per-stream resources (hi/lo plane workspace, balanced-schedule hand-off buffers, split-K partial area): one slot per
// stream that has called into the library, so calls on different streams never share scratch memory.  Up to 8 slots are
// kept for streams that were never captured: when a ninth such stream shows up the least recently used un-pinned slot is
// recycled (after a device synchronise; it keeps its buffers).  Pinned slots (used under stream capture: their buffers
// may live on in graphs) are never recycled; the deque simply grows.  During stream capture nothing is allocated: what a
// captured call needs must exist from an earlier eager call on the same stream (else: unbalanced schedule for the GEMM,
// HEAL_ERR_WORKSPACE for the planes).  Call with g_xf_mu held.
State::Xfer *acquire_slot(cudaStream_t stream, bool capturing)
{
    static uint64_t tick = 0;
    State::Xfer *slot = nullptr;
    for (auto &x : g.xf)
        if (x.used && x.stream == stream) { slot = &x; break; }
    if (!slot && !capturing) {
        for (auto &x : g.xf)
            if (!x.used) { slot = &x; break; }
        if (!slot) {
            int unpinned = 0;
            for (auto &x : g.xf) unpinned += x.pinned ? 0 : 1;
            if (unpinned >= 8 && cudaDeviceSynchronize() == cudaSuccess) {
                for (auto &x : g.xf)
                    if (!x.pinned && (!slot || x.last_use < slot->last_use)) slot = &x;
            }
            if (!slot) {
                g.xf.emplace_back();
                slot = &g.xf.back();
            }
        }
        slot->stream = stream;
        slot->used = true;
    }
    if (slot) {
        slot->last_use = ++tick;
        if (capturing) slot->pinned = true;
    }
    return slot;
}

// Replace a slot buffer by a larger one.  An un-pinned slot: wait for the stream (earlier calls may still use the old
// buffer) and free it.  A pinned slot: a captured graph may replay the old address at any time, so it stays allocated for
// the life of the process (g.retired) and only new calls use the new one.
int grow_buffer(State::Xfer *slot, cudaStream_t stream, void **buf, size_t *have, size_t want)
{
    if (*buf) {
        if (slot->pinned) {
            g.retired.push_back(*buf);
        } else {
            HEAL_CUDA(cudaStreamSynchronize(stream));
            HEAL_CUDA(cudaFree(*buf));
        }
    }
    *buf = nullptr;
    *have = 0;
    HEAL_CUDA(cudaMalloc(buf, want));
    *have = want;
    return HEAL_OK;
}

bool stream_capturing(cudaStream_t stream)
{
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    return cudaStreamIsCapturing(stream, &cap) != cudaSuccess || cap != cudaStreamCaptureStatusNone;
}

bool bind_xfer(GemmArgs &args, cudaStream_t stream, size_t part_bytes = 0)
{
    std::lock_guard<std::mutex> lk(g_xf_mu);
    const bool capturing = stream_capturing(stream);
    State::Xfer *slot = acquire_slot(stream, capturing);
    if (!slot) return false;
    if (!slot->xfer) {                                   // 19 MB of hand-off slots + flags, first use only
        if (capturing) return false;
        float *xf = nullptr;
        uint32_t *fl = nullptr;
        if (cudaMalloc(&xf, static_cast<size_t>(g.num_sms) * kBM * 256 * sizeof(float)) != cudaSuccess) return false;
        if (cudaMalloc(&fl, static_cast<size_t>(g.num_sms) * sizeof(uint32_t)) != cudaSuccess ||
            cudaMemset(fl, 0, static_cast<size_t>(g.num_sms) * sizeof(uint32_t)) != cudaSuccess) {
            cudaFree(xf);
            if (fl) cudaFree(fl);
            return false;
        }
        slot->xfer = xf;
        slot->flags = fl;
    }
    if (part_bytes > slot->part_bytes) {
        if (capturing) return false;
        void *p = slot->part;
        const int st = grow_buffer(slot, stream, &p, &slot->part_bytes, part_bytes);
        slot->part = static_cast<float *>(p);
        if (st) return false;
    }
    args.xfer = slot->xfer;
    args.flags = slot->flags;
    args.part = slot->part;
    return true;
}

// Balanced schedule when whole tiles do not divide evenly over the G_max CTAs (or CTA pairs); numerically
// invisible.  Returns the number of CTAs (pairs) to launch.
//  * tiles >= G_max: full waves stay tile-granular; the ragged remainder (plus one full wave when the remainder
//    alone would leave less than half a tile per CTA) is cut at K-segment granularity.
//  * tiles < G_max (mid-size M, small N): ordered split-K, see below.
// the ordered split-K rule of set_balance(), without side effects: decides which kernel instantiation to launch
// Ordered split-K pays while a CTA gets few units: a parked unit costs about `a/b` plain segments more than a unit of a
// whole tile (its partial travels to L2 and back through the reduce kernel), whole tiles cost n_seg segments per CTA.
// HEAL_SK_RULE="a,b" overrides the measured default (debug / tuning).
bool sk_rule(int64_t units_per_cta, int64_t n_seg, int64_t tiles, int64_t G_max)
{
    static int a = 12, b = 5;
    static const bool init = [] {
        if (const char *e = std::getenv("HEAL_SK_RULE")) {
            int x = 0, y = 0;
            if (std::sscanf(e, "%d,%d", &x, &y) == 2 && x > 0 && y > 0) { a = x; b = y; }
        }
        return true;
    }();
    (void)init;
    // two segments only (K <= 1024): worth it when the tiles fill at most a quarter of the machine (measured: 1024^3 three
    // products 22.9 -> 18.8 us; with more tiles the parked partials cost more than the idle SMs)
    if (n_seg == 2) return units_per_cta == 1 && 4 * tiles <= G_max;
    return a * units_per_cta < b * n_seg;
}

bool wants_split_k(int64_t tiles, int64_t n_seg, int64_t G_max, int ctas_per_tile, int bn)
{
    if (tiles >= G_max || n_seg <= 1 || std::getenv("HEAL_NO_BALANCE")) return false;
    const int64_t units = tiles * n_seg;
    const int64_t G = units < G_max ? units : G_max;
    const size_t part_bytes = static_cast<size_t>(units) * ctas_per_tile * kBM * bn * sizeof(float);
    return G > tiles && sk_rule((units + G - 1) / G, n_seg, tiles, G_max) && part_bytes <= (static_cast<size_t>(128) << 20);
}

int64_t set_balance(GemmArgs &args, int64_t tiles, int64_t n_seg, int64_t G_max, int ctas_per_tile, int bn, bool full_kernel,
                    cudaStream_t stream)
{
    static const int group_m = std::getenv("HEAL_GROUP_M") ? std::atoi(std::getenv("HEAL_GROUP_M")) : kGroupM;      // tuning
    args.group_m = group_m > 0 ? group_m : kGroupM;
    args.xfer = nullptr;
    args.flags = nullptr;
    args.part = nullptr;
    args.sk = 0;
    static const bool no_balance = std::getenv("HEAL_NO_BALANCE") != nullptr;      // debug only
    args.balance = 0;
    args.dp_tiles = static_cast<int>(tiles);
    if (tiles < G_max) {
        // Ordered split-K: (tile, segment) units are dealt contiguously to up to tiles * n_seg CTAs; every
        // segment partial is parked in global memory and the CTAs of a tile each finish a share of its columns.
        const int64_t units = tiles * n_seg;
        const int64_t G = units < G_max ? units : G_max;
        const size_t part_bytes = static_cast<size_t>(units) * ctas_per_tile * kBM * bn * sizeof(float);
        // Worth it only while a CTA gets few units: parking and re-reading a partial costs about 1.4 segments of
        // L2 traffic (measured: a parked unit takes 2.4x a plain segment), whole tiles cost n_seg segments.
        const int64_t units_per_cta = (units + G - 1) / G;
        if (full_kernel && !no_balance && n_seg > 1 && G > tiles && sk_rule(units_per_cta, n_seg, tiles, G_max) &&
            part_bytes <= (static_cast<size_t>(128) << 20) && bind_xfer(args, stream, part_bytes)) {
            args.balance = 1;
            args.sk = 1;
            args.dp_tiles = 0;
            return G;
        }
        return tiles;
    }
    if (!no_balance && tiles % G_max != 0) {
        const int64_t waves = tiles / G_max, rem = tiles % G_max;
        int64_t sk = rem;
        if (rem * 2 < G_max && waves >= 1) sk += G_max;
        if (bind_xfer(args, stream)) {
            args.balance = 1;
            args.dp_tiles = static_cast<int>(tiles - sk);
        }
    }
    return G_max;
}

// Balanced-schedule launches spin on a flag written by a lower-indexed CTA (epi_take_prefix).  0 = plain launch (relies on
// in-order block dispatch), 1 = cooperative launch instead of PDL, 2 = cooperative + PDL (the default: measured at no cost on
// the headline GEMM).  HEAL_COOP overrides (debug).
int coop_mode()
{
    static const int mode = [] {
        const char *e = std::getenv("HEAL_COOP");
        return e ? std::atoi(e) : 0;
    }();
    return mode;
}

// second half of the ordered split-K schedule: ascending-segment FP32 RN sums of the parked partials + step E
template <int BN>
int launch_sk_reduce(const GemmArgs &args, int ctas_per_tile, int64_t tiles, cudaStream_t stream)
{
    const int n_seg = (args.K + kKSeg - 1) / kKSeg;
    const int64_t units = tiles * ctas_per_tile;
    constexpr int NC = BN / 8;                                    // float4 chunks per thread
    int64_t shares = (2 * static_cast<int64_t>(g.num_sms) + units - 1) / units;     // about two waves of 256-thread CTAs
    if (shares > NC) shares = NC;
    if (shares < 1) shares = 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(units * shares));
    cfg.blockDim = dim3(256);
    cfg.stream = stream;
    cudaLaunchAttribute attr[3];
    cfg.numAttrs = fill_attrs(attr, 1);
    cfg.attrs = attr;
    HEAL_CUDA(cudaLaunchKernelEx(&cfg, heal_splitk_reduce_kernel<BN>, static_cast<const float *>(args.part), n_seg, ctas_per_tile,
                                 args.tiles_m, args.tiles_n, args.group_m, static_cast<int>(shares), args.out, args.M, args.N));
    g_launches.fetch_add(1);
    return HEAL_OK;
}

// ---- steps G + E launch -----------------------------------------------------------------------
template <class Cfg>
int launch_gemm_cfg(int64_t M, int64_t N, int64_t K, const void *A_hi, const void *A_lo, int64_t lda, const void *B_hi,
                    const void *B_lo, int64_t ldb, const OutArgs &out, cudaStream_t stream)
{
    static std::atomic<bool> attr_set{false};          // setting the attribute twice from two threads is harmless
    auto kern = heal_gemm_umma_kernel<Cfg>;
    if (!attr_set.load(std::memory_order_acquire)) {
        HEAL_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES));
        attr_set.store(true, std::memory_order_release);
    }
    CUtensorMap ta_hi, ta_lo, tb_hi, tb_lo;
    int st = encode_f16_2d(&ta_hi, A_hi, K, M, lda, kBK, kBM);
    if (st) return st;
    if (Cfg::A_PLANES == 2) {
        st = encode_f16_2d(&ta_lo, A_lo, K, M, lda, kBK, kBM);
        if (st) return st;
    } else {
        ta_lo = ta_hi;
    }
    if (Cfg::B_MN) st = encode_f16_2d(&tb_hi, B_hi, N, K, ldb, 64, kBK);
    else           st = encode_f16_2d(&tb_hi, B_hi, K, N, ldb, kBK, Cfg::BN);
    if (st) return st;
    if (Cfg::B_PLANES == 2) {
        if (Cfg::B_MN) st = encode_f16_2d(&tb_lo, B_lo, N, K, ldb, 64, kBK);
        else           st = encode_f16_2d(&tb_lo, B_lo, K, N, ldb, kBK, Cfg::BN);
        if (st) return st;
    } else {
        tb_lo = tb_hi;
    }
    GemmArgs args;
    args.out = out;
    args.M = static_cast<int>(M);
    args.N = static_cast<int>(N);
    args.K = static_cast<int>(K);
    args.tiles_m = static_cast<int>((M + kBM - 1) / kBM);
    args.tiles_n = static_cast<int>((N + Cfg::BN - 1) / Cfg::BN);
    args.diag = g.diag;
    const int64_t tiles = static_cast<int64_t>(args.tiles_m) * args.tiles_n;
    const unsigned grid = static_cast<unsigned>(set_balance(args, tiles, (K + kKSeg - 1) / kKSeg, g.num_sms, 1, Cfg::BN, Cfg::FULL, stream));
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(kGemmThreads);
    cfg.dynamicSmemBytes = Cfg::SMEM_BYTES;
    cfg.stream = stream;
    cudaLaunchAttribute attr[3];
    cfg.numAttrs = fill_attrs(attr, 1, (args.balance && !args.sk) ? coop_mode() : 0);
    cfg.attrs = attr;
    HEAL_CUDA(cudaLaunchKernelEx(&cfg, kern, ta_hi, ta_lo, tb_hi, tb_lo, args));
    g_launches.fetch_add(1);
    static const std::string name = kernel_name("heal_gemm_umma_kernel", Cfg::BN, Cfg::NPROD, Cfg::B_MN, Cfg::FULL ? ",full" : "");
    t_last_kernel = name.c_str();
    if (args.sk) return launch_sk_reduce<Cfg::BN>(args, 1, tiles, stream);
    return HEAL_OK;
}

// CTA-pair (cta_group::2) variant: 256 x BN tiles, cluster of 2
template <class Cfg>
int launch_gemm2_cfg(int64_t M, int64_t N, int64_t K, const void *A_hi, const void *A_lo, int64_t lda, const void *B_hi,
                     const void *B_lo, int64_t ldb, const OutArgs &out, cudaStream_t stream)
{
    static std::atomic<bool> attr_set{false};
    auto kern = heal_gemm_umma2_kernel<Cfg>;
    if (!attr_set.load(std::memory_order_acquire)) {
        HEAL_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES));
        attr_set.store(true, std::memory_order_release);
    }
    CUtensorMap ta_hi, ta_lo, tb_hi, tb_lo;
    int st = encode_f16_2d(&ta_hi, A_hi, K, M, lda, kBK, kBM);
    if (st) return st;
    if (Cfg::A_PLANES == 2) {
        st = encode_f16_2d(&ta_lo, A_lo, K, M, lda, kBK, kBM);
        if (st) return st;
    } else {
        ta_lo = ta_hi;
    }
    if (Cfg::B_MN) st = encode_f16_2d(&tb_hi, B_hi, N, K, ldb, 64, kBK);
    else           st = encode_f16_2d(&tb_hi, B_hi, K, N, ldb, kBK, Cfg::BH);
    if (st) return st;
    if (Cfg::B_PLANES == 2) {
        if (Cfg::B_MN) st = encode_f16_2d(&tb_lo, B_lo, N, K, ldb, 64, kBK);
        else           st = encode_f16_2d(&tb_lo, B_lo, K, N, ldb, kBK, Cfg::BH);
        if (st) return st;
    } else {
        tb_lo = tb_hi;
    }
    GemmArgs args;
    args.out = out;
    args.M = static_cast<int>(M);
    args.N = static_cast<int>(N);
    args.K = static_cast<int>(K);
    args.tiles_m = static_cast<int>((M + 2 * kBM - 1) / (2 * kBM));
    args.tiles_n = static_cast<int>((N + Cfg::BN - 1) / Cfg::BN);
    args.diag = g.diag;
    const int64_t tiles = static_cast<int64_t>(args.tiles_m) * args.tiles_n;
    const int64_t G = set_balance(args, tiles, (K + kKSeg - 1) / kKSeg, g.num_sms / 2, 2, Cfg::BN, Cfg::FULL, stream);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(2 * G));
    cfg.blockDim = dim3(kGemmThreads);
    cfg.dynamicSmemBytes = Cfg::SMEM_BYTES;
    cfg.stream = stream;
    cudaLaunchAttribute attr[3];
    cfg.numAttrs = fill_attrs(attr, 2, (args.balance && !args.sk) ? coop_mode() : 0);
    cfg.attrs = attr;
    HEAL_CUDA(cudaLaunchKernelEx(&cfg, kern, ta_hi, ta_lo, tb_hi, tb_lo, args));
    g_launches.fetch_add(1);
    static const std::string name = kernel_name("heal_gemm_umma2_kernel", Cfg::BN, Cfg::NPROD, Cfg::B_MN, Cfg::FULL ? ",full,cta_group::2" : ",cta_group::2");
    t_last_kernel = name.c_str();
    if (args.sk) return launch_sk_reduce<Cfg::BN>(args, 2, tiles, stream);
    return HEAL_OK;
}

// CTA-pair kernel with the activation split fused in (heal_gemm_umma2f.cuh): A is the FP32 matrix itself
template <class Cfg>
int launch_gemm2f_cfg(int64_t M, int64_t N, int64_t K, const float *A, int64_t lda, const void *B_hi, const void *B_lo,
                      int64_t ldb, const OutArgs &out, cudaStream_t stream)
{
    static std::atomic<bool> attr_set{false};
    auto kern = heal_gemm_umma2f_kernel<Cfg>;
    if (!attr_set.load(std::memory_order_acquire)) {
        HEAL_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES));
        attr_set.store(true, std::memory_order_release);
    }
    CUtensorMap ta, tb_hi, tb_lo;
    int st = encode_2d(&ta, A, K, M, lda, 32, kBM, 1);          // FP32, two boxes of 32 k per k-tile
    if (st) return st;
    if (Cfg::B_MN) st = encode_f16_2d(&tb_hi, B_hi, N, K, ldb, 64, kBK);
    else           st = encode_f16_2d(&tb_hi, B_hi, K, N, ldb, kBK, Cfg::BH);
    if (st) return st;
    if (Cfg::B_PLANES == 2) {
        if (Cfg::B_MN) st = encode_f16_2d(&tb_lo, B_lo, N, K, ldb, 64, kBK);
        else           st = encode_f16_2d(&tb_lo, B_lo, K, N, ldb, kBK, Cfg::BH);
        if (st) return st;
    } else {
        tb_lo = tb_hi;
    }
    GemmArgs args;
    args.out = out;
    args.M = static_cast<int>(M);
    args.N = static_cast<int>(N);
    args.K = static_cast<int>(K);
    args.tiles_m = static_cast<int>((M + 2 * kBM - 1) / (2 * kBM));
    args.tiles_n = static_cast<int>((N + Cfg::BN - 1) / Cfg::BN);
    args.diag = g.diag;
    const int64_t tiles = static_cast<int64_t>(args.tiles_m) * args.tiles_n;
    const int64_t G = set_balance(args, tiles, (K + kKSeg - 1) / kKSeg, g.num_sms / 2, 2, Cfg::BN, Cfg::FULL, stream);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(2 * G));
    cfg.blockDim = dim3(kFusedThreads);
    cfg.dynamicSmemBytes = Cfg::SMEM_BYTES;
    cfg.stream = stream;
    cudaLaunchAttribute attr[3];
    cfg.numAttrs = fill_attrs(attr, 2, (args.balance && !args.sk) ? coop_mode() : 0);
    cfg.attrs = attr;
    HEAL_CUDA(cudaLaunchKernelEx(&cfg, kern, ta, tb_hi, tb_lo, args));
    g_launches.fetch_add(1);
    static const std::string name = kernel_name("heal_gemm_umma2f_kernel", Cfg::BN, Cfg::NPROD, Cfg::B_MN, Cfg::FULL ? ",full,cta_group::2,fused split" : ",cta_group::2,fused split");
    t_last_kernel = name.c_str();
    if (args.sk) return launch_sk_reduce<Cfg::BN>(args, 2, tiles, stream);
    return HEAL_OK;
}

inline bool needs_ext(const OutArgs &out) { return out.hi != nullptr || out.accumulate != 0 || out.silu != 0 || out.scale != 1.0f || out.C == nullptr; }

template <bool B_MN>
int launch_gemm2_np(int nprod, int64_t M, int64_t N, int64_t K, const void *A_hi, const void *A_lo, int64_t lda,
                    const void *B_hi, const void *B_lo, int64_t ldb, const OutArgs &out, cudaStream_t s)
{
    const int64_t tiles = ((M + 2 * kBM - 1) / (2 * kBM)) * ((N + 255) / 256);
    if (nprod == kScaledLo || needs_ext(out) || wants_split_k(tiles, (K + kKSeg - 1) / kKSeg, g.num_sms / 2, 2, 256)) {
        switch (nprod) {
        case 1: return launch_gemm2_cfg<Gemm2Cfg<256, 1, B_MN, true>>(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
        case 2: return launch_gemm2_cfg<Gemm2Cfg<256, 2, B_MN, true>>(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
        case 3: return launch_gemm2_cfg<Gemm2Cfg<256, 3, B_MN, true>>(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
        case 4: return launch_gemm2_cfg<Gemm2Cfg<256, 4, B_MN, true>>(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
        case kScaledLo: return launch_gemm2_cfg<Gemm2Cfg<256, kScaledLo, B_MN, true>>(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
        }
        return HEAL_ERR_UNSUPPORTED_MODE;
    }
    switch (nprod) {
    case 1: return launch_gemm2_cfg<Gemm2Cfg<256, 1, B_MN>>(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
    case 2: return launch_gemm2_cfg<Gemm2Cfg<256, 2, B_MN>>(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
    case 3: return launch_gemm2_cfg<Gemm2Cfg<256, 3, B_MN>>(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
    case 4: return launch_gemm2_cfg<Gemm2Cfg<256, 4, B_MN, true>>(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);   // diagnostic mode: one instantiation
    }
    return HEAL_ERR_UNSUPPORTED_MODE;
}

template <bool B_MN>
int launch_gemm2f_np(int nprod, int64_t M, int64_t N, int64_t K, const float *A, int64_t lda, const void *B_hi, const void *B_lo,
                     int64_t ldb, const OutArgs &out, cudaStream_t s)
{
    const int64_t tiles = ((M + 2 * kBM - 1) / (2 * kBM)) * ((N + 255) / 256);
    if (needs_ext(out) || wants_split_k(tiles, (K + kKSeg - 1) / kKSeg, g.num_sms / 2, 2, 256)) {
        if (nprod == 2) return launch_gemm2f_cfg<Gemm2FCfg<2, B_MN, true>>(M, N, K, A, lda, B_hi, B_lo, ldb, out, s);
        return launch_gemm2f_cfg<Gemm2FCfg<3, B_MN, true>>(M, N, K, A, lda, B_hi, B_lo, ldb, out, s);
    }
    if (nprod == 2) return launch_gemm2f_cfg<Gemm2FCfg<2, B_MN>>(M, N, K, A, lda, B_hi, B_lo, ldb, out, s);
    return launch_gemm2f_cfg<Gemm2FCfg<3, B_MN>>(M, N, K, A, lda, B_hi, B_lo, ldb, out, s);
}

template <int BN, bool B_MN>
int launch_gemm_np(int nprod, int64_t M, int64_t N, int64_t K, const void *A_hi, const void *A_lo, int64_t lda,
                   const void *B_hi, const void *B_lo, int64_t ldb, const OutArgs &out, cudaStream_t s)
{
    const int64_t tiles = ((M + kBM - 1) / kBM) * ((N + BN - 1) / BN);
    if (nprod == kScaledLo || needs_ext(out) || wants_split_k(tiles, (K + kKSeg - 1) / kKSeg, g.num_sms, 1, BN)) {
        switch (nprod) {
        case 1: return launch_gemm_cfg<GemmCfg<BN, 1, B_MN, true>>(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
        case 2: return launch_gemm_cfg<GemmCfg<BN, 2, B_MN, true>>(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
        case 3: return launch_gemm_cfg<GemmCfg<BN, 3, B_MN, true>>(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
        case 4: return launch_gemm_cfg<GemmCfg<BN, 4, B_MN, true>>(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
        case kScaledLo: return launch_gemm_cfg<GemmCfg<BN, kScaledLo, B_MN, true>>(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
        }
        return HEAL_ERR_UNSUPPORTED_MODE;
    }
    switch (nprod) {
    case 1: return launch_gemm_cfg<GemmCfg<BN, 1, B_MN>>(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
    case 2: return launch_gemm_cfg<GemmCfg<BN, 2, B_MN>>(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
    case 3: return launch_gemm_cfg<GemmCfg<BN, 3, B_MN>>(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
    case 4: return launch_gemm_cfg<GemmCfg<BN, 4, B_MN, true>>(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);      // diagnostic mode: one instantiation
    }
    return HEAL_ERR_UNSUPPORTED_MODE;
}

// Tile width: a function of N only (never of M), so the schedule cannot make results depend on M.
template <bool B_MN>
int launch_gemm_bn(int nprod, int64_t M, int64_t N, int64_t K, const void *A_hi, const void *A_lo, int64_t lda,
                   const void *B_hi, const void *B_lo, int64_t ldb, const OutArgs &out, cudaStream_t s)
{
    if (N <= 64) return launch_gemm_np<64, B_MN>(nprod, M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
    if (N <= 128) return launch_gemm_np<128, B_MN>(nprod, M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
    return launch_gemm_np<256, B_MN>(nprod, M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, s);
}

#ifdef HEAL_TRACE
unsigned long long *g_trace = nullptr;
unsigned g_trace_seq = 0;
#endif

// ---- small-M (decode) launch: swap-AB, K segments spread over a cluster ----------------------------
// Activations come either as hi/lo planes (A_hi/A_lo, pitch lda) or, with Cfg::FUSED, as the FP32 matrix
// A32 (pitch lda32) which the kernel splits itself.
struct SmallIn {
    const void *A_hi, *A_lo;
    int64_t lda;
    const float *A32;
    int64_t lda32;
    bool b_static;
    bool fused_any = false;    // FUSED: take the fused kernel also where planes would be faster (the caller cannot have planes)
};

// st.async pushes (lowest latency) pay off while a thread sends few values: up to 8 of any width, or up to 32 8-byte
// vectors (the plain path has no 8-byte form and falls back to 4-byte remote stores, which are slow; measured: M = 16,
// K = 6144 21.7 -> 15.7 us, K = 14336 36.9 -> 26.9 us).
// Token rows finished by one rank of a cluster of c.  A remote store costs about 300 cycles whatever its width (st.async, one warp per
// scheduler: clock stamps), so the rows are dealt in the widest vectors the token count allows: blocks of 4 rows from 3 tokens on
// (16-byte pushes; fewer ranks then own rows), 2 rows for 2 tokens.  Measured: 16 x 4096 x 4096 10.5 -> 9.9 us with 4 pushes of 16
// bytes instead of 8 of 8, M = 24 decode 16.5 us with 4-byte pushes vs 9.9 us at M = 32.
// `narrow`: one or two rows per rank stay as they are (4- and 8-byte pushes, twice as many, but a quarter or half of the partial-sum area).
inline int64_t rows_per_rank(int64_t M, int64_t c, bool narrow = false)
{
    if (c <= 1) return 0;
    const int64_t r = (M + c - 1) / c;
    if (r >= 3 || (M >= 3 && !narrow)) return (r + 3) / 4 * 4;
    return M == 2 ? 2 : r;
}

inline bool async_push_ok(int64_t pushes, int64_t vw)
{
    static const long lim = std::getenv("HEAL_ASYNC_MAX") ? std::atol(std::getenv("HEAL_ASYNC_MAX")) : 8;      // tuning
    return pushes <= lim || (vw == 2 && pushes <= 32);
}

template <class Cfg>
int launch_small_cfg(int64_t M, int64_t N, int64_t K, const SmallIn &in, const void *B_hi, const void *B_lo, int64_t ldb,
                     const OutArgs &out, cudaStream_t stream, bool *handled)
{
    *handled = false;
    const int n_seg = static_cast<int>((K + kKSeg - 1) / kKSeg);
    const int64_t panels = (N + kSmallBNW - 1) / kSmallBNW;
    // Cluster size: the smallest that gives about 1.4 CTAs per SM (measured: enough to saturate HBM), at most 8
    // and at most n_seg.  Purely a performance choice: the result does not depend on it (segment sums are exact copies).
    int cs = 1;
    while (!Cfg::PAIR && cs * 2 <= 8 && cs * 2 <= n_seg && panels * cs * 5 < 7 * g.num_sms) cs *= 2;
    // The doubling above ignores balance: with n_seg = 28 (K = 14336) a cluster of 8 leaves four ranks with 4 segments
    // and four with 3.  For few tokens (cheap reduction) take instead the smallest cluster, down to cs/2 + 1, that keeps
    // the longest rank as short, as long as about 1.2 CTAs per SM remain (measured: K = 14336 M = 1 26.1 -> 23.6 us with
    // 7 ranks, K = 6144 M = 8 16.5 -> 13.3 us with 6).
    if (cs > 2 && M <= 16) {
        const int longest = (n_seg + cs - 1) / cs;
        for (int c = cs / 2 + 1; c < cs; ++c) {
            const int64_t r = rows_per_rank(M, c);                              // pushes per thread follow from it
            const int64_t vw = (r & 3) == 0 ? 4 : ((r & 1) == 0 ? 2 : 1);
            if ((n_seg + c - 1) / c == longest && panels * c * 5 >= 6 * g.num_sms && async_push_ok(longest * ((M + vw - 1) / vw), vw)) {
                cs = c;                                                          // (only while the pushes stay st.async)
                break;
            }
        }
    }
    bool forced_cs = false;
    if (const char *e = std::getenv("HEAL_SMALL_CS")) {                          // debug only
        const int want = std::atoi(e);
        if (!Cfg::PAIR && want >= 1 && want <= 8) cs = want <= n_seg ? want : cs;
        forced_cs = true;
    }
    // CTAs of this kernel the GPU holds at once for a cluster size and a shared-memory size.  The driver's occupancy calls answer
    // "one CTA per SM" for every kernel that allocates tensor memory, whatever its size (the hardware does co-locate them: phase
    // stamps show up to three of these CTAs per SM), so the estimate is made here: CTAs per SM by shared memory and registers, and
    // for clusters the driver's own cudaOccupancyMaxActiveClusters table of a plain 192-thread kernel on this 148-SM part (a cluster
    // has to fit into one GPC, and the GPCs have different sizes: e.g. 37 clusters of 7 at two CTAs per SM, not 42).
    static const int reg_limit = [] {                    // CTAs per SM the register file allows (64 K registers, 256 per warp at a time)
        cudaFuncAttributes fa;
        if (cudaFuncGetAttributes(&fa, heal_gemm_smallm_kernel<Cfg>) != cudaSuccess || fa.numRegs <= 0) return 1;
        const int per_warp = (fa.numRegs * 32 + 255) / 256 * 256;
        return 65536 / (per_warp * (kSmallThreads / 32));
    }();
    auto resident = [&](int c, size_t smem_bytes) -> int64_t {
        static const int kClusters148[3][8] = {{148, 74, 45, 33, 26, 22, 15, 15},          // one CTA per SM, cluster size 1..8
                                               {296, 148, 93, 71, 56, 45, 37, 33},         // two
                                               {444, 222, 142, 104, 82, 71, 56, 48}};      // three
        int64_t per_sm = static_cast<int64_t>((228 * 1024) / (smem_bytes + 1024));
        if (per_sm > reg_limit) per_sm = reg_limit;
        if (per_sm < 1) per_sm = 1;
        const int cx = Cfg::PAIR ? 2 : c;
        if (g.num_sms == 148 && per_sm <= 3) return static_cast<int64_t>(kClusters148[per_sm - 1][cx - 1]) * cx;
        if (g.num_sms == 148) return static_cast<int64_t>(kClusters148[2][cx - 1]) * cx * per_sm / 3;
        return per_sm * g.num_sms / cx * cx * (cx > 2 ? 9 : 10) / 10;                      // other parts: a tenth lost to GPC boundaries
    };
    // Everything else follows from the cluster size c and two options (at most two pipeline stages; partial sums overlaid on the
    // pipeline even when small).  status: 0 = launchable, 1 = leave to the large-M kernel.
    struct Plan {
        int status, cs, max_local, ring, tmem_cols, rpr, stages;
        size_t red, smem;
        bool red_alias;
        int64_t grid, slots;               // CTAs of the launch; CTAs the GPU holds at once
        int64_t cost() const { return (grid + slots - 1) / slots * max_local; }     // waves x segments per CTA
        bool fits() const { return grid <= slots; }
    };
    auto plan = [&](int c, bool two_stages, bool force_alias, bool never_alias = false, bool narrow = false) {
        Plan q = {};
        q.status = 1;
        q.cs = c;
        q.max_local = (n_seg + c - 1) / c;
        // One CTA per panel reading planes, and the segments would need more than 256 TMEM columns (one CTA per SM):
        // they cycle through a ring of TMEM slots instead (256 columns, so two CTAs fit per SM and one's epilogue
        // overlaps the other's stream) and the epilogue keeps the running sum.  Measured: LM head M = 64 227 -> 202 us;
        // where everything fits in 256 columns anyway the plain "drain at the end" epilogue is faster (LM head M = 1
        // 161 vs 168 us), so the ring is used only when needed.
        const bool use_ring = c == 1 && !Cfg::FUSED && n_seg * Cfg::MPAD > 256;
        if (use_ring) {
            q.ring = 256 / Cfg::MPAD;
            if (q.ring > n_seg) q.ring = n_seg;
            if (q.ring > 16) q.ring = 16;
        }
        q.tmem_cols = 32;
        while (q.tmem_cols < (use_ring ? q.ring : q.max_local) * Cfg::MPAD) q.tmem_cols *= 2;
        if (q.tmem_cols > 512) return q;
        q.rpr = static_cast<int>(rows_per_rank(M, c, narrow));
        q.red = c > 1 ? static_cast<size_t>(n_seg) * q.rpr * kSmallBNW * 4 : 0;
        // Shared memory.  Measured on B200 (decode 4096 x 4096, LM head): what matters is how many CTAs are resident
        // -- the next kernel's CTAs run their prologue (and with HEAL_B_STATIC prefetch W) beside this kernel's --
        // rather than the depth of one CTA's pipeline: aim for three CTAs per SM (two when a stage exceeds 24 KB,
        // one when the CTA needs more than half of TMEM), at least 2 stages, at most 8 and no more than the CTA
        // has k-tiles.
        // Partial sums pushed by the cluster: a dedicated area when small (decode), else overlaid on the pipeline.
        static const size_t alias_min = std::getenv("HEAL_RED_ALIAS_MIN") ? static_cast<size_t>(std::atol(std::getenv("HEAL_RED_ALIAS_MIN"))) : 16 * 1024;   // debug only
        q.red_alias = !never_alias && (q.red > alias_min || (force_alias && q.red > 0));
        const size_t fixed = (q.red_alias ? 0 : q.red) + Cfg::BAR_BYTES;          // no alignment slack: see the kernel
        size_t budget = q.tmem_cols > 256 ? static_cast<size_t>(kSmemLimit)
                        : (Cfg::STAGE_BYTES <= 24 * 1024 && c > 1 ? static_cast<size_t>(74 * 1024) : static_cast<size_t>(112 * 1024));
        const size_t min_stages = two_stages ? 2 : 3;
        if (budget < fixed + min_stages * static_cast<size_t>(Cfg::STAGE_BYTES) && budget < static_cast<size_t>(112 * 1024)) budget = static_cast<size_t>(112 * 1024);
        if (budget < fixed + min_stages * static_cast<size_t>(Cfg::STAGE_BYTES)) budget = static_cast<size_t>(kSmemLimit);
        if (budget < fixed + 2 * static_cast<size_t>(Cfg::STAGE_BYTES)) return q;            // large-M kernel
        if (q.red_alias && fixed + q.red > static_cast<size_t>(kSmemLimit)) return q;
        q.stages = static_cast<int>((budget - fixed) / Cfg::STAGE_BYTES);
        if (q.stages > (two_stages ? 2 : kSmallMaxStages)) q.stages = two_stages ? 2 : kSmallMaxStages;
        const int steps = q.max_local * kTilesPerSeg * (Cfg::SCALED ? 2 : 1);
        if (q.stages > steps) q.stages = steps;
        if (const char *e = std::getenv("HEAL_SMALL_STAGES")) {                      // debug only
            const int want = std::atoi(e);
            if (want >= 2 && want <= kSmallMaxStages && fixed + static_cast<size_t>(want) * Cfg::STAGE_BYTES <= static_cast<size_t>(kSmemLimit)) q.stages = want;
        }
        q.smem = fixed + static_cast<size_t>(q.stages) * Cfg::STAGE_BYTES;
        if (q.red_alias && q.smem < fixed + q.red) q.smem = fixed + q.red;
        // TMEM must never be oversubscribed by the CTAs an SM can hold: a CTA blocked in tcgen05.alloc has not yet arrived at
        // its cluster barrier, its peers hold TMEM elsewhere while they wait for it, and a cycle of such waits across clusters
        // (or across kernels on concurrent streams) would hang.  Every kernel of the library therefore takes at least the
        // same fraction of an SM's shared memory (228 KB, 1 KB reserved per CTA) as of its 512 TMEM columns, so whatever mix
        // of the library's CTAs fits into an SM's shared memory also fits into its TMEM.
        const size_t need = (static_cast<size_t>(q.tmem_cols) * (228 * 1024) + 511) / 512;
        if (q.smem + 1024 < need) q.smem = need - 1024;
        if (q.smem > static_cast<size_t>(kSmemLimit)) q.smem = static_cast<size_t>(kSmemLimit);
        q.slots = resident(c, q.smem);
        q.grid = Cfg::PAIR ? (panels + 1) / 2 * 2 : panels * c;
        q.status = 0;
        return q;
    };
    // TMEM: a cluster too small for its segments grows (as long as K allows)
    while (!(cs == 1 && !Cfg::FUSED) && ((n_seg + cs - 1) / cs) * Cfg::MPAD > 512 && cs * 2 <= 8 && cs * 2 <= n_seg) cs *= 2;
    Plan pl = plan(cs, false, false);
    if (pl.status) return HEAL_OK;                              // leave to the large-M kernel
    // More than 16 tokens (few tokens: the rule above, which also keeps the pushes st.async): among the cluster sizes from cs/2 + 1
    // that still give about 1.2 CTAs per SM and whose grid is resident, take the one with the fewest segments on its longest rank,
    // the smallest on a tie -- K = 5120 has 10 segments: 5 ranks of 2 instead of 8 ranks of 2 or 1 (measured, planes:
    // 24 x 5120 x 5120 19.2 -> 17.0 us, 64 x 5120 x 5120 25.2 -> 21.3 us, 32 x 7168 x 5120 22.2 -> 20.4 us with 5 ranks instead of 4).
    static const bool no_wave_fit = std::getenv("HEAL_NO_WAVE_CAP") != nullptr;      // debug only
    // All CTAs of the grid should be resident at once: a small second wave pays a whole first-tile latency and streams on a
    // fraction of the SMs (measured: 32 x 6144 x 4096, 384 CTAs of 88 KB, 19.1 us with 88 CTAs in a second wave, 13.7 us in one).
    // If the plan does not fit: two pipeline stages, then the partial sums overlaid on the pipeline, then both.
    if (!pl.fits() && cs > 1 && !forced_cs && !no_wave_fit) {
        for (int opt = 1; opt < 4; ++opt) {
            const Plan q = plan(cs, (opt & 1) != 0, (opt & 2) != 0);
            if (q.status == 0 && q.fits()) { pl = q; break; }
        }
    }
    if (!Cfg::PAIR && !forced_cs && M > 16 && cs > 1) {
        Plan best = pl;
        for (int c = cs / 2 + 1; c <= 8 && c <= n_seg; ++c) {
            if (c == cs || panels * c * 5 < 6 * static_cast<int64_t>(g.num_sms)) continue;
            const Plan q = plan(c, false, false);
            if (q.status == 0 && q.fits() && (q.cost() < best.cost() || (q.cost() == best.cost() && (!best.fits() || q.cs < best.cs)))) best = q;
        }
        pl = best;
    }
    // fused split on one CTA per panel (large N: every CTA walks the whole of K): the per-k-tile hand-over between the converter warps
    // and the MMA thread costs more over 64+ k-tiles than the split launch it saves (measured, M = 1 / 16: 28672 x 4096 41.0 / 43.9 us
    // fused vs 38.0 / 38.4 us on planes, LM head 175 / 186 vs 170 / 175 us, 65536 x 5120 110 / 116 vs 107 / 110 us)
    static const bool fused_long = std::getenv("HEAL_FUSED_LONG") != nullptr;      // debug only
    if (Cfg::FUSED && pl.cs == 1 && n_seg >= 4 && !forced_cs && !fused_long && !in.fused_any) return HEAL_OK;
    // fused split with more than 16 tokens: the converter warps only keep up while at most two CTAs share an SM; past that the
    // caller splits first and comes back with planes (measured, M = 32: 5120 x 5120 32.2 fused vs 19.5 us, 6144 x 4096 21.1 vs 15.6 us)
    if (Cfg::FUSED && M > 16 && pl.grid > 2 * static_cast<int64_t>(g.num_sms) && !forced_cs && !in.fused_any) return HEAL_OK;
    // Still not resident: the cluster size (and options) with the fewest waves x segments per CTA, the smallest such cluster first
    // (measured: 24 x 5120 x 17408 90 -> 40 us with clusters of 6 instead of 8, 64 x 10240 x 8192 80 -> 53 us,
    // 32 x 8192 x 28672 138 -> 99 us).
    if (!pl.fits() && cs > 1 && !forced_cs && !no_wave_fit) {
        for (int c = 1; c <= 8; ++c) {
            if (c > n_seg || c == cs) continue;
            for (int opt = 0; opt < 4; ++opt) {
                const Plan q = plan(c, (opt & 1) != 0, (opt & 2) != 0);
                if (q.status == 0 && q.cost() < pl.cost()) pl = q;
            }
        }
    }
    // Partial sums overlaid on the pipeline cost a second cluster barrier -- nobody may push before every rank's main loop is over, so
    // the pushes (about 300 cycles each) no longer overlap the wait for the slowest rank.  A dedicated area is better whenever the grid
    // stays resident with at least three stages (measured: 8 x 8192 x 8192 27.3 -> 24.6 us, 16 x 8192 x 8192 28.9 -> 25.7 us,
    // 2 x 4096 x 14336 27.0 -> 23.1 us; with two stages it is worse: 16 x 4096 x 14336 29.2 vs 38.9 us).
    static const bool no_dedicated = std::getenv("HEAL_NO_DEDICATED_RED") != nullptr;      // debug only
    static const long dedicated_max_m = std::getenv("HEAL_DEDICATED_MAX_M") ? std::atol(std::getenv("HEAL_DEDICATED_MAX_M")) : 64;      // tuning
    if (pl.red_alias && pl.cs > 1 && M <= dedicated_max_m && !no_dedicated) {       // (beyond 16 tokens it rarely fits: 24 x 6144 x 4096 16.3 -> 15.8 us)
        for (int narrow = 0; narrow < 2; ++narrow) {       // (narrow rows: 8 x 4096 x 14336 28.0 us overlaid -> 25.3 us dedicated with 8-byte pushes)
            const Plan q = plan(pl.cs, false, false, true, narrow != 0);
            if (q.status == 0 && q.fits() && q.stages >= 3 && !q.red_alias) { pl = q; break; }
        }
    }
    static const bool plan_debug = std::getenv("HEAL_PLAN_DEBUG") != nullptr;      // debug only
    if (plan_debug)
        std::fprintf(stderr, "[heal plan] M=%lld N=%lld K=%lld MPAD=%d fused=%d: cs %d -> %d, grid %lld slots %lld, max_local %d, tmem %d, stages %d, smem %zu, red %zu alias %d\n",
                     (long long)M, (long long)N, (long long)K, Cfg::MPAD, (int)Cfg::FUSED, cs, pl.cs, (long long)pl.grid, (long long)pl.slots, pl.max_local, pl.tmem_cols,
                     pl.stages, pl.smem, pl.red, (int)pl.red_alias);
    cs = pl.cs;
    const int max_local = pl.max_local, ring = pl.ring, tmem_cols = pl.tmem_cols, rpr = pl.rpr, stages = pl.stages;
    const size_t red = pl.red, smem = pl.smem;
    const bool red_alias = pl.red_alias;
    auto kern = heal_gemm_smallm_kernel<Cfg>;
    static std::atomic<size_t> attr_smem{0};           // only ever raised: a concurrent smaller request cannot lower it
    if (smem > attr_smem.load(std::memory_order_acquire)) {
        HEAL_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(kSmemLimit)));
        attr_smem.store(static_cast<size_t>(kSmemLimit), std::memory_order_release);
    }
    CUtensorMap tx_hi, tx_lo, tw_hi, tw_lo;
    int st;
    if (Cfg::B_MN) st = encode_f16_2d(&tw_hi, B_hi, N, K, ldb, 64, kBK);
    else           st = encode_f16_2d(&tw_hi, B_hi, K, N, ldb, kBK, kSmallBNW);
    if (st) return st;
    if (Cfg::B_PLANES == 2) {
        if (Cfg::B_MN) st = encode_f16_2d(&tw_lo, B_lo, N, K, ldb, 64, kBK);
        else           st = encode_f16_2d(&tw_lo, B_lo, K, N, ldb, kBK, kSmallBNW);
        if (st) return st;
    } else {
        tw_lo = tw_hi;
    }
    if (Cfg::FUSED) {
        tx_hi = tx_lo = tw_hi;                                  // unused by the fused kernel
    } else {
        st = encode_f16_2d(&tx_hi, in.A_hi, K, M, in.lda, kBK, Cfg::XROWS);
        if (st) return st;
        if (Cfg::A_PLANES == 2) {
            st = encode_f16_2d(&tx_lo, in.A_lo, K, M, in.lda, kBK, Cfg::XROWS);
            if (st) return st;
        } else {
            tx_lo = tx_hi;
        }
    }
    SmallArgs args;
    args.out = out;
    args.A = in.A32;
    args.lda = in.lda32;
    args.M = static_cast<int>(M);
    args.N = static_cast<int>(N);
    args.K = static_cast<int>(K);
    args.n_seg = n_seg;
    args.max_local = max_local;
    args.tmem_cols = tmem_cols;
    args.stages = stages;
    args.rows_per_rank = rpr;
    args.red_bytes = static_cast<int>(red);
    args.red_alias = red_alias ? 1 : 0;
    {
        // pushes per thread: few -> st.async (lowest latency), many -> plain remote stores + one fence/arrive per warp
        const int vw = (rpr & 3) == 0 ? 4 : ((rpr & 1) == 0 ? 2 : 1);
        const int64_t pushes = cs > 1 ? static_cast<int64_t>(max_local) * ((M + vw - 1) / vw) : 0;
        static const bool no_async = std::getenv("HEAL_NO_ASYNC_PUSH") != nullptr;        // debug only
        args.red_async = (cs > 1 && async_push_ok(pushes, vw) && !no_async) ? 1 : 0;
    }
    args.ring = ring;
    static const bool no_early = std::getenv("HEAL_NO_EARLY_PUSH") != nullptr;      // debug only
    args.early_push = (cs > 1 && !red_alias && max_local >= 2 && max_local <= 16 && !no_early) ? 1 : 0;
    static const bool no_static = std::getenv("HEAL_NO_STATIC") != nullptr;       // debug only
    args.b_static = (in.b_static && !no_static) ? 1 : 0;
    args.diag = g.diag;
    args.trace = nullptr;
#ifdef HEAL_TRACE
    if (g_trace) {                      // 16 rotating regions of 1024 CTAs x 16 stamps
        args.trace = g_trace + (g_trace_seq % 16) * (1024 * 64);
        ++g_trace_seq;
    }
#endif
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(Cfg::PAIR ? (panels + 1) / 2 * 2 : panels * cs));
    cfg.blockDim = dim3(kSmallThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[3];
    cfg.numAttrs = fill_attrs(attr, Cfg::PAIR ? 2u : static_cast<unsigned>(cs));
    cfg.attrs = attr;
    HEAL_CUDA(cudaLaunchKernelEx(&cfg, kern, tx_hi, tx_lo, tw_hi, tw_lo, args));
    g_launches.fetch_add(1);
    static const std::string name = kernel_name("heal_gemm_smallm_kernel", Cfg::MPAD, Cfg::NPROD, Cfg::B_MN,
                                                Cfg::FUSED ? ",fused split"
                                                           : (Cfg::SCALED ? (Cfg::PAIR ? ",cta_group::2,scaled lo" : ",scaled lo")
                                                                          : (Cfg::PAIR ? ",cta_group::2" : "")));
    t_last_kernel = name.c_str();
    *handled = true;
    return HEAL_OK;
}

template <int MPAD, bool B_MN>
int launch_small_np(int nprod, int64_t M, int64_t N, int64_t K, const SmallIn &in, const void *B_hi, const void *B_lo,
                    int64_t ldb, const OutArgs &out, cudaStream_t s, bool *handled)
{
    if (in.A32) {                                               // fused split: FP16 weights only
        switch (nprod) {
        case 1: return launch_small_cfg<SmallCfg<MPAD, 1, B_MN, true>>(M, N, K, in, B_hi, B_lo, ldb, out, s, handled);
        case 2: return launch_small_cfg<SmallCfg<MPAD, 2, B_MN, true>>(M, N, K, in, B_hi, B_lo, ldb, out, s, handled);
        }
        return HEAL_ERR_UNSUPPORTED_MODE;
    }
    // Large N (no K split) and more than 32 tokens: pairs of panels share one cta_group::2 MMA, so each CTA receives only
    // half of the token tile (at MPAD = 64 it is as large as the weight tile, and the unpaired kernel runs into the
    // L2 -> SM delivery cap).  Same bits.
    if constexpr (MPAD == 64) {
        static const bool no_pair = std::getenv("HEAL_NO_PAIR") != nullptr;      // debug only
        const int64_t panels = (N + kSmallBNW - 1) / kSmallBNW;
        if (!no_pair && panels * 5 >= 7 * g.num_sms) {
            switch (nprod) {
            case 1: return launch_small_cfg<SmallCfg<MPAD, 1, B_MN, false, true>>(M, N, K, in, B_hi, B_lo, ldb, out, s, handled);
            case 2: return launch_small_cfg<SmallCfg<MPAD, 2, B_MN, false, true>>(M, N, K, in, B_hi, B_lo, ldb, out, s, handled);
            case 3: return launch_small_cfg<SmallCfg<MPAD, 3, B_MN, false, true>>(M, N, K, in, B_hi, B_lo, ldb, out, s, handled);
            case 4: return launch_small_cfg<SmallCfg<MPAD, 4, B_MN, false, true>>(M, N, K, in, B_hi, B_lo, ldb, out, s, handled);
            case kScaledLo: return launch_small_cfg<SmallCfg<MPAD, kScaledLo, B_MN, false, true>>(M, N, K, in, B_hi, B_lo, ldb, out, s, handled);
            }
        }
    }
    switch (nprod) {
    case 1: return launch_small_cfg<SmallCfg<MPAD, 1, B_MN, false>>(M, N, K, in, B_hi, B_lo, ldb, out, s, handled);
    case 2: return launch_small_cfg<SmallCfg<MPAD, 2, B_MN, false>>(M, N, K, in, B_hi, B_lo, ldb, out, s, handled);
    case 3: return launch_small_cfg<SmallCfg<MPAD, 3, B_MN, false>>(M, N, K, in, B_hi, B_lo, ldb, out, s, handled);
    case 4: return launch_small_cfg<SmallCfg<MPAD, 4, B_MN, false>>(M, N, K, in, B_hi, B_lo, ldb, out, s, handled);
    case kScaledLo: return launch_small_cfg<SmallCfg<MPAD, kScaledLo, B_MN, false>>(M, N, K, in, B_hi, B_lo, ldb, out, s, handled);
    }
    return HEAL_ERR_UNSUPPORTED_MODE;
}

template <bool B_MN>
int launch_small(int nprod, int64_t M, int64_t N, int64_t K, const SmallIn &in, const void *B_hi, const void *B_lo,
                 int64_t ldb, const OutArgs &out, cudaStream_t s, bool *handled)
{
    if (M <= 16) return launch_small_np<16, B_MN>(nprod, M, N, K, in, B_hi, B_lo, ldb, out, s, handled);
    if (M <= 32) return launch_small_np<32, B_MN>(nprod, M, N, K, in, B_hi, B_lo, ldb, out, s, handled);
    return launch_small_np<64, B_MN>(nprod, M, N, K, in, B_hi, B_lo, ldb, out, s, handled);
}

// Debug only: HEAL_FORCE_KERNEL=large|small|1cta (or heal_debug_force_kernel) overrides the kernel choice;
// results are bit-identical whichever kernel runs.
std::atomic<int> g_force{-1};
int forced_kernel()
{
    int v = g_force.load();
    if (v < 0) {
        const char *e = std::getenv("HEAL_FORCE_KERNEL");
        v = !e ? 0 : (e[0] == 'l' ? 1 : (e[0] == 's' ? 2 : (e[0] == '1' ? 3 : 0)));
        g_force.store(v);
    }
    return v;
}

int validate_mode(uint32_t mode, int *nprod, bool *b_nk)
{
    if (mode & ~(HEAL_MODE_PRODUCTS_MASK | HEAL_B_NK | HEAL_B_STATIC | HEAL_LO_SCALED | HEAL_EPI_SILU_MUL | HEAL_EPI_ACCUMULATE | HEAL_FUSE_SPLIT))
        return HEAL_ERR_UNSUPPORTED_MODE;
    const uint32_t p = mode & HEAL_MODE_PRODUCTS_MASK;
    if (p < 1 || p > 4) return HEAL_ERR_UNSUPPORTED_MODE;
    if ((mode & HEAL_LO_SCALED) && p != 2) return HEAL_ERR_UNSUPPORTED_MODE;      // Eq. 10 as printed: two products only
    *nprod = static_cast<int>(p);
    *b_nk = (mode & HEAL_B_NK) != 0;
    return HEAL_OK;
}

// A32 != nullptr: FP32 activations for the fused small-M kernel (M <= 64, FP16 weights) instead of planes
int presplit_impl(int64_t M, int64_t N, int64_t K, const void *A_hi, const void *A_lo, int64_t lda, const void *B_hi,
                  const void *B_lo, int64_t ldb, const OutArgs &out, int nprod, bool b_nk, bool b_static,
                  cudaStream_t stream, const float *A32 = nullptr, int64_t lda32 = 0, bool *handled_out = nullptr, bool fused_any = false)
{
    if (handled_out) *handled_out = true;
    if (K == 0) {                                       // empty sum: zeros in every requested output (SiLU(0) * 0 = 0 as well)
        const int64_t n_out = out.silu ? N / 2 : N;
        if (out.C && !out.accumulate)                    // accumulate: C + 0 = C
            HEAL_CUDA(cudaMemset2DAsync(out.C, static_cast<size_t>(out.ldc) * 4, 0, static_cast<size_t>(n_out) * 4,
                                        static_cast<size_t>(M), stream));
        if (out.hi && out.accumulate)                    // planes of the unchanged residual
            return launch_split(M, n_out, out.C, out.ldc, out.hi, out.lo, out.ld16, stream);
        if (out.hi) {
            HEAL_CUDA(cudaMemset2DAsync(out.hi, static_cast<size_t>(out.ld16) * 2, 0, static_cast<size_t>(n_out) * 2,
                                        static_cast<size_t>(M), stream));
            HEAL_CUDA(cudaMemset2DAsync(out.lo, static_cast<size_t>(out.ld16) * 2, 0, static_cast<size_t>(n_out) * 2,
                                        static_cast<size_t>(M), stream));
        }
        return HEAL_OK;
    }
    const int force = forced_kernel();
    // Scaled residual: the small-M kernel reads every weight tile twice (the second time out of L2), which pays up to 32 tokens
    // (measured: 8 x 4096 x 4096 15.3 vs 24.2 us, LM head M = 1 225 vs 300 us; but M = 64 22.0 vs 21.3 and 310 vs 271 us)
    const int64_t small_max = nprod == kScaledLo && force != 2 ? 32 : 64;
    if (M <= small_max && force != 1) {
        bool handled = false;
        const SmallIn in{A_hi, A_lo, lda, A32, lda32, b_static, fused_any};
        int st = b_nk ? launch_small<false>(nprod, M, N, K, in, B_hi, B_lo, ldb, out, stream, &handled)
                      : launch_small<true>(nprod, M, N, K, in, B_hi, B_lo, ldb, out, stream, &handled);
        if (st || handled) return st;
    }
    if (A32) {                                         // the caller must split first and come back with planes
        *handled_out = false;
        return HEAL_OK;
    }
    if (M > kBM && N > 128 && force != 3) {          // CTA pairs: 256 x 256 tiles
        if (b_nk)
            return launch_gemm2_np<false>(nprod, M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, stream);
        return launch_gemm2_np<true>(nprod, M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, stream);
    }
    if (b_nk)
        return launch_gemm_bn<false>(nprod, M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, stream);
    return launch_gemm_bn<true>(nprod, M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, stream);
}

// workspace layout for heal_gemm: [A_hi][A_lo][B_hi][B_lo], each plane 256-byte aligned
struct WsPlan {
    int64_t lda_p, ldb_p;          // plane pitches (elements)
    size_t a_plane, b_plane;       // bytes per plane (0 if not needed)
    size_t total;
};
WsPlan plan_ws(int64_t M, int64_t N, int64_t K, int nprod, bool b_nk)
{
    WsPlan p;
    p.lda_p = round_up(K, 8);
    p.a_plane = static_cast<size_t>(round_up(M * p.lda_p * 2, 256));
    if (nprod >= 3) {
        const int64_t brows = b_nk ? N : K, bcols = b_nk ? K : N;
        p.ldb_p = round_up(bcols, 8);
        p.b_plane = static_cast<size_t>(round_up(brows * p.ldb_p * 2, 256));
    } else {
        p.ldb_p = 0;
        p.b_plane = 0;
    }
    p.total = 2 * p.a_plane + 2 * p.b_plane;
    return p;
}

int get_ws(size_t bytes, cudaStream_t stream, void **out)
{
    {
        std::lock_guard<std::mutex> lk(g_mu);            // (held for this lookup only, never across a launch)
        if (g.user_ws) {                                 // caller-owned: shared by all streams, the caller serialises
            if (bytes > g.user_ws_bytes) return HEAL_ERR_WORKSPACE;
            *out = g.user_ws;
            return HEAL_OK;
        }
    }
    std::lock_guard<std::mutex> lk(g_xf_mu);
    const bool capturing = stream_capturing(stream);
    State::Xfer *slot = acquire_slot(stream, capturing);
    if (!slot) return HEAL_ERR_WORKSPACE;                // capturing on a stream the library has never seen
    if (bytes > slot->ws_bytes) {
        if (capturing) return HEAL_ERR_WORKSPACE;        // run the call once eagerly, or supply a workspace
        const int st = grow_buffer(slot, stream, &slot->ws, &slot->ws_bytes, bytes);
        if (st) return st;
    }
    *out = slot->ws;
    return HEAL_OK;
}

// Scaled-lo variant (HEAL_LO_SCALED; the paper's h = h_hi + h_lo / 2^10 and Eq. 10 as printed): one kernel, one
// accumulator, two passes per K segment with tcgen05's scale_input_d (GemmCfg::SCALED in heal_gemm_umma.cuh, SmallCfg::SCALED in
// heal_gemm_smallm.cuh).  Same kernel choice by shape as every other mode, same bits whichever kernel runs.
int scaled_impl(int64_t M, int64_t N, int64_t K, const void *A_hi, const void *A_lo, int64_t lda, const void *B, int64_t ldb,
                const OutArgs &out, bool b_nk, bool b_static, cudaStream_t stream)
{
    static_assert(kLoShift == HEAL_LO_SHIFT, "the kernels' scale_input_d immediate is the header's HEAL_LO_SHIFT");
    return presplit_impl(M, N, K, A_hi, A_lo, lda, B, nullptr, ldb, out, kScaledLo, b_nk, b_static, stream);
}

// ---- heal_gemm_static: the allocation-free entry point --------------------------------------------------------------------------
// Scratch of heal_gemm_static (include/heal.h): [0, 256) the kernels' diagnostic words, then the hi and lo FP16 planes of the
// activations.  File-scope device memory: every GPU that loads the library holds these 8 MiB + 256 B until the process exits.  In
// host code the NAME of the array is only a stand-in for the symbol; the device address comes from cudaGetSymbolAddress, taken
// once per device with that device current (static_scratch()).  Zero-initialised at module load, which is all the diagnostic words
// need; the planes are rewritten by step S of every call (rows >= M and columns >= K are never read: the tensor maps end at M and K).
constexpr size_t kStaticDiagBytes = 256;
constexpr size_t kStaticScratchBytes = HEAL_STATIC_SCRATCH_BYTES;
static __device__ __align__(256) unsigned char g_static_scratch[kStaticDiagBytes + kStaticScratchBytes];

int static_scratch(unsigned char **out)
{
    constexpr int kMaxDev = 64;
    static std::mutex mu;
    static unsigned char *ptrs[kMaxDev] = {};
    int dev = -1;
    HEAL_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDev) return HEAL_ERR_UNSUPPORTED_DEVICE;
    std::lock_guard<std::mutex> lk(mu);
    if (!ptrs[dev]) {
        void *p = nullptr;
        HEAL_CUDA(cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p) return HEAL_ERR_CUDA;
        ptrs[dev] = static_cast<unsigned char *>(p);
    }
    *out = ptrs[dev];
    return HEAL_OK;
}

// ensure_init() without its cudaMalloc: if the library has not been initialised yet, the diagnostic words live in the static array
int ensure_init_static(unsigned char *scratch)
{
    {
        std::lock_guard<std::mutex> lk(g_mu);
        if (!g.init) {
            g.init = true;
            auto fail = [&](int st) { g.init_status = st; return st; };
            int dev = 0;
            cudaError_t e = cudaGetDevice(&dev);
            if (e != cudaSuccess) return fail(cuda_fail(e));
            cudaDeviceProp prop;
            e = cudaGetDeviceProperties(&prop, dev);
            if (e != cudaSuccess) return fail(cuda_fail(e));
            if (prop.major != 10) return fail(HEAL_ERR_UNSUPPORTED_DEVICE);
            g.device = dev;
            g.num_sms = prop.multiProcessorCount;
            void *fn = nullptr;
            cudaDriverEntryPointQueryResult qres;
            e = cudaGetDriverEntryPointByVersion("cuTensorMapEncodeTiled", &fn, 12000, cudaEnableDefault, &qres);
            if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn)
                return fail(cuda_fail(e != cudaSuccess ? e : cudaErrorUnknown));
            g.encode = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(fn);
            g.diag = reinterpret_cast<int *>(scratch);
            return HEAL_OK;
        }
    }
    return ensure_init();                  // already initialised: only the status / device check
}

}  // namespace

// =============================================== C ABI ===========================================
extern "C" {

int heal_version(void) { return 100; }

int heal_debug_force_kernel(int which)
{
    if (which < 0 || which > 3) return HEAL_ERR_INVALID_VALUE;
    g_force.store(which);
    return HEAL_OK;
}

#ifdef HEAL_TRACE
// trace builds only (not part of include/heal.h): the pair kernel's wait counters of the most recent launch, 8 values per CTA pair
int heal_debug_read_pair_trace(unsigned long long *host, int n)
{
    return static_cast<int>(cudaMemcpyFromSymbol(host, heal::g_pair_trace, static_cast<size_t>(n) * sizeof(unsigned long long)));
}
// trace builds only (not part of include/heal.h): device buffer of 16 x 1024 x 16 uint64 phase stamps
int heal_debug_set_trace(void *ptr)
{
    g_trace = static_cast<unsigned long long *>(ptr);
    g_trace_seq = 0;
    return HEAL_OK;
}
#endif

int heal_last_cuda_error(void) { return g_last_cuda_error.load(); }

const char *heal_last_kernel(void) { return t_last_kernel; }

uint64_t heal_launch_count(void) { return g_launches.load(); }

const char *heal_status_string(int status)
{
    switch (status) {
    case HEAL_OK: return "HEAL_OK";
    case HEAL_ERR_INVALID_VALUE: return "HEAL_ERR_INVALID_VALUE: negative dimension or leading dimension too small";
    case HEAL_ERR_NULL_POINTER: return "HEAL_ERR_NULL_POINTER: null matrix pointer for a non-empty problem";
    case HEAL_ERR_MISALIGNED: return "HEAL_ERR_MISALIGNED: pointer or leading dimension not 16-byte aligned";
    case HEAL_ERR_UNSUPPORTED_MODE: return "HEAL_ERR_UNSUPPORTED_MODE: unknown mode bits";
    case HEAL_ERR_CUDA: return "HEAL_ERR_CUDA: a CUDA call failed (see heal_last_cuda_error)";
    case HEAL_ERR_WORKSPACE: return "HEAL_ERR_WORKSPACE: supplied workspace too small";
    case HEAL_ERR_UNSUPPORTED_DEVICE:
        return "HEAL_ERR_UNSUPPORTED_DEVICE: current device is not sm_100, or not the device of this process's first call";
    }
    return "unknown heal_status";
}

size_t heal_workspace_size(int64_t M, int64_t N, int64_t K, uint32_t mode)
{
    int nprod;
    bool b_nk;
    if (validate_mode(mode, &nprod, &b_nk) || M < 0 || N < 0 || K < 0) return 0;
    return plan_ws(M, N, K, nprod, b_nk).total;
}

int heal_set_workspace(void *ptr, size_t bytes)
{
    if (ptr && (reinterpret_cast<uintptr_t>(ptr) & 255u)) return HEAL_ERR_MISALIGNED;
    std::lock_guard<std::mutex> lk(g_mu);
    g.user_ws = ptr;
    g.user_ws_bytes = ptr ? bytes : 0;
    return HEAL_OK;
}

int heal_split(int64_t rows, int64_t cols, const void *X, int64_t ldx, void *hi, void *lo, int64_t ld, void *stream)
{
    return heal_split_scaled(rows, cols, X, ldx, hi, lo, ld, 0, stream);
}

int heal_split_scaled(int64_t rows, int64_t cols, const void *X, int64_t ldx, void *hi, void *lo, int64_t ld,
                      int32_t lo_shift, void *stream)
{
    if (lo_shift < 0 || lo_shift > 16) return HEAL_ERR_INVALID_VALUE;
    if (rows < 0 || cols < 0 || ldx < cols || ld < cols) return HEAL_ERR_INVALID_VALUE;
    if (rows == 0 || cols == 0) return HEAL_OK;
    if (!X || !hi || !lo) return HEAL_ERR_NULL_POINTER;
    if (!aligned16(X) || !aligned16(hi) || !aligned16(lo) || (ldx & 3) || (ld & 7)) return HEAL_ERR_MISALIGNED;
    int st = ensure_init();
    if (st) return st;
    return launch_split(rows, cols, static_cast<const float *>(X), ldx, static_cast<__half *>(hi),
                        static_cast<__half *>(lo), ld, static_cast<cudaStream_t>(stream), lo_shift);
}

int heal_rmsnorm_split(int64_t rows, int64_t cols, const void *X, int64_t ldx, const void *gamma, float eps, void *hi, void *lo,
                       int64_t ld, void *Y, int64_t ldy, void *stream)
{
    if (rows < 0 || cols < 0 || ldx < cols || ld < cols || (Y && ldy < cols) || !(eps >= 0.0f)) return HEAL_ERR_INVALID_VALUE;
    if (rows == 0 || cols == 0) return HEAL_OK;
    if (!X || !hi || !lo) return HEAL_ERR_NULL_POINTER;
    if (!aligned16(X) || !aligned16(hi) || !aligned16(lo) || !aligned16(gamma) || !aligned16(Y) || (ldx & 3) || (ld & 7) || (Y && (ldy & 3)))
        return HEAL_ERR_MISALIGNED;
    int st = ensure_init();
    if (st) return st;
    cudaLaunchConfig_t cfg = {};
    const int64_t cap = static_cast<int64_t>(g.num_sms) * 8;
    cfg.gridDim = dim3(static_cast<unsigned>(rows < cap ? rows : cap));
    cfg.blockDim = dim3(256);
    cfg.stream = static_cast<cudaStream_t>(stream);
    cudaLaunchAttribute attr[3];
    cfg.numAttrs = fill_attrs(attr, 1);
    cfg.attrs = attr;
    HEAL_CUDA(cudaLaunchKernelEx(&cfg, heal_rmsnorm_split_kernel, static_cast<const float *>(X), ldx, rows, cols,
                                 static_cast<const float *>(gamma), eps, static_cast<__half *>(hi), static_cast<__half *>(lo), ld,
                                 static_cast<float *>(Y), ldy));
    g_launches.fetch_add(1);
    return HEAL_OK;
}

// Output validation shared by the _ex entry points: builds the OutArgs of step E.
static int make_out(int64_t M, int64_t N, void *C, int64_t ldc, void *C_hi, void *C_lo, int64_t ldc16, int scale_exp,
                    uint32_t mode, heal::OutArgs *out)
{
    const bool silu = (mode & HEAL_EPI_SILU_MUL) != 0, acc = (mode & HEAL_EPI_ACCUMULATE) != 0;
    if (scale_exp < -126 || scale_exp > 126) return HEAL_ERR_INVALID_VALUE;
    if (silu && (N & 1)) return HEAL_ERR_INVALID_VALUE;                    // (gate, up) column pairs
    const int64_t n_out = silu ? N / 2 : N;
    if ((C || !C_hi) && ldc < n_out) return HEAL_ERR_INVALID_VALUE;
    if ((C_hi || C_lo) && ldc16 < n_out) return HEAL_ERR_INVALID_VALUE;
    if (M == 0 || N == 0) return HEAL_OK;
    if (!C && !C_hi) return HEAL_ERR_NULL_POINTER;
    if (acc && !C) return HEAL_ERR_NULL_POINTER;                           // the residual lives in C
    if ((C_hi == nullptr) != (C_lo == nullptr)) return HEAL_ERR_NULL_POINTER;
    if (C && (!aligned16(C) || (ldc & 3))) return HEAL_ERR_MISALIGNED;
    if (C_hi && (!aligned16(C_hi) || !aligned16(C_lo) || (ldc16 & 7))) return HEAL_ERR_MISALIGNED;
    out->C = static_cast<float *>(C);
    out->ldc = ldc;
    out->hi = static_cast<__half *>(C_hi);
    out->lo = static_cast<__half *>(C_lo);
    out->ld16 = ldc16;
    // 2^-scale_exp, built from its bit pattern (normal for |scale_exp| <= 126)
    const uint32_t bits = static_cast<uint32_t>(127 - scale_exp) << 23;
    float sc;
    memcpy(&sc, &bits, 4);
    out->scale = sc;
    out->accumulate = acc ? 1 : 0;
    out->silu = silu ? 1 : 0;
    return HEAL_OK;
}

int heal_gemm_presplit_ex(int64_t M, int64_t N, int64_t K, const void *A_hi, const void *A_lo, int64_t lda,
                          const void *B_hi, const void *B_lo, int64_t ldb, void *C, int64_t ldc, void *C_hi, void *C_lo,
                          int64_t ldc16, int32_t scale_exp, uint32_t mode, void *stream)
{
    int nprod;
    bool b_nk;
    int st = validate_mode(mode, &nprod, &b_nk);
    if (st) return st;
    if (M < 0 || N < 0 || K < 0) return HEAL_ERR_INVALID_VALUE;
    if (M > 0x7fffff00 || N > 0x7fffff00 || K > 0x7fffff00) return HEAL_ERR_INVALID_VALUE;
    if (lda < K || ldb < (b_nk ? K : N)) return HEAL_ERR_INVALID_VALUE;
    heal::OutArgs out = {};
    st = make_out(M, N, C, ldc, C_hi, C_lo, ldc16, scale_exp, mode, &out);
    if (st) return st;
    if (M == 0 || N == 0) return HEAL_OK;
    if (K > 0) {
        if (!A_hi || !B_hi) return HEAL_ERR_NULL_POINTER;
        if (nprod >= 2 && !A_lo) return HEAL_ERR_NULL_POINTER;
        if (nprod >= 3 && !B_lo) return HEAL_ERR_NULL_POINTER;
        if (!aligned16(A_hi) || !aligned16(A_lo) || !aligned16(B_hi) || !aligned16(B_lo) || (lda & 7) || (ldb & 7))
            return HEAL_ERR_MISALIGNED;
    }
    st = ensure_init();
    if (st) return st;
    if ((mode & HEAL_LO_SCALED) && K > 0)          // A_lo holds r16((x - hi) * 2^10), e.g. from heal_split_scaled(.., 10, ..)
        return scaled_impl(M, N, K, A_hi, A_lo, lda, B_hi, ldb, out, b_nk, (mode & HEAL_B_STATIC) != 0, static_cast<cudaStream_t>(stream));
    return presplit_impl(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, out, nprod, b_nk, (mode & HEAL_B_STATIC) != 0,
                         static_cast<cudaStream_t>(stream));
}

int heal_gemm_presplit(int64_t M, int64_t N, int64_t K, const void *A_hi, const void *A_lo, int64_t lda,
                       const void *B_hi, const void *B_lo, int64_t ldb, void *C, int64_t ldc, uint32_t mode,
                       void *stream)
{
    return heal_gemm_presplit_ex(M, N, K, A_hi, A_lo, lda, B_hi, B_lo, ldb, C, ldc, nullptr, nullptr, 0, 0, mode, stream);
}

int heal_gemm_ex(int64_t M, int64_t N, int64_t K, const void *A, int64_t lda, const void *B, int64_t ldb, void *C,
                 int64_t ldc, void *C_hi, void *C_lo, int64_t ldc16, int32_t scale_exp, uint32_t mode, void *stream_)
{
    int nprod;
    bool b_nk;
    int st = validate_mode(mode, &nprod, &b_nk);
    if (st) return st;
    if (M < 0 || N < 0 || K < 0) return HEAL_ERR_INVALID_VALUE;
    if (M > 0x7fffff00 || N > 0x7fffff00 || K > 0x7fffff00) return HEAL_ERR_INVALID_VALUE;
    if (lda < K || ldb < (b_nk ? K : N)) return HEAL_ERR_INVALID_VALUE;
    heal::OutArgs out = {};
    st = make_out(M, N, C, ldc, C_hi, C_lo, ldc16, scale_exp, mode, &out);
    if (st) return st;
    if (M == 0 || N == 0) return HEAL_OK;
    const bool b_f32 = nprod >= 3;
    if (K > 0) {
        if (!A || !B) return HEAL_ERR_NULL_POINTER;
        if (!aligned16(A) || !aligned16(B) || (lda & 3) || (ldb & (b_f32 ? 3 : 7))) return HEAL_ERR_MISALIGNED;
    }
    st = ensure_init();
    if (st) return st;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const bool b_static = (mode & HEAL_B_STATIC) != 0;
    if (K == 0) return presplit_impl(M, N, K, nullptr, nullptr, lda, nullptr, nullptr, ldb, out, nprod, b_nk, b_static, stream);
    static const bool no_fused = std::getenv("HEAL_NO_FUSED") != nullptr;          // debug only
    const bool lo_scaled = (mode & HEAL_LO_SCALED) != 0;
    // Decode shapes with FP16 weights: step S runs inside the small-M GEMM kernel (no planes, one launch) while the conversion
    // work of a CTA stays small next to its weight stream: up to 16 tokens always (K <= 16384), up to 32 tokens for small
    // problems, where the second launch costs more than the conversion (measured with the packed conversion of split2:
    // 32 x 4096 x 4096 12.1 -> 10.9 us, 24 x 6144 x 4096 22.0 -> 19.9 us, 1 x 4096 x 14336 25.6 -> 23.8 us; but
    // 32 x 28672 x 4096 44.8 vs 51.0 us, 32 x 4096 x 14336 36.0 vs 39.7 us, LM head M = 32 177 vs 199 us fused).
    static const long fused_max_m = std::getenv("HEAL_FUSED_MAX_M") ? std::atol(std::getenv("HEAL_FUSED_MAX_M")) : 0;        // tuning
    const bool fuse_small = fused_max_m > 0 ? (M <= fused_max_m && K <= 16384)
                                            : ((M <= 16 && K <= 16384) || (M <= 32 && K <= 8192 && N * K <= (static_cast<int64_t>(32) << 20)));
    if (fuse_small && !b_f32 && !no_fused && !lo_scaled && forced_kernel() != 1) {
        bool handled = false;
        st = presplit_impl(M, N, K, nullptr, nullptr, 0, B, nullptr, ldb, out, nprod, b_nk, b_static, stream,
                           static_cast<const float *>(A), lda, &handled);
        if (st || handled) return st;
        // left to split + planes because that is faster -- but a captured call on a stream without a workspace cannot have planes:
        // the fused kernel then, rather than HEAL_ERR_WORKSPACE
        if (stream_capturing(stream)) {
            void *probe = nullptr;
            if (get_ws(plan_ws(M, N, K, nprod, b_nk).total, stream, &probe) == HEAL_ERR_WORKSPACE) {
                st = presplit_impl(M, N, K, nullptr, nullptr, 0, B, nullptr, ldb, out, nprod, b_nk, b_static, stream,
                                   static_cast<const float *>(A), lda, &handled, true);
                if (st || handled) return st;
            }
        }
    }

    // Prefill shapes served by the CTA-pair kernel (M > 128, N > 128), two or three products: step S of the activations can run
    // inside the GEMM kernel (heal_gemm_umma2f.cuh) -- one launch and no workspace for FP16 weights.  Measured on B200 it is
    // 0-13 % slower than split + GEMM (the in-place conversion shares the shared-memory bandwidth with the tensor core:
    // 176 KB instead of 112 KB per k-tile), so it is used on request (HEAL_FUSE_SPLIT) and whenever the planes cannot be
    // had: a captured call on a stream whose library workspace is missing or too small (instead of HEAL_ERR_WORKSPACE).
    static const bool force_fused_large = std::getenv("HEAL_FUSED_LARGE") != nullptr;      // debug only
    bool fuse_a = M > kBM && N > 128 && (nprod == 2 || nprod == 3) && !lo_scaled && !no_fused && forced_kernel() == 0;
    if (fuse_a && !(mode & HEAL_FUSE_SPLIT) && !force_fused_large) {
        fuse_a = false;
        if (!b_f32 && stream_capturing(stream)) {
            void *probe = nullptr;
            if (get_ws(plan_ws(M, N, K, nprod, b_nk).total, stream, &probe) == HEAL_ERR_WORKSPACE) fuse_a = true;
        }
    }
    const WsPlan p = plan_ws(M, N, K, nprod, b_nk);
    void *ws = nullptr;
    if (!(fuse_a && !b_f32)) {
        st = get_ws(p.total, stream, &ws);
        if (st) return st;
    }
    char *w = static_cast<char *>(ws);
    if (fuse_a) {
        const void *b_hi = B, *b_lo = nullptr;
        int64_t ldb_eff = ldb;
        if (b_f32) {
            __half *bh = reinterpret_cast<__half *>(w + 2 * p.a_plane);
            __half *bl = reinterpret_cast<__half *>(w + 2 * p.a_plane + p.b_plane);
            const int64_t brows = b_nk ? N : K, bcols = b_nk ? K : N;
            st = launch_split(brows, bcols, static_cast<const float *>(B), ldb, bh, bl, p.ldb_p, stream);
            if (st) return st;
            b_hi = bh;
            b_lo = bl;
            ldb_eff = p.ldb_p;
        }
        if (b_nk) return launch_gemm2f_np<false>(nprod, M, N, K, static_cast<const float *>(A), lda, b_hi, b_lo, ldb_eff, out, stream);
        return launch_gemm2f_np<true>(nprod, M, N, K, static_cast<const float *>(A), lda, b_hi, b_lo, ldb_eff, out, stream);
    }
    __half *a_hi = reinterpret_cast<__half *>(w);
    __half *a_lo = reinterpret_cast<__half *>(w + p.a_plane);
    // step S on the activations; in 1P only the hi plane is consumed
    st = launch_split(M, K, static_cast<const float *>(A), lda, a_hi, a_lo, p.lda_p, stream, lo_scaled ? HEAL_LO_SHIFT : 0);
    if (st) return st;
    if (lo_scaled) return scaled_impl(M, N, K, a_hi, a_lo, p.lda_p, B, ldb, out, b_nk, (mode & HEAL_B_STATIC) != 0, stream);
    const void *b_hi = B, *b_lo = nullptr;
    int64_t ldb_eff = ldb;
    if (b_f32) {
        __half *bh = reinterpret_cast<__half *>(w + 2 * p.a_plane);
        __half *bl = reinterpret_cast<__half *>(w + 2 * p.a_plane + p.b_plane);
        const int64_t brows = b_nk ? N : K, bcols = b_nk ? K : N;
        st = launch_split(brows, bcols, static_cast<const float *>(B), ldb, bh, bl, p.ldb_p, stream);
        if (st) return st;
        b_hi = bh;
        b_lo = bl;
        ldb_eff = p.ldb_p;
    }
    // FP32 B: its planes were written by the split kernel just launched on this stream, so the static-weights
    // promise cannot be passed on (the GEMM would prefetch them before that kernel has finished)
    return presplit_impl(M, N, K, a_hi, a_lo, p.lda_p, b_hi, b_lo, ldb_eff, out, nprod, b_nk, b_static && !b_f32, stream);
}

int heal_gemm(int64_t M, int64_t N, int64_t K, const void *A, int64_t lda, const void *B, int64_t ldb, void *C,
              int64_t ldc, uint32_t mode, void *stream_)
{
    return heal_gemm_ex(M, N, K, A, lda, B, ldb, C, ldc, nullptr, nullptr, 0, 0, mode, stream_);
}

int heal_gemm_static(int64_t M, int64_t N, int64_t K, const void *A, int64_t lda, const void *B, int64_t ldb, void *C,
                     int64_t ldc, uint32_t mode, void *stream_)
{
    int nprod;
    bool b_nk;
    int st = validate_mode(mode, &nprod, &b_nk);
    if (st) return st;
    if (nprod > 2 || (mode & ~(HEAL_MODE_PRODUCTS_MASK | HEAL_B_NK | HEAL_B_STATIC))) return HEAL_ERR_UNSUPPORTED_MODE;
    if (M < 0 || N < 0 || K < 0) return HEAL_ERR_INVALID_VALUE;
    if (N > 0x7fffff00 || K > 0x7fffff00) return HEAL_ERR_INVALID_VALUE;
    if (lda < K || ldb < (b_nk ? K : N) || ldc < N) return HEAL_ERR_INVALID_VALUE;
    if (M > HEAL_STATIC_MAX_M) return HEAL_ERR_WORKSPACE;                        // the decode kernel's range
    const int64_t lda_p = round_up(K > 0 ? K : 1, 8);
    const size_t a_plane = static_cast<size_t>(round_up(M * lda_p * 2, 256));
    if (2 * a_plane > kStaticScratchBytes) return HEAL_ERR_WORKSPACE;            // the planes do not fit the static scratch
    if (M == 0 || N == 0) return HEAL_OK;
    if (!C) return HEAL_ERR_NULL_POINTER;
    if (!aligned16(C) || (ldc & 3)) return HEAL_ERR_MISALIGNED;
    if (K > 0) {
        if (!A || !B) return HEAL_ERR_NULL_POINTER;
        if (!aligned16(A) || !aligned16(B) || (lda & 3) || (ldb & 7)) return HEAL_ERR_MISALIGNED;
    }
    unsigned char *scratch = nullptr;
    st = static_scratch(&scratch);
    if (st) return st;
    st = ensure_init_static(scratch);
    if (st) return st;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    heal::OutArgs out = {};
    out.C = static_cast<float *>(C);
    out.ldc = ldc;
    out.scale = 1.0f;
    const bool b_static = (mode & HEAL_B_STATIC) != 0;
    if (K == 0) return presplit_impl(M, N, K, nullptr, nullptr, lda, nullptr, nullptr, ldb, out, nprod, b_nk, b_static, stream);
    __half *a_hi = reinterpret_cast<__half *>(scratch + kStaticDiagBytes);
    __half *a_lo = reinterpret_cast<__half *>(scratch + kStaticDiagBytes + a_plane);
    st = launch_split(M, K, static_cast<const float *>(A), lda, a_hi, a_lo, lda_p, stream);      // step S into the static planes
    if (st) return st;
    // steps G + E: the small-M kernel only (it needs no further scratch; the large-M kernels' schedules may allocate hand-off buffers)
    bool handled = false;
    const SmallIn in{a_hi, a_lo, lda_p, nullptr, 0, b_static};
    st = b_nk ? launch_small<false>(nprod, M, N, K, in, B, nullptr, ldb, out, stream, &handled)
              : launch_small<true>(nprod, M, N, K, in, B, nullptr, ldb, out, stream, &handled);
    if (st) return st;
    return handled ? HEAL_OK : HEAL_ERR_WORKSPACE;         // (K beyond what 512 TMEM columns and a cluster of 8 hold at this M)
}

int heal_gemm_host(int64_t M, int64_t N, int64_t K, const void *A_host, int64_t lda, const void *B_host, int64_t ldb,
                   void *C_host, int64_t ldc, uint32_t mode, void *stream_)
{
    int nprod;
    bool b_nk;
    int st = validate_mode(mode, &nprod, &b_nk);
    if (st) return st;
    if (M < 0 || N < 0 || K < 0) return HEAL_ERR_INVALID_VALUE;
    if (mode & (HEAL_EPI_SILU_MUL | HEAL_EPI_ACCUMULATE)) return HEAL_ERR_UNSUPPORTED_MODE;     // device entry points only
    if (lda < K || ldc < N || ldb < (b_nk ? K : N)) return HEAL_ERR_INVALID_VALUE;
    if (M == 0 || N == 0) return HEAL_OK;
    if (!C_host || (K > 0 && (!A_host || !B_host))) return HEAL_ERR_NULL_POINTER;
    st = ensure_init();
    if (st) return st;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const size_t b_es = nprod >= 3 ? 4 : 2;
    const int64_t brows = b_nk ? N : K, bcols = b_nk ? K : N;
    // dense device copies with 16-byte-aligned pitches
    const int64_t dlda = round_up(K > 0 ? K : 1, 8), dldb = round_up(bcols > 0 ? bcols : 1, 8), dldc = round_up(N, 4);
    const size_t a_bytes = static_cast<size_t>(round_up(M * dlda * 4, 256));
    const size_t b_bytes = static_cast<size_t>(round_up(brows * dldb * static_cast<int64_t>(b_es), 256));
    const size_t c_bytes = static_cast<size_t>(round_up(M * dldc * 4, 256));
    // one host-variant call at a time: the staging buffers, copy streams and events below are shared
    std::lock_guard<std::mutex> host_lk(g_host_mu);
    // on an error return, nothing may still be reading or writing the caller's host buffers
    struct Drain {
        cudaStream_t s;
        bool armed = true;
        ~Drain()
        {
            if (!armed) return;
            cudaStreamSynchronize(s);
            if (g.copy_in) cudaStreamSynchronize(g.copy_in);
            if (g.copy_out) cudaStreamSynchronize(g.copy_out);
        }
    } drain{stream};
    {
        const size_t need = a_bytes + b_bytes + c_bytes;
        if (need > g.stage_bytes) {
            HEAL_CUDA(cudaStreamSynchronize(stream));
            if (g.stage) HEAL_CUDA(cudaFree(g.stage));
            g.stage = nullptr;
            g.stage_bytes = 0;
            HEAL_CUDA(cudaMalloc(&g.stage, need));
            g.stage_bytes = need;
        }
    }
    char *dA = static_cast<char *>(g.stage), *dB = dA + a_bytes, *dC = dB + b_bytes;
    // Large problems are pipelined over blocks of weight columns: block b's weights travel host -> device on one copy
    // stream while block b-1 is computed and block b-2's results travel device -> host on another, so the two PCIe
    // directions work at the same time.  The per-element reduction order does not depend on the tile or block an
    // element falls in, so the result is bit-identical to the one-shot path.
    const int64_t kBlockCols = 2048;
    const int64_t nb = (K > 0 && N > kBlockCols && static_cast<size_t>(K) * N * b_es >= (static_cast<size_t>(32) << 20)) ? (N + kBlockCols - 1) / kBlockCols : 1;
    if (nb == 1) {
        if (K > 0) {
            HEAL_CUDA(cudaMemcpy2DAsync(dA, dlda * 4, A_host, lda * 4, K * 4, M, cudaMemcpyHostToDevice, stream));
            HEAL_CUDA(cudaMemcpy2DAsync(dB, dldb * b_es, B_host, ldb * b_es, bcols * b_es, brows, cudaMemcpyHostToDevice,
                                        stream));
        }
        st = heal_gemm(M, N, K, dA, dlda, dB, dldb, dC, dldc, mode, stream_);
        if (st) return st;
        HEAL_CUDA(cudaMemcpy2DAsync(C_host, ldc * 4, dC, dldc * 4, N * 4, M, cudaMemcpyDeviceToHost, stream));
        HEAL_CUDA(cudaStreamSynchronize(stream));
        drain.armed = false;
        return HEAL_OK;
    }
    if (!g.copy_in) {
        HEAL_CUDA(cudaStreamCreateWithFlags(&g.copy_in, cudaStreamNonBlocking));
        HEAL_CUDA(cudaStreamCreateWithFlags(&g.copy_out, cudaStreamNonBlocking));
        for (auto &e : g.ev_in) HEAL_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        for (auto &e : g.ev_done) HEAL_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        HEAL_CUDA(cudaEventCreateWithFlags(&g.ev_start, cudaEventDisableTiming));
    }
    constexpr int kEv = 8;                                       // events are recycled round-robin; a block's events are
                                                                 // re-recorded only after the stream that waits on them got there
    HEAL_CUDA(cudaEventRecord(g.ev_start, stream));              // staging buffers are free once earlier work on `stream` is done
    HEAL_CUDA(cudaStreamWaitEvent(g.copy_in, g.ev_start, 0));
    HEAL_CUDA(cudaStreamWaitEvent(g.copy_out, g.ev_start, 0));
    HEAL_CUDA(cudaMemcpy2DAsync(dA, dlda * 4, A_host, lda * 4, K * 4, M, cudaMemcpyHostToDevice, g.copy_in));
    const char *Bh = static_cast<const char *>(B_host);
    // The activations are the same for every block: with FP16 weights and more tokens than the fused decode path takes, split
    // them once (step S) instead of once per block; the blocks then run steps G + E on the planes.  Same bits either way.
    __half *a_hi = nullptr, *a_lo = nullptr;
    int64_t lda_p = 0;
    if (nprod <= 2 && M > 32 && !(mode & (HEAL_LO_SCALED | HEAL_FUSE_SPLIT))) {
        const WsPlan p = plan_ws(M, kBlockCols, K, nprod, b_nk);
        void *ws = nullptr;
        st = get_ws(p.total, stream, &ws);
        if (st) return st;
        a_hi = static_cast<__half *>(ws);
        a_lo = reinterpret_cast<__half *>(static_cast<char *>(ws) + p.a_plane);
        lda_p = p.lda_p;
        HEAL_CUDA(cudaEventRecord(g.ev_start, g.copy_in));                   // A has arrived
        HEAL_CUDA(cudaStreamWaitEvent(stream, g.ev_start, 0));
        st = launch_split(M, K, reinterpret_cast<const float *>(dA), dlda, a_hi, a_lo, lda_p, stream);
        if (st) return st;
    }
    for (int64_t b = 0; b < nb; ++b) {
        const int64_t c0 = b * kBlockCols, cw = (N - c0 < kBlockCols) ? N - c0 : kBlockCols;
        if (b >= kEv) HEAL_CUDA(cudaEventSynchronize(g.ev_done[b % kEv]));       // block b - kEv fully consumed: its events are free
        // weights of this block: columns c0.. (K x N storage) or rows c0.. (N x K storage)
        if (b_nk)
            HEAL_CUDA(cudaMemcpy2DAsync(dB + c0 * dldb * b_es, dldb * b_es, Bh + c0 * ldb * b_es, ldb * b_es, K * b_es, cw,
                                        cudaMemcpyHostToDevice, g.copy_in));
        else
            HEAL_CUDA(cudaMemcpy2DAsync(dB + c0 * b_es, dldb * b_es, Bh + c0 * b_es, ldb * b_es, cw * b_es, K,
                                        cudaMemcpyHostToDevice, g.copy_in));
        HEAL_CUDA(cudaEventRecord(g.ev_in[b % kEv], g.copy_in));
        HEAL_CUDA(cudaStreamWaitEvent(stream, g.ev_in[b % kEv], 0));
        const void *Bblk = b_nk ? dB + c0 * dldb * b_es : dB + c0 * b_es;
        if (a_hi) {
            // FP16 weights, activations split once before the loop: steps G + E on the planes
            heal::OutArgs out = {};
            out.C = reinterpret_cast<float *>(dC + c0 * 4);
            out.ldc = dldc;
            out.scale = 1.0f;
            st = presplit_impl(M, cw, K, a_hi, a_lo, lda_p, Bblk, nullptr, dldb, out, nprod, b_nk, false, stream);
        } else {
            st = heal_gemm(M, cw, K, dA, dlda, Bblk, dldb, dC + c0 * 4, dldc, mode, stream_);
        }
        if (st) return st;
        HEAL_CUDA(cudaEventRecord(g.ev_done[b % kEv], stream));
        HEAL_CUDA(cudaStreamWaitEvent(g.copy_out, g.ev_done[b % kEv], 0));
        HEAL_CUDA(cudaMemcpy2DAsync(static_cast<char *>(C_host) + c0 * 4, ldc * 4, dC + c0 * 4, dldc * 4, cw * 4, M,
                                    cudaMemcpyDeviceToHost, g.copy_out));
    }
    HEAL_CUDA(cudaStreamSynchronize(g.copy_out));
    HEAL_CUDA(cudaStreamSynchronize(stream));
    drain.armed = false;
    return HEAL_OK;
}

int heal_gemm_host_act(int64_t M, int64_t N, int64_t K, const void *A_host, int64_t lda, const void *B, int64_t ldb,
                       void *C_host, int64_t ldc, uint32_t mode, void *stream_)
{
    int nprod;
    bool b_nk;
    int st = validate_mode(mode, &nprod, &b_nk);
    if (st) return st;
    if (M < 0 || N < 0 || K < 0) return HEAL_ERR_INVALID_VALUE;
    if (mode & (HEAL_EPI_SILU_MUL | HEAL_EPI_ACCUMULATE)) return HEAL_ERR_UNSUPPORTED_MODE;     // device entry points only
    if (lda < K || ldc < N || ldb < (b_nk ? K : N)) return HEAL_ERR_INVALID_VALUE;
    if (M == 0 || N == 0) return HEAL_OK;
    if (!C_host || (K > 0 && (!A_host || !B))) return HEAL_ERR_NULL_POINTER;
    if (K > 0 && (!aligned16(B) || (ldb & (nprod >= 3 ? 3 : 7)))) return HEAL_ERR_MISALIGNED;
    st = ensure_init();
    if (st) return st;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const int64_t dlda = round_up(K > 0 ? K : 1, 8), dldc = round_up(N, 4);
    const size_t a_bytes = static_cast<size_t>(round_up(M * dlda * 4, 256));
    const size_t c_bytes = static_cast<size_t>(round_up(M * dldc * 4, 256));
    std::lock_guard<std::mutex> host_lk(g_host_mu);
    struct Drain {
        cudaStream_t s;
        bool armed = true;
        ~Drain()
        {
            if (!armed) return;
            cudaStreamSynchronize(s);
            if (g.copy_in) cudaStreamSynchronize(g.copy_in);
            if (g.copy_out) cudaStreamSynchronize(g.copy_out);
        }
    } drain{stream};
    if (a_bytes + c_bytes > g.stage_bytes) {
        HEAL_CUDA(cudaStreamSynchronize(stream));
        if (g.stage) HEAL_CUDA(cudaFree(g.stage));
        g.stage = nullptr;
        g.stage_bytes = 0;
        HEAL_CUDA(cudaMalloc(&g.stage, a_bytes + c_bytes));
        g.stage_bytes = a_bytes + c_bytes;
    }
    char *dA = static_cast<char *>(g.stage), *dC = dA + a_bytes;
    if (!g.copy_in) {
        HEAL_CUDA(cudaStreamCreateWithFlags(&g.copy_in, cudaStreamNonBlocking));
        HEAL_CUDA(cudaStreamCreateWithFlags(&g.copy_out, cudaStreamNonBlocking));
        for (auto &e : g.ev_in) HEAL_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        for (auto &e : g.ev_done) HEAL_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        HEAL_CUDA(cudaEventCreateWithFlags(&g.ev_start, cudaEventDisableTiming));
    }
    // Blocks of token rows: block b's activations travel in while block b-1 is computed and block b-2's results travel out.  Rows are
    // independent and the reduction order does not depend on M, so the result is bit-identical to one heal_gemm over all rows.
    const int64_t kBlockRows = 512;
    const int64_t nb = (M + kBlockRows - 1) / kBlockRows;
    constexpr int kEv = 8;
    HEAL_CUDA(cudaEventRecord(g.ev_start, stream));
    HEAL_CUDA(cudaStreamWaitEvent(g.copy_in, g.ev_start, 0));
    HEAL_CUDA(cudaStreamWaitEvent(g.copy_out, g.ev_start, 0));
    for (int64_t b = 0; b < nb; ++b) {
        const int64_t r0 = b * kBlockRows, rows = (M - r0 < kBlockRows) ? M - r0 : kBlockRows;
        if (b >= kEv) HEAL_CUDA(cudaEventSynchronize(g.ev_done[b % kEv]));
        if (K > 0)
            HEAL_CUDA(cudaMemcpy2DAsync(dA + r0 * dlda * 4, dlda * 4, static_cast<const char *>(A_host) + r0 * lda * 4, lda * 4, K * 4, rows,
                                        cudaMemcpyHostToDevice, g.copy_in));
        HEAL_CUDA(cudaEventRecord(g.ev_in[b % kEv], g.copy_in));
        HEAL_CUDA(cudaStreamWaitEvent(stream, g.ev_in[b % kEv], 0));
        st = heal_gemm(rows, N, K, dA + r0 * dlda * 4, dlda, B, ldb, dC + r0 * dldc * 4, dldc, mode, stream_);
        if (st) return st;
        HEAL_CUDA(cudaEventRecord(g.ev_done[b % kEv], stream));
        HEAL_CUDA(cudaStreamWaitEvent(g.copy_out, g.ev_done[b % kEv], 0));
        HEAL_CUDA(cudaMemcpy2DAsync(static_cast<char *>(C_host) + r0 * ldc * 4, ldc * 4, dC + r0 * dldc * 4, dldc * 4, N * 4, rows,
                                    cudaMemcpyDeviceToHost, g.copy_out));
    }
    HEAL_CUDA(cudaStreamSynchronize(g.copy_out));
    HEAL_CUDA(cudaStreamSynchronize(stream));
    drain.armed = false;
    return HEAL_OK;
}

}  // extern "C"
