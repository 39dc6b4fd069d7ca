// heal_sched.h -- work distribution of the large-M GEMM kernels: plain C++ (no CUDA types), shared by the kernels and by
// the CPU test that checks it (tests/sched_check.cpp: every (tile, K segment) unit is covered exactly once, hand-offs
// form chains in ascending CTA order).  Host logic only -- none of the method's arithmetic lives here.
#pragma once
#if defined(__CUDACC__)
#define HEAL_HD __host__ __device__ __forceinline__
#else
#define HEAL_HD inline
#endif

namespace heal {

// Tile index -> (row tile, column tile).  Tiles are numbered in groups of kGroupM row tiles: inside a group the row tile runs fastest,
// then the column tile; a group is finished before the next one starts.  A wave of consecutive tiles therefore covers a roughly square
// patch (about 8 row tiles x G/8 column tiles), so per k-step the wave reads few distinct activation AND weight slabs and they stay
// shared in L2 -- with plain row-fastest numbering every wave of a tall problem (8192^3: 32 row tiles) re-read all of A from HBM.
// With at most kGroupM row tiles (all the LLM shapes at M <= 2048) this IS the row-fastest order.  Scheduling only: no bits change.
constexpr int kGroupM = 8;
HEAL_HD void tile_coords(int tile, int tiles_m, int tiles_n, int &tm, int &tn, int group_m = kGroupM)
{
    const int per_group = group_m * tiles_n;
    const int g = tile / per_group;
    const int first_m = g * group_m;
    const int gm = (tiles_m - first_m < group_m) ? tiles_m - first_m : group_m;
    const int r = tile - g * per_group;
    tm = first_m + r % gm;
    tn = r / gm;
}

// Work distribution.  The unit of work is (tile, K segment).  The first `dp_tiles` tiles (a multiple of
// gridDim.x) are dealt round-robin, whole tiles, so the CTAs of a wave walk K in lockstep and share W / A
// panels in L2.  With `balance`, the remaining tiles (the ragged last wave) are cut at segment granularity
// into gridDim.x contiguous, equal ranges, so a tile may be shared by neighbouring CTAs: CTA c computes
// the first segments of a tile and hands the FP32 running sum to CTA c+1, which adds the following ones --
// the same ascending-segment sum, copied, never re-associated, so the result is bit-identical to the
// unbalanced schedule.  Within its range a CTA processes its "head" (the part it hands on) first and its
// "tail" (the part that needs a neighbour's prefix) last, so the prefix is almost never waited for.
struct TileSched {
    int n_seg, n_dp, n_sk, dp_tiles;
    int t_first, t_last, s_first, s_last_end, has_head, has_tail;
    int n_chunks, bid, G;
    // bid / G_: index of this CTA (or CTA pair) and number of CTAs (pairs) sharing the work
    HEAL_HD void init(int num_tiles, int balance, int dp_tiles_, int n_seg_, int bid_, int G_)
    {
        n_seg = n_seg_;
        bid = bid_;
        G = G_;
        dp_tiles = balance ? dp_tiles_ : num_tiles;
        n_dp = (dp_tiles > bid) ? (dp_tiles - 1 - bid) / G + 1 : 0;
        n_sk = 0;
        has_head = has_tail = 0;
        t_first = t_last = s_first = s_last_end = 0;
        if (balance) {
            const long long total = static_cast<long long>(num_tiles - dp_tiles) * n_seg;
            const long long u0 = total * bid / G, u1 = total * (bid + 1) / G;
            if (u1 > u0) {
                t_first = static_cast<int>(u0 / n_seg);
                s_first = static_cast<int>(u0 % n_seg);
                t_last = static_cast<int>((u1 - 1) / n_seg);
                s_last_end = static_cast<int>((u1 - 1) % n_seg) + 1;
                n_sk = t_last - t_first + 1;
                if (n_sk > 1) {
                    has_head = (s_last_end < n_seg) ? 1 : 0;
                    has_tail = (s_first > 0) ? 1 : 0;
                }
            }
        }
        n_chunks = n_dp + n_sk;
    }
    // i-th chunk in processing order: tile index and its segment range [sb, se)
    HEAL_HD void get(int i, int &tile, int &sb, int &se) const
    {
        if (i < n_dp) {
            tile = bid + i * G;
            sb = 0;
            se = n_seg;
            return;
        }
        i -= n_dp;
        if (n_sk == 1) {                       // one (possibly partial, possibly interior) piece of a tile
            tile = dp_tiles + t_first;
            sb = s_first;
            se = s_last_end;
        } else if (has_head && i == 0) {
            tile = dp_tiles + t_last;
            sb = 0;
            se = s_last_end;
        } else if (has_tail && i == n_sk - 1) {
            tile = dp_tiles + t_first;
            sb = s_first;
            se = n_seg;
        } else {
            tile = dp_tiles + t_first + has_tail + (i - has_head);
            sb = 0;
            se = n_seg;
        }
    }
};

}  // namespace heal
