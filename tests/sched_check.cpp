// Test helper (CPU, g++): the work distribution of the large-M GEMM kernels (paper_2606_21023_b200/csrc/heal_sched.h).
// For many (tiles, n_seg, G, balance, dp_tiles) it checks that
//   * every (tile, K segment) unit is computed exactly once;
//   * a CTA's pieces of a tile are contiguous segment ranges; a tile's pieces, in ascending CTA order, are consecutive
//     ranges starting at segment 0 (so the FP32 running sum can be handed from CTA c to CTA c + 1 / parked partials
//     are complete);
//   * in the chained schedule a CTA processes the piece it hands on before the piece that needs a prefix.
// Prints "checked <n> configurations, 0 failures".
#include <cstdio>
#include <vector>

#include "../paper_2606_21023_b200/csrc/heal_sched.h"

static int check(int tiles, int n_seg, int G, int balance, int dp_tiles)
{
    std::vector<int> cover(static_cast<size_t>(tiles) * n_seg, 0);
    std::vector<int> next_seg(tiles, 0), last_cta(tiles, -1);
    for (int c = 0; c < G; ++c) {
        heal::TileSched s;
        s.init(tiles, balance, dp_tiles, n_seg, c, G);
        int seen_tail = 0;
        for (int i = 0; i < s.n_chunks; ++i) {
            int tile, sb, se;
            s.get(i, tile, sb, se);
            if (tile < 0 || tile >= tiles || sb < 0 || se > n_seg || sb >= se) return 1;
            for (int k = sb; k < se; ++k) cover[static_cast<size_t>(tile) * n_seg + k]++;
            if (sb > 0) seen_tail = 1;                       // needs a prefix from an earlier CTA
            if (se < n_seg && seen_tail && sb == 0) return 2; // a piece that is handed on must come before the tail piece
        }
    }
    for (int v : cover)
        if (v != 1) return 3;
    // pieces of a tile in ascending CTA order are consecutive ranges from segment 0
    for (int c = 0; c < G; ++c) {
        heal::TileSched s;
        s.init(tiles, balance, dp_tiles, n_seg, c, G);
        // collect this CTA's pieces sorted by tile (at most one piece per tile per CTA)
        for (int i = 0; i < s.n_chunks; ++i) {
            int tile, sb, se;
            s.get(i, tile, sb, se);
            if (last_cta[tile] == c) return 4;               // two pieces of one tile in one CTA
            if (sb != next_seg[tile]) {
                // pieces of other CTAs may not have been visited yet only if they belong to a LOWER CTA index: error
                return 5;
            }
            next_seg[tile] = se;
            last_cta[tile] = c;
        }
    }
    for (int t = 0; t < tiles; ++t)
        if (next_seg[t] != n_seg) return 6;
    return 0;
}

// tile_coords is a bijection tile <-> (row tile, column tile)
static int check_coords(int tiles_m, int tiles_n)
{
    std::vector<int> seen(static_cast<size_t>(tiles_m) * tiles_n, 0);
    for (int t = 0; t < tiles_m * tiles_n; ++t) {
        int tm = -1, tn = -1;
        heal::tile_coords(t, tiles_m, tiles_n, tm, tn);
        if (tm < 0 || tm >= tiles_m || tn < 0 || tn >= tiles_n) return 1;
        if (seen[static_cast<size_t>(tm) * tiles_n + tn]++) return 2;
    }
    return 0;
}

int main()
{
    long n = 0, bad = 0;
    for (int tm = 1; tm <= 40; ++tm)
        for (int tn = 1; tn <= 70; tn += (tn < 10 ? 1 : 7)) {
            ++n;
            if (check_coords(tm, tn)) { ++bad; std::printf("coords FAIL tiles_m %d tiles_n %d\n", tm, tn); }
        }
    const int Gs[] = {1, 2, 3, 7, 74, 148};
    for (int G : Gs)
        for (int tiles = 1; tiles <= 700; tiles += (tiles < 40 ? 1 : 37))
            for (int n_seg = 1; n_seg <= 29; n_seg += (n_seg < 9 ? 1 : 5)) {
                // plain
                int r = check(tiles, n_seg, tiles < G ? tiles : G, 0, tiles);
                ++n; if (r) { ++bad; std::printf("plain tiles %d n_seg %d G %d -> %d\n", tiles, n_seg, G, r); }
                if (tiles >= G && tiles % G != 0) {           // ragged last wave, cut at segment granularity (set_balance)
                    const int waves = tiles / G, rem = tiles % G;
                    int sk = rem;
                    if (rem * 2 < G && waves >= 1) sk += G;
                    r = check(tiles, n_seg, G, 1, tiles - sk);
                    ++n; if (r) { ++bad; std::printf("balanced tiles %d n_seg %d G %d -> %d\n", tiles, n_seg, G, r); }
                }
                if (tiles < G && n_seg > 1) {                 // ordered split-K: all tiles cut, up to tiles * n_seg CTAs
                    const long units = static_cast<long>(tiles) * n_seg;
                    const int g = units < G ? static_cast<int>(units) : G;
                    r = check(tiles, n_seg, g, 1, 0);
                    ++n; if (r) { ++bad; std::printf("split-K tiles %d n_seg %d G %d -> %d\n", tiles, n_seg, g, r); }
                }
            }
    std::printf("checked %ld configurations, %ld failures\n", n, bad);
    return bad != 0;
}
