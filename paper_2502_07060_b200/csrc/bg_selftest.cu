// bg_selftest.cu -- host-side validation of the compile-time work schedules of the tiled kernels.
//
// The level sweep of Eq.(6) is driven by constexpr tables (bg_tables.cuh for
// bg_tile_kernel / bg_split_kernel, make_level_program in bg_level.cuh for bg_level_kernel).
// bg_selftest_schedules() rebuilds the same tables on the host and checks, for every compiled
// (n, warps) pair, that every splitting of every current is executed exactly once, that a
// current is either finished by the warp that owns all of it or has its parts gathered exactly
// once from distinct scratch slots, and that the barriers of a level are taken by every warp.
// Pure host code: callable without a GPU (tests/test_abi.py).
#include <stdint.h>

#include "../../include/bg.h"
#include "bg_level.cuh"
#include "bg_tables.cuh"

namespace {

using namespace bg;

// ---- bg_level.cuh task lists --------------------------------------------------------------------
template <int N, int W>
int check_level_program()
{
    constexpr int M = N - 1;
    static const LevelProgram<N, W> p = make_level_program<N, W>();
    int prev_end = 0;
    for (int L = 2; L <= M; ++L) {
        const int NU = L - 1, NC = M - L + 1;
        int covered[16][16] = {};          // [ci][unit] -> times executed
        int fin[16] = {}, parts[16] = {};
        uint32_t part_slots[16] = {}, gather_mask[16] = {};
        uint32_t level_slots = 0;
        int bars[W] = {};
        bool any_gather = false;
        if (p.beg[L][0] != prev_end) return -100 - L;                       // lists are contiguous
        for (int w = 0; w < W; ++w) {
            if (p.beg[L][w + 1] < p.beg[L][w]) return -200 - L;
            bool seen_bar = false;
            for (int t = p.beg[L][w]; t < p.beg[L][w + 1]; ++t) {
                const uint32_t a = p.task[t].a, mask = p.task[t].mask;
                const int ci = a & 15u, lo = a >> 4 & 15u, hi = a >> 8 & 15u, slot = a >> 12 & 15u;
                if (a & LT_BAR) { ++bars[w]; seen_bar = true; }
                if (!(a & (LT_FIN | LT_PART))) continue;
                if (ci >= NC || lo > hi || hi > NU) return -300 - L;
                for (int u = lo; u < hi; ++u) ++covered[ci][u];
                if (a & LT_PART) {
                    if (seen_bar || mask || lo == hi) return -400 - L;    // parts come before the barrier
                    if (slot >= 2 * W || (level_slots >> slot & 1u)) return -500 - L;
                    level_slots |= 1u << slot;
                    part_slots[ci] |= 1u << slot;
                    ++parts[ci];
                } else {
                    ++fin[ci];
                    if (mask) {                                             // gather task
                        if (!seen_bar || lo != hi) return -600 - L;
                        gather_mask[ci] = mask;
                        any_gather = true;
                    } else if (lo != 0 || hi != NU || seen_bar) {
                        return -700 - L;                                    // inline finish owns the whole current
                    }
                }
            }
        }
        for (int ci = 0; ci < NC; ++ci) {
            for (int u = 0; u < NU; ++u)
                if (covered[ci][u] != 1) return -800 - L;
            if (fin[ci] != 1) return -900 - L;
            if (parts[ci] == 1 || part_slots[ci] != gather_mask[ci]) return -1000 - L;
        }
        for (int w = 0; w < W; ++w)
            if (bars[w] != (any_gather ? 1 : 0)) return -1100 - L;
        prev_end = p.beg[L][W];
    }
    return 0;
}

// ---- bg_tables.cuh item lists --------------------------------------------------------------------
template <int N, int W>
int check_tile_tables()
{
    constexpr int M = N - 1;
    static const TileTables<N, W> t = make_tile_tables<N, W>();
    int base = 0;
    for (int L = 2; L <= M; ++L) {
        const int NC = M - L + 1, per = (L - 1) + (L - 1) * (L - 2) / 2, cnt = NC * per;
        if (t.beg[L][0] != base || t.beg[L][W] != base + cnt) return -100 - L;
        uint32_t level_slots = 0, part_slots[16] = {}, job_mask[16] = {};
        int njob[16] = {};
        for (int w = 0; w < W; ++w) {
            const int b = t.beg[L][w], e = t.beg[L][w + 1];
            if (e < b) return -200 - L;
            for (int q = b; q < e; ++q) {
                const int rel = q - base, cur = rel / per, pos = rel % per, i = cur + 1;
                const uint32_t x = t.items[q].x, y = t.items[q].y, fl = x >> 24;
                // which splitting is item `pos` of a current: la-major, the 3-split then its 4-splits
                int la = 1, r = pos;
                while (r >= 1 + (L - la - 1)) { r -= 1 + (L - la - 1); ++la; }
                const int lb = r;                                           // 0: the 3-gluon split
                const uint32_t want_a = (uint32_t)tt_row(N, i, la);
                const uint32_t want_b = lb == 0 ? (uint32_t)tt_row(N, i + la, L - la) : (uint32_t)tt_row(N, i + la, lb);
                const uint32_t want_c = lb == 0 ? (uint32_t)(i + la - 1) : (uint32_t)tt_row(N, i + la + lb, L - la - lb);
                if ((x & 255u) != want_a || (x >> 8 & 255u) != want_b || (x >> 16 & 255u) != want_c) return -300 - L;
                if (((fl & IT_KIND4) != 0) != (lb != 0)) return -400 - L;
                if ((y & 255u) != (uint32_t)(i - 1) || (y >> 8 & 255u) != (uint32_t)(i - 1 + L) ||
                    (y >> 16 & 255u) != (uint32_t)tt_row(N, i, L))
                    return -500 - L;
                const bool first = q == b || pos == 0, last = q == e - 1 || pos == per - 1;
                if (((fl & IT_SEG_START) != 0) != first || ((fl & IT_SEG_END) != 0) != last) return -600 - L;
                if (first && !(fl & IT_LOAD_A)) return -700 - L;
                if (last) {
                    const int seg_begin = base + cur * per > b ? base + cur * per : b;
                    const bool whole = seg_begin == base + cur * per && pos == per - 1;
                    if (((fl & IT_COMPLETE) != 0) != whole) return -800 - L;
                    if (!whole) {
                        const uint32_t slot = y >> 24;
                        if (slot >= 2u * W || (level_slots >> slot & 1u)) return -900 - L;
                        level_slots |= 1u << slot;
                        part_slots[cur] |= 1u << slot;
                    }
                }
            }
        }
        if (t.njobs[L] > W) return -1000 - L;
        for (int j = 0; j < t.njobs[L]; ++j) {
            const uint32_t y = t.jobs[L][j].y;
            const int cur = (int)(y & 255u);
            if (cur >= NC || (y >> 8 & 255u) != (uint32_t)(cur + L) || (y >> 16 & 255u) != (uint32_t)tt_row(N, cur + 1, L))
                return -1100 - L;
            job_mask[cur] = t.jobs[L][j].x;
            ++njob[cur];
        }
        for (int cur = 0; cur < NC; ++cur) {
            if (njob[cur] != (part_slots[cur] ? 1 : 0) || job_mask[cur] != part_slots[cur]) return -1200 - L;
            if (part_slots[cur] && !(part_slots[cur] & (part_slots[cur] - 1))) return -1300 - L;   // at least two parts
        }
        base += cnt;
    }
    return 0;
}

}  // namespace

extern "C" int bg_selftest_schedules(void)
{
    int rc = 0;
// every (n, warps) pair instantiated in bg_api.cu
    if ((rc = check_level_program<8, 4>())) return rc - 10000;
    if ((rc = check_level_program<8, 6>())) return rc - 20000;
    if ((rc = check_level_program<4, 1>())) return rc - 30000;
    if ((rc = check_level_program<6, 2>())) return rc - 40000;
    if ((rc = check_level_program<6, 4>())) return rc - 50000;
    if ((rc = check_level_program<10, 8>())) return rc - 60000;
    if ((rc = check_level_program<12, 8>())) return rc - 70000;
    if ((rc = check_level_program<9, 4>())) return rc - 80000;
    if ((rc = check_level_program<5, 1>())) return rc - 81000;
    if ((rc = check_level_program<7, 4>())) return rc - 82000;
    if ((rc = check_level_program<4, 1>())) return rc - 83000;
    if ((rc = check_tile_tables<8, 4>())) return rc - 110000;
    if ((rc = check_tile_tables<8, 8>())) return rc - 120000;
    if ((rc = check_tile_tables<4, 1>())) return rc - 130000;
    if ((rc = check_tile_tables<10, 8>())) return rc - 140000;
    if ((rc = check_tile_tables<12, 8>())) return rc - 150000;
    if ((rc = check_tile_tables<6, 4>())) return rc - 160000;
    if ((rc = check_tile_tables<6, 2>())) return rc - 170000;
    if ((rc = check_tile_tables<16, 8>())) return rc - 180000;
    if ((rc = check_tile_tables<12, 16>())) return rc - 190000;
    if ((rc = check_tile_tables<4, 2>())) return rc - 200000;
    if ((rc = check_tile_tables<5, 2>())) return rc - 201000;
    if ((rc = check_tile_tables<7, 4>())) return rc - 202000;
    if ((rc = check_tile_tables<9, 8>())) return rc - 203000;
    return rc;
}
