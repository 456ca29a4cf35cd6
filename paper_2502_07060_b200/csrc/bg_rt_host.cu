// bg_rt_host.cu -- builds the schedule of bg_rt_kernel at run time: the same make_level_program / flat_build that
// the compiler evaluates for the kernels with a compile-time n (bg_schedule.cuh, bg_unit.cuh), called as ordinary
// host functions.
#include "bg_rt_host.h"

#include <string.h>

#include "bg_entries.h"
#include "bg_unit.cuh"

namespace {

template <int N, int W>
bool make_for(int eb, int u, int d, int s, bool multi, RtHost* out)
{
    constexpr int M = N - 1, R = M * (M - 1) / 2 - 1;
    const bg::LevelProgram<N, W> p = bg::make_level_program<N, W>();
    const int tp = 32 / s;
    bg::RtLayout& L = out->lay;
    L.n = N; L.m = M; L.r = R;
    const int j_rows = N + R;
    L.ps0 = j_rows;
    const int vec_units = (j_rows + M + 1) * d / u;            // odd number of vector units: conflict-free lanes
    L.vstride = (vec_units % 2 == 1 ? vec_units : vec_units + 1) * u;
    L.sc_v = j_rows;
    L.sc_w = multi ? j_rows + R : N;                           // 1/P^2: a table of its own, or parked in the U slots of
    L.sc_scr = j_rows + R + (multi ? R : 0);                   // the multi-gluon rows (as TileCfg's KW, bg_tile.cuh)
    L.nslots = p.nslots;
    L.nscal = L.sc_scr + L.nslots * (d + 1);
    out->s = s;
    out->threads = 32 * W;
    out->points_per_block = tp;
    out->smem = (size_t)tp * (L.vstride + L.nscal) * eb + (size_t)(tp + 32 * L.nslots) * sizeof(uint32_t);
    static_assert(W + 1 <= 16, "RtTables::beg");
    memset(&out->tab, 0, sizeof(out->tab));
    if (bg::flat_count<N, W>(p) > bg::kRtMaxOps || bg::flat_count_quads(N) > bg::kRtMaxQuad || R > bg::kRtMaxRanges)
        return false;
    bg::flat_build<N, W>(p, bg::FlatLayout{d, eb, tp, L.ps0, 0, L.sc_v}, out->tab.ops, out->tab.quad, out->tab.beg);
    int r = 0;
    for (int len = 2; len <= N - 2; ++len)
        for (int i = 0; i + len <= N - 1; ++i) out->tab.ranges[r++] = (uint16_t)(i | (i + len) << 8);
    return true;
}

}  // namespace

bool bg_rt_make(int eb, int u, int n, int d, int s, bool multi, RtHost* out)
{
    if (d % s != 0 || (long)(n + (n - 1) * (n - 2) / 2 + n) * d * eb >= 65536) return false;   // 16-bit row offsets
    switch (n) {
#define BG_CASE(N) case N: return make_for<N, (N <= 8 ? 4 : 8)>(eb, u, d, s, multi, out);   // bg_rt_warps(n)
        BG_CASE(4) BG_CASE(5) BG_CASE(6) BG_CASE(7) BG_CASE(8) BG_CASE(9) BG_CASE(10)
        BG_CASE(11) BG_CASE(12) BG_CASE(13) BG_CASE(14) BG_CASE(15) BG_CASE(16)
#undef BG_CASE
    }
    return false;
}
