// bg_selftest.cu -- host-side validation of the compile-time work schedules of the tiled kernels.
//
// The level sweep of Eq.(6) is driven by constexpr task lists (make_level_program in
// bg_schedule.cuh).  bg_selftest_schedules() rebuilds the same lists on the host and checks, for every compiled
// (n, warps) pair, that every splitting of every current is executed exactly once; that a current is either
// finished by the warp that owns all of it, or by the owner of its first units as the LAST task of that warp,
// with every other part the FIRST task of another warp, parked in a scratch slot of its own that the finisher
// adds exactly once; and that finisher and parts agree on the named barrier and on the number of warps that
// meet there (a mismatch would hang the block).
// Pure host code: callable without a GPU (tests/test_abi.py).
#include <stdint.h>

#include <string.h>

#include "../../include/bg.h"
#include "bg_rt_host.h"
#include "bg_schedule.cuh"
#include "bg_unit.cuh"

namespace {

using namespace bg;

template <int N, int W>
int check_level_program()
{
    constexpr int M = N - 1;
    static const LevelProgram<N, W> p = make_level_program<N, W>();
    int prev_end = 0;
    for (int L = 2; L <= M; ++L) {
        const int NU = L - 1, NC = M - L + 1;
        int covered[16][16] = {};          // [ci][unit] -> times executed
        int fin[16] = {}, parts[16] = {}, fin_bar[16] = {}, fin_nwarps[16] = {}, part_bar_ok[16] = {};
        uint32_t part_slots[16] = {}, fin_mask[16] = {};
        uint32_t level_slots = 0, level_bars = 0;
        if (p.beg[L][0] != prev_end) return -100 - L;                       // lists are contiguous
        for (int w = 0; w < W; ++w) {
            if (p.beg[L][w + 1] < p.beg[L][w]) return -200 - L;
            for (int t = p.beg[L][w]; t < p.beg[L][w + 1]; ++t) {
                const LevelTask& k = p.task[t];
                const uint32_t a = k.a;
                const int ci = a & 15u, lo = a >> 4 & 15u, hi = a >> 8 & 15u, slot = a >> 12 & 63u;
                const bool first = t == p.beg[L][w], last = t + 1 == p.beg[L][w + 1];
                if (!(a & (LT_FIN | LT_PART)) || ((a & LT_FIN) && (a & LT_PART))) return -250 - L;
                if (ci >= NC || lo >= hi || hi > NU) return -300 - L;
                for (int u = lo; u < hi; ++u) ++covered[ci][u];
                if (a & LT_PART) {
                    if (lo == 0 || !first || k.mask) return -400 - L;     // later parts are first tasks
                    if (slot >= p.nslots || (level_slots >> slot & 1u)) return -500 - L;
                    level_slots |= 1u << slot;
                    part_slots[ci] |= 1u << slot;
                    ++parts[ci];
                    if (fin[ci] != 1 || k.bar != fin_bar[ci] || k.nwarps != fin_nwarps[ci]) return -550 - L;
                    ++part_bar_ok[ci];
                } else {
                    ++fin[ci];
                    if (lo != 0) return -600 - L;
                    if (hi < NU) {                                          // finisher of a shared current
                        if (!last || !k.mask || k.bar < 1 || k.bar > 15 || (level_bars >> k.bar & 1u)) return -650 - L;
                        level_bars |= 1u << k.bar;
                        fin_mask[ci] = k.mask;
                        fin_bar[ci] = k.bar;
                        fin_nwarps[ci] = k.nwarps;
                    } else if (k.mask || k.bar || k.nwarps) {
                        return -700 - L;
                    }
                }
            }
        }
        for (int ci = 0; ci < NC; ++ci) {
            for (int u = 0; u < NU; ++u)
                if (covered[ci][u] != 1) return -800 - L;
            if (fin[ci] != 1) return -900 - L;
            if (part_slots[ci] != fin_mask[ci]) return -1000 - L;
            if (parts[ci] && fin_nwarps[ci] != parts[ci] + 1) return -1100 - L;
            if (parts[ci] > W - 1) return -1200 - L;
        }
        prev_end = p.beg[L][W];
    }
    return 0;
}

// the schedule the host builds at run time for bg_rt_kernel (bg_rt_host.cu) against the one the compiler evaluated
// for the compiled instance of the same shape: same ops, same 4-gluon-split table, same warp bounds, same layout
template <class F, int N, int D, int W, int S>
int check_rt_tables()
{
    typedef TileCfg<F, N, D, W, S, false> C;
    static const FlatProgram<N, W> fp = make_flat_program<F, N, D, W, S>();
    static RtHost h;
    if (!bg_rt_make((int)sizeof(typename F::E), C::U, N, D, S, false, &h)) return -1;
    if (h.lay.n != N || h.lay.ps0 != C::PS0 || h.lay.vstride != C::VSTRIDE || h.lay.sc_v != C::SC_V ||
        h.lay.sc_w != C::SC_W || h.lay.sc_scr != C::SC_SCR || h.lay.nscal != C::NSCAL || h.lay.nslots != C::NSLOTS ||
        h.smem != C::SMEM_BYTES || h.threads != 32 * W || h.points_per_block != C::TP)
        return -2;
    if (memcmp(h.tab.ops, fp.op, sizeof(fp.op)) != 0) return -3;
    if (FlatProgram<N, W>::NQUAD > 0 && memcmp(h.tab.quad, fp.quad, sizeof(uint32_t) * FlatProgram<N, W>::NQUAD) != 0) return -4;
    if (memcmp(h.tab.beg, fp.beg, sizeof(fp.beg)) != 0) return -5;
    // the layout of the MULTI instantiation (propagator table of its own) against TileCfg's KW layout
    typedef TileCfg<F, N, D, W, S, true> CK;
    static RtHost hk;
    if (!bg_rt_make((int)sizeof(typename F::E), CK::U, N, D, S, true, &hk)) return -6;
    if (hk.lay.ps0 != CK::PS0 || hk.lay.vstride != CK::VSTRIDE || hk.lay.sc_v != CK::SC_V || hk.lay.sc_w != CK::SC_W ||
        hk.lay.sc_scr != CK::SC_SCR || hk.lay.nscal != CK::NSCAL || hk.lay.nslots != CK::NSLOTS || hk.smem != CK::SMEM_BYTES)
        return -7;
    if (memcmp(&hk.tab, &h.tab, sizeof(h.tab)) != 0) return -8;       // same program: the ops do not name the W table
    return 0;
}

}  // namespace

extern "C" int bg_selftest_schedules(void)
{
    int rc = 0;
// every (n, warps) pair instantiated in the bg_inst_*.cu tables (and n = 16 as the largest legal n)
    if ((rc = check_level_program<8, 4>())) return rc - 10000;
    if ((rc = check_level_program<8, 6>())) return rc - 20000;
    if ((rc = check_level_program<8, 2>())) return rc - 30000;
    if ((rc = check_level_program<4, 1>())) return rc - 40000;
    if ((rc = check_level_program<4, 2>())) return rc - 50000;
    if ((rc = check_level_program<5, 1>())) return rc - 60000;
    if ((rc = check_level_program<5, 2>())) return rc - 70000;
    if ((rc = check_level_program<6, 2>())) return rc - 80000;
    if ((rc = check_level_program<6, 4>())) return rc - 90000;
    if ((rc = check_level_program<7, 4>())) return rc - 100000;
    if ((rc = check_level_program<9, 4>())) return rc - 110000;
    if ((rc = check_level_program<9, 8>())) return rc - 120000;
    if ((rc = check_level_program<10, 8>())) return rc - 130000;
    if ((rc = check_level_program<10, 4>())) return rc - 140000;
    if ((rc = check_level_program<12, 8>())) return rc - 150000;
    if ((rc = check_level_program<12, 16>())) return rc - 160000;
    if ((rc = check_level_program<12, 4>())) return rc - 170000;
    if ((rc = check_level_program<16, 8>())) return rc - 180000;
    if ((rc = check_level_program<11, 8>())) return rc - 190000;
    if ((rc = check_level_program<12, 12>())) return rc - 200000;
    if ((rc = check_level_program<8, 3>())) return rc - 210000;
    if ((rc = check_level_program<16, 16>())) return rc - 220000;
    if ((rc = check_level_program<10, 6>())) return rc - 230000;
    // bg_rt_make picks 4 warps per tile for n <= 8 and 8 above (bg_rt_warps): shapes whose compiled instance agrees
    if ((rc = check_rt_tables<bg::Fp31, 8, 6, 4, 1>())) return rc - 300000;
    if ((rc = check_rt_tables<bg::Fp31, 10, 8, 8, 1>())) return rc - 310000;
    if ((rc = check_rt_tables<bg::Fp31, 12, 6, 8, 1>())) return rc - 320000;
    if ((rc = check_rt_tables<bg::C128, 9, 6, 8, 2>())) return rc - 330000;
    return rc;
}
