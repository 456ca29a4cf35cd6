// bg_schedule.cuh -- compile-time work schedule of the tiled Berends-Giele kernel (bg_unit.cuh).
//
// A block owns a TILE of points and has W warps; the warps split the WORK of a recursion level
// of Eq.(6).  The unit of work is
//
//   unit la of the current (i..j), length L:  the 3-gluon split (i..i+la-1 | i+la..j) together
//          with its 4-gluon splits (i..i+la-1 | .. | ..j) that share the left factor,
//
// and what is left at run time is a short list of TASKS per (level, warp):
//
//   task = (current ci = i-1, unit range [lo, hi), flags)
//
// The units of a level, in the order (current, unit), are cut into W contiguous chunks so that the
// largest modelled chunk cost is smallest (dynamic programming, make_level_program).  A current whose
// units all fall to one warp is finished by it (propagator, store, U/V).  One that straddles chunks is
// finished by the warp that owns its FIRST units -- the last task of that warp at the level: the owners of
// the other parts park their partial sums in shared scratch and raise a per-lane flag, the finisher checks
// the flags, adds the parked sums to its own registers and finishes.  The other parts are first tasks of
// their warps, so the finisher practically never waits, there is no separate gather phase, and the only
// block-wide barrier of a level is the one at its end.  (Round 2 ran the gathers as a second phase behind a
// block barrier: modelled efficiency 0.74 at n = 8 with 4 warps.  Named hardware barriers -- bar.arrive /
// bar.sync with a thread count -- do the same job but make ptxas drop the uniform datapath for the whole
// sweep: 0.93 -> 1.09 ms at cfg2.)
// Everything here is evaluated by the compiler (constexpr) and validated on the host by
// bg_selftest_schedules().
#pragma once
#include <stdint.h>

namespace bg {

__host__ __device__ constexpr int tt_lvl_base(int M, int L) { return (L - 2) * M - (L - 1) * (L - 2) / 2; }
// row of J(i..i+L-1) in the vector record: eps_1..eps_n first, then level-major (i 1-based)
__host__ __device__ constexpr int tt_row(int N, int i, int L)
{
    return L == 1 ? i - 1 : N + tt_lvl_base(N - 1, L) + i - 1;
}

constexpr uint32_t LT_FIN = 2u << 20;    // finish the current after the units (and the gather, if mask != 0)
constexpr uint32_t LT_PART = 4u << 20;   // park the partial sums in scratch slot `slot`, raise its flag

struct LevelTask {
    uint32_t a;       // ci | lo << 4 | hi << 8 | slot << 12 (6 bits) | flags      (ci = i-1)
    uint32_t mask;    // finisher of a shared current: scratch slots to add
    uint8_t bar;      // shared current: its number within the level (1..W-1)
    uint8_t nwarps;   // ... and the warps taking part (parts + finisher)
};

// estimated cost (instructions) of the pieces, used to balance the chunks
struct LevelWeights {
    int w3, w4, wstart, wfin, wpart, wgather;
};
#ifndef BG_LEVEL_WEIGHTS
#define BG_LEVEL_WEIGHTS {95, 36, 80, 130, 200, 35}   // instruction counts of the pieces; start and park set by measurement (cfg2, cfg3)
#endif
constexpr LevelWeights kLevelWeights = BG_LEVEL_WEIGHTS;

template <int N, int W>
struct LevelProgram {
    static constexpr int M = N - 1;
    static constexpr int MAXT = M * (M + 1) / 2 + 2 * W * M;
    LevelTask task[MAXT];
    uint16_t beg[M + 1][W + 1];          // tasks of warp w at level L: [beg[L][w], beg[L][w+1])
    int nslots;                          // scratch slots in use at once (slots are numbered per level)
};

template <int N, int W>
constexpr LevelProgram<N, W> make_level_program(LevelWeights wt = kLevelWeights)
{
    static_assert(W <= 16 && N <= 16, "ci, lo, hi are 4-bit fields of a task word; slots are mask bits");
    LevelProgram<N, W> p{};
    constexpr int M = N - 1;
    constexpr int MAXCNT = (M / 2 + 1) * (M / 2 + 1);   // >= (L-1)(M-L+1) units of any level
    int nt = 0;
    for (int L = 0; L <= M; ++L)
        for (int w = 0; w <= W; ++w) p.beg[L][w] = 0;
    for (int L = 2; L <= M; ++L) {
        const int NU = L - 1, NC = M - L + 1, cnt = NU * NC;
        // cost of the chunk [pp, q) of the flattened units q = ci * NU + (la - 1): its units, a start per
        // current it touches, and per current the finish (whole current, or its first part: then also a gather)
        // or the parking of a later part
        long pre[MAXCNT + 1] = {};
        for (int q = 0; q < cnt; ++q) pre[q + 1] = pre[q] + wt.w3 + (long)(NU - 1 - q % NU) * wt.w4;
        long bestv[W + 1][MAXCNT + 1] = {};
        int arg[W + 1][MAXCNT + 1] = {};
        for (int w = 0; w <= W; ++w)
            for (int q = 0; q <= cnt; ++q) bestv[w][q] = q == 0 && w == 0 ? 0 : (long)1 << 60;
        for (int w = 1; w <= W; ++w)
            for (int q = 0; q <= cnt; ++q)
                for (int pp = 0; pp <= q; ++pp) {
                    if (bestv[w - 1][pp] >= bestv[w][q]) continue;
                    long c = 0;
                    if (pp < q) {
                        c = pre[q] - pre[pp];
                        for (int ci = pp / NU; ci <= (q - 1) / NU; ++ci) {
                            const int lo = pp - ci * NU > 0 ? pp - ci * NU : 0;
                            const int hi = q - ci * NU < NU ? q - ci * NU : NU;
                            c += wt.wstart + (lo > 0 ? wt.wpart : hi == NU ? wt.wfin : wt.wfin + wt.wgather);
                        }
                    }
                    const long v = bestv[w - 1][pp] > c ? bestv[w - 1][pp] : c;
                    if (v < bestv[w][q]) { bestv[w][q] = v; arg[w][q] = pp; }
                }
        int cut[W + 1] = {};
        for (int w = W, q = cnt; w >= 1; --w) { cut[w] = q; q = arg[w][q]; }
        // tasks; the parts of a shared current are consecutive in warp order, finisher first
        int nslot = 0, nbar = 0;
        int fin_task[16] = {};               // per current: task index of its finisher (shared currents)
        for (int ci = 0; ci < 16; ++ci) fin_task[ci] = -1;
        for (int w = 0; w < W; ++w) {
            p.beg[L][w] = (uint16_t)nt;
            const int ub = cut[w], ue = cut[w + 1];
            if (ub >= ue) continue;
            for (int ci = ub / NU; ci <= (ue - 1) / NU; ++ci) {
                const int lo = ub - ci * NU > 0 ? ub - ci * NU : 0;
                const int hi = ue - ci * NU < NU ? ue - ci * NU : NU;
                LevelTask& t = p.task[nt];
                t.mask = 0;
                t.bar = 0;
                t.nwarps = 0;
                if (lo == 0) {
                    t.a = (uint32_t)ci | (uint32_t)lo << 4 | (uint32_t)hi << 8 | LT_FIN;
                    if (hi < NU) {                            // finisher of a shared current
                        fin_task[ci] = nt;
                        t.bar = (uint8_t)++nbar;
                        t.nwarps = 1;
                    }
                } else {
                    const int slot = nslot++;
                    t.a = (uint32_t)ci | (uint32_t)lo << 4 | (uint32_t)hi << 8 | (uint32_t)slot << 12 | LT_PART;
                    LevelTask& f = p.task[fin_task[ci]];
                    f.mask |= 1u << slot;
                    ++f.nwarps;
                    t.bar = f.bar;
                }
                ++nt;
            }
        }
        p.beg[L][W] = (uint16_t)nt;
        // every part knows how many warps meet at its barrier
        for (int t = p.beg[L][0]; t < nt; ++t)
            if (p.task[t].a & LT_PART) p.task[t].nwarps = p.task[fin_task[p.task[t].a & 15u]].nwarps;
        if (nslot > p.nslots) p.nslots = nslot;
    }
    return p;
}

// the schedule of (n, warps), evaluated once per instantiation
template <int N, int W>
struct LevelProgramOf {
    static constexpr LevelProgram<N, W> value = make_level_program<N, W>();
};

// row of J(1..la) in the vector record; J(i..i+la-1) is row lv_rowbase(la) + (i-1)
template <int N>
__host__ __device__ constexpr int lv_rowbase(int la)
{
    return la == 1 ? 0 : N + tt_lvl_base(N - 1, la);
}

}  // namespace bg
