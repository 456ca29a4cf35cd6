// bg_schedule.cuh -- compile-time work schedule of the tiled Berends-Giele kernel (bg_unit.cuh).
//
// A block owns a TILE of points and has W warps; the warps split the WORK of a recursion level
// of Eq.(6).  The unit of work is
//
//   unit la of the current (i..j), length L:  the 3-gluon split (i..i+la-1 | i+la..j) together
//          with its 4-gluon splits (i..i+la-1 | .. | ..j) that share the left factor,
//
// and what is left at run time is a short list of TASKS per (level, warp) in constant memory:
//
//   task = (current ci = i-1, unit range [lo, hi), flags)
//
// The units of a level are cut into W contiguous chunks by dynamic programming over a cost model
// of the level (make_level_program); a current whose units all fall to one warp is finished by
// it (propagator, store, U/V); one that straddles chunks has its partial sums parked in shared
// scratch and is finished by a gather task after a block barrier.  Everything here is evaluated
// by the compiler (constexpr) and validated on the host by bg_selftest_schedules().
#pragma once
#include <stdint.h>

namespace bg {

__host__ __device__ constexpr int tt_lvl_base(int M, int L) { return (L - 2) * M - (L - 1) * (L - 2) / 2; }
// row of J(i..i+L-1) in the vector record: eps_1..eps_n first, then level-major (i 1-based)
__host__ __device__ constexpr int tt_row(int N, int i, int L)
{
    return L == 1 ? i - 1 : N + tt_lvl_base(N - 1, L) + i - 1;
}

constexpr uint32_t LT_BAR = 1u << 20;    // block barrier before this task (first gather task of the level)
constexpr uint32_t LT_FIN = 2u << 20;    // finish the current after the units / the gather
constexpr uint32_t LT_PART = 4u << 20;   // park the partial sums in scratch slot `slot`

struct LevelTask {
    uint32_t a;       // ci | lo << 4 | hi << 8 | slot << 12 (6 bits) | flags      (ci = i-1)
    uint32_t mask;    // gather task: scratch slots to sum
};

// estimated cost (instructions) of the pieces, used to balance the chunks
struct LevelWeights {
    int w3, w4, wstart, wfin, wpart, wgather;
};
#ifndef BG_LEVEL_WEIGHTS
#define BG_LEVEL_WEIGHTS {95, 30, 50, 125, 60, 30}   // from the ncu source view, profiles/r01b
#endif
constexpr LevelWeights kLevelWeights = BG_LEVEL_WEIGHTS;

template <int N, int W>
struct LevelProgram {
    static constexpr int M = N - 1;
    static constexpr int MAXT = M * (M + 1) / 2 + 4 * W * M;
    LevelTask task[MAXT];
    uint16_t beg[M + 1][W + 1];          // tasks of warp w at level L: [beg[L][w], beg[L][w+1])
    int nslots;                          // scratch slots in use at once (slots are numbered per level)
};

template <int N, int W>
constexpr LevelProgram<N, W> make_level_program(LevelWeights wt = kLevelWeights)
{
    static_assert(2 * W <= 32 && N <= 16, "ci, lo, hi are 4-bit fields of a task word; slots are bits of a 32-bit mask");
    LevelProgram<N, W> p{};
    constexpr int M = N - 1;
    constexpr int PER = M + W + 2;       // tasks per (level, warp) at most
    constexpr int MAXCNT = (M / 2 + 1) * (M / 2 + 1);   // >= (L-1)(M-L+1) units of any level
    int nt = 0;
    for (int L = 0; L <= M; ++L)
        for (int w = 0; w <= W; ++w) p.beg[L][w] = 0;
    for (int L = 2; L <= M; ++L) {
        const int NU = L - 1, NC = M - L + 1, cnt = NU * NC;
        // chunk boundaries in flattened unit index q = ci * NU + (la - 1): the contiguous partition
        // into W chunks with the smallest modelled level time, found by dynamic programming over
        // the cut positions (cost of a chunk = its units + start + finish or partial store of
        // every current it touches); candidates with a penalty on shared currents are compared by
        // the full model (largest chunk + largest gather load, as executed around the barrier).
        int cut[W + 1] = {};
        {
            long pre[MAXCNT + 1] = {};
            for (int q = 0; q < cnt; ++q) pre[q + 1] = pre[q] + wt.w3 + (long)(NU - 1 - q % NU) * wt.w4;
            long best_time = -1;
            for (int cand = 0; cand < 3; ++cand) {
                const long pen = cand == 0 ? 0 : cand == 1 ? 100 : 100000;    // 100000: whole currents only
                long bestv[W + 1][MAXCNT + 1] = {};
                int arg[W + 1][MAXCNT + 1] = {};
                for (int w = 0; w <= W; ++w)
                    for (int q = 0; q <= cnt; ++q) bestv[w][q] = q == 0 && w == 0 ? 0 : (long)1 << 60;
                for (int w = 1; w <= W; ++w)
                    for (int q = 0; q <= cnt; ++q)
                        for (int pp = 0; pp <= q; ++pp) {
                            long c = 0;
                            if (pp < q) {
                                c = pre[q] - pre[pp];
                                for (int ci = pp / NU; ci <= (q - 1) / NU; ++ci) {
                                    const int lo = pp - ci * NU > 0 ? pp - ci * NU : 0;
                                    const int hi = q - ci * NU < NU ? q - ci * NU : NU;
                                    c += wt.wstart + (lo == 0 && hi == NU ? wt.wfin : wt.wpart + pen);
                                }
                            }
                            const long v = bestv[w - 1][pp] > c ? bestv[w - 1][pp] : c;
                            if (v < bestv[w][q]) { bestv[w][q] = v; arg[w][q] = pp; }
                        }
                int cc[W + 1] = {};
                for (int w = W, q = cnt; w >= 1; --w) { cc[w] = q; q = arg[w][q]; }
                // full model of this candidate
                long la = 0, load[W] = {}, gl[W] = {};
                int shared[MAXCNT + 1] = {};
                for (int w = 0; w < W; ++w) {
                    const int ub = cc[w], ue = cc[w + 1];
                    if (ub >= ue) continue;
                    load[w] = pre[ue] - pre[ub];
                    for (int ci = ub / NU; ci <= (ue - 1) / NU; ++ci) {
                        const int lo = ub - ci * NU > 0 ? ub - ci * NU : 0;
                        const int hi = ue - ci * NU < NU ? ue - ci * NU : NU;
                        const bool complete = lo == 0 && hi == NU;
                        load[w] += wt.wstart + (complete ? wt.wfin : wt.wpart);
                        if (!complete) ++shared[ci];
                    }
                    if (load[w] > la) la = load[w];
                }
                long lb = 0;
                for (int ci = 0; ci < NC; ++ci)
                    if (shared[ci]) {
                        int b = 0;
                        for (int w = 1; w < W; ++w)
                            if (load[w] + gl[w] < load[b] + gl[b]) b = w;
                        gl[b] += wt.wfin + (long)shared[ci] * wt.wgather;
                        if (gl[b] > lb) lb = gl[b];
                    }
                if (best_time < 0 || la + lb < best_time) {
                    best_time = la + lb;
                    for (int w = 0; w <= W; ++w) cut[w] = cc[w];
                }
            }
        }
        LevelTask tmp[W][PER] = {};
        int ntw[W] = {};
        long load[W] = {};
        int nslot = 0;
        // phase A tasks
        for (int w = 0; w < W; ++w) {
            const int ub = cut[w], ue = cut[w + 1];
            if (ub >= ue) continue;
            for (int ci = ub / NU; ci <= (ue - 1) / NU; ++ci) {
                const int lo = ub - ci * NU > 0 ? ub - ci * NU : 0;
                const int hi = ue - ci * NU < NU ? ue - ci * NU : NU;
                const bool complete = lo == 0 && hi == NU;
                const int slot = complete ? 0 : nslot++;
                tmp[w][ntw[w]].a = (uint32_t)ci | (uint32_t)lo << 4 | (uint32_t)hi << 8 |
                                   (complete ? LT_FIN : ((uint32_t)slot << 12 | LT_PART));
                tmp[w][ntw[w]].mask = 0;
                ++ntw[w];
                for (int u = lo; u < hi; ++u) load[w] += wt.w3 + (long)(NU - 1 - u) * wt.w4;
                load[w] += wt.wstart + (complete ? wt.wfin : wt.wpart);
            }
        }
        // gather tasks: one per current shared between warps, given to the least loaded warp
        int nb[W] = {};
        int njobs = 0;
        for (int ci = 0; ci < NC; ++ci) {
            uint32_t mask = 0;
            int parts = 0;
            for (int w = 0; w < W; ++w)
                for (int t = 0; t < ntw[w]; ++t)
                    if ((tmp[w][t].a & LT_PART) && (int)(tmp[w][t].a & 15u) == ci) {
                        mask |= 1u << (tmp[w][t].a >> 12 & 63u);
                        ++parts;
                    }
            if (!parts) continue;
            int best = 0;
            for (int w = 1; w < W; ++w)
                if (load[w] < load[best]) best = w;
            LevelTask& g = tmp[best][ntw[best] + nb[best]];
            g.a = (uint32_t)ci | LT_FIN | (nb[best] == 0 ? LT_BAR : 0u);
            g.mask = mask;
            ++nb[best];
            load[best] += wt.wfin + (long)parts * wt.wgather;
            ++njobs;
        }
        for (int w = 0; w < W; ++w) {
            if (njobs && nb[w] == 0) {            // every warp takes part in the barrier
                tmp[w][ntw[w]].a = LT_BAR;
                tmp[w][ntw[w]].mask = 0;
                nb[w] = 1;
            }
            p.beg[L][w] = (uint16_t)nt;
            for (int t = 0; t < ntw[w] + nb[w]; ++t) p.task[nt++] = tmp[w][t];
        }
        p.beg[L][W] = (uint16_t)nt;
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
