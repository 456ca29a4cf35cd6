// bg_level.cuh -- the Berends-Giele level sweep with the splitting sums of every level
// unrolled at compile time: the fast path for the BASELINE shapes.
//
// Same mapping and shared-memory layout as bg_tile.cuh (a block owns a TILE of 32 points and
// has W warps; lane l of every warp works on point l), same algebra (factored form of the
// i-free V3, V4 of Eq.(7)).  What differs is how the sums over splittings
// of Eq.(6) are driven.  bg_tile.cuh loops over a table of single splittings
// and pays ~22 instructions of decode per splitting; here the level L is a template
// parameter, the code of ONE current of length L is straight-line (every splitting
// unrolled), and the position i of the current only enters through two base pointers:
// row(i, la) = rowbase(la) + (i-1), so every operand is [base + immediate].  What is left
// at run time is a short list of TASKS per (level, warp) in constant memory:
//
//   task = (current i, unit range [lo, hi), flags)      unit la = the 3-gluon split
//          (i..i+la-1 | i+la..j) together with its 4-gluon splits (i..i+la-1 | .. | ..j)
//
// The units of a level are cut into W chunks of equal estimated cost (make_level_program);
// a current whose units all fall to one warp is finished by it (propagator, store, U/V); one
// that straddles chunks has its partial sums parked in shared scratch and is finished by a
// gather task after a block barrier.
//
// Multiplier-pipe economy (profiles/r01b: IMAD.WIDE.U32 issues at 8 lanes/clk/SMSP, a quarter
// of the ALU rate, and is the binding pipe): every IMAD.WIDE below is a field
// multiplication of the algorithm; accumulator headroom is bought with F::relief (one
// VIADDMNMX on the upper word), whose placement is resolved at compile time.
#pragma once
#include "bg_field.cuh"
#include "bg_recursion.cuh"
#include "bg_tables.cuh"
#include "bg_tile.cuh"

namespace bg {

constexpr uint32_t LT_BAR = 1u << 16;    // block barrier before this task (first gather task of the level)
constexpr uint32_t LT_FIN = 2u << 16;    // finish the current after the units / the gather
constexpr uint32_t LT_PART = 4u << 16;   // park the partial sums in scratch slot `slot`

struct LevelTask {
    uint32_t a;       // ci | lo << 4 | hi << 8 | slot << 12 | flags      (ci = i-1)
    uint32_t mask;    // gather task: scratch slots to sum
};

// estimated cost (instructions) of the pieces, used to balance the chunks
struct LevelWeights {
    int w3, w4, wstart, wfin, wpart, wgather;
};
constexpr LevelWeights kLevelWeights = {95, 30, 50, 125, 60, 30};   // from the ncu source view, profiles/r01b

template <int N, int W>
struct LevelProgram {
    static constexpr int M = N - 1;
    static constexpr int MAXT = M * (M + 1) / 2 + 4 * W * M;
    LevelTask task[MAXT];
    uint16_t beg[M + 1][W + 1];          // tasks of warp w at level L: [beg[L][w], beg[L][w+1])
};

template <int N, int W>
constexpr LevelProgram<N, W> make_level_program(LevelWeights wt = kLevelWeights)
{
    static_assert(2 * W <= 16 && N <= 16, "slot, ci, lo, hi are 4-bit fields of a task word");
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
        // phase A tasks
        for (int w = 0; w < W; ++w) {
            const int ub = cut[w], ue = cut[w + 1];
            if (ub >= ue) continue;
            for (int ci = ub / NU; ci <= (ue - 1) / NU; ++ci) {
                const int lo = ub - ci * NU > 0 ? ub - ci * NU : 0;
                const int hi = ue - ci * NU < NU ? ue - ci * NU : NU;
                const bool complete = lo == 0 && hi == NU;
                const int slot = 2 * w + (lo > 0 ? 0 : 1);
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
                        mask |= 1u << (tmp[w][t].a >> 12 & 15u);
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
    }
    return p;
}

template <class F, int N, int D, int W>
__constant__ LevelProgram<N, W> c_level_program = make_level_program<N, W>();

// row of J(1..la) in the vector record; J(i..i+la-1) is row lv_rowbase(la) + (i-1)
template <int N>
__host__ __device__ constexpr int lv_rowbase(int la)
{
    return la == 1 ? 0 : N + tt_lvl_base(N - 1, la);
}

// One unit of the current (ci, L): the 3-gluon split with left factor J(i..i+LA-1) and the
// 4-gluon splits with the same left factor.  Entry and exit: every acc[] has room for kCapR
// more products.
template <class F, int N, int D, int W, int L, int LA>
__device__ __forceinline__ void level_unit(const typename F::E* __restrict__ ri,
                                           const typename F::E* __restrict__ si,
                                           const typename F::E (&x2)[D], typename F::A (&acc)[D],
                                           typename F::E& hsum)
{
    typedef TileCfg<F, N, D, W> C;
    typedef typename F::E E;
    constexpr int RA = lv_rowbase<N>(LA), RB = lv_rowbase<N>(L - LA) + LA;
    E a[D], b[D], s[D];
    ld_vec<F, D>(ri + RA * D, a);
    ld_vec<F, D>(ri + RB * D, b);
    ld_vec<F, D>(ri + (C::PS0 + LA) * D, s);                       // PS2_k, k = i+LA-1
    const E ua = si[(C::SC_U + RA) * 32], vb = si[(C::SC_V + RB) * 32];
    const E na0 = F::neg(a[0]);
    const E h = F::neg(F::reduce(dot_neg<F, D>(na0, a, b)));       // A.B
    const E xa = F::reduce(dot_plain<F, D>(x2, a));                // 2 X.A
    const E xb = F::reduce(dot_plain<F, D>(x2, b));                // 2 X.B
    const E cb = F::sub(xa, ua);
    const E ca = F::sub(vb, xb);
    hsum = F::add(hsum, h);
    int room = F::kCapR;
    auto need = [&](int k) {
        if (room < k) {
#pragma unroll
            for (int mu = 0; mu < D; ++mu) acc[mu] = F::relief(acc[mu]);
            room = F::kCapR;
        }
        room -= k;
    };
    need(2);
#pragma unroll
    for (int mu = 0; mu < D; ++mu) {
        acc[mu] = F::mad(h, s[mu], acc[mu]);
        acc[mu] = F::mad(cb, b[mu], acc[mu]);
    }
    need(1);
#pragma unroll
    for (int mu = 0; mu < D; ++mu) acc[mu] = F::mad(ca, a[mu], acc[mu]);
#pragma unroll
    for (int lb = 1; lb <= L - LA - 1; ++lb) {
        // (i..k | k+1..l | l+1..j), l = k+lb: 2 (A.C) J(k+1..l)
        E bm[D], c[D];
        ld_vec<F, D>(ri + (lv_rowbase<N>(lb) + LA) * D, bm);
        ld_vec<F, D>(ri + (lv_rowbase<N>(L - LA - lb) + LA + lb) * D, c);
        const E cc = F::neg(F::dbl(F::reduce(dot_neg<F, D>(na0, a, c))));
        need(1);
#pragma unroll
        for (int mu = 0; mu < D; ++mu) acc[mu] = F::mad(cc, bm[mu], acc[mu]);
    }
    if (room < F::kCapR) {
#pragma unroll
        for (int mu = 0; mu < D; ++mu) acc[mu] = F::relief(acc[mu]);
    }
}

template <class F, int N, int D, int W, int L, int LA>
struct LevelUnits {
    __device__ __forceinline__ static void run(const typename F::E* __restrict__ ri,
                                               const typename F::E* __restrict__ si, int lo, int hi,
                                               const typename F::E (&x2)[D], typename F::A (&acc)[D],
                                               typename F::E& hsum)
    {
        if (LA - 1 >= lo && LA - 1 < hi) level_unit<F, N, D, W, L, LA>(ri, si, x2, acc, hsum);
        LevelUnits<F, N, D, W, L, LA + 1>::run(ri, si, lo, hi, x2, acc, hsum);
    }
};
template <class F, int N, int D, int W, int L>
struct LevelUnits<F, N, D, W, L, L> {
    __device__ __forceinline__ static void run(const typename F::E*, const typename F::E*, int, int,
                                               const typename F::E (&)[D], typename F::A (&)[D], typename F::E&)
    {
    }
};

// All tasks of this warp at level L, then the level barrier; recurses to L+1.
template <class F, int N, int D, int W, int L>
struct LevelSweep {
    __device__ __forceinline__ static void run(typename F::E* __restrict__ rec, typename F::E* __restrict__ sc,
                                               int warp, const TileParams<typename F::E>& prm, long long pt,
                                               bool live)
    {
        typedef TileCfg<F, N, D, W> C;
        typedef typename F::E E;
        typedef typename F::A A;
        constexpr int M = N - 1;
        constexpr bool TOP = L == M;
        constexpr int OWN = lv_rowbase<N>(L);
        const LevelProgram<N, W>& tb = c_level_program<F, N, D, W>;
        const int t0 = tb.beg[L][warp], t1 = tb.beg[L][warp + 1];
#pragma unroll 1
        for (int t = t0; t < t1; ++t) {
            const uint32_t ta = tb.task[t].a;
            if (ta & LT_BAR) __syncthreads();
            if (!(ta & (LT_FIN | LT_PART))) continue;
            const int ci = ta & 15u, lo = ta >> 4 & 15u, hi = ta >> 8 & 15u;
            E* ri = rec + ci * D;
            E* si = sc + ci * 32;
            E l[D], h[D], x2[D];
            ld_vec<F, D>(ri + C::PS0 * D, l);                     // PS2_{i-1}
            ld_vec<F, D>(ri + (C::PS0 + L) * D, h);               // PS2_j
            x2[0] = F::sub(h[0], l[0]);                            // 2 * covariant P_{i,j}
#pragma unroll
            for (int mu = 1; mu < D; ++mu) x2[mu] = F::sub(l[mu], h[mu]);
            A acc[D];
#pragma unroll
            for (int mu = 0; mu < D; ++mu) acc[mu] = F::zero();
            E hsum = F::ezero();
            LevelUnits<F, N, D, W, L, 1>::run(ri, si, lo, hi, x2, acc, hsum);
            uint32_t mask = tb.task[t].mask;
            while (mask) {                                         // gather task
                const int slot = __ffs(mask) - 1;
                mask &= mask - 1;
                const E* scr = sc + (C::SC_SCR + slot * (D + 1)) * 32;
#pragma unroll
                for (int mu = 0; mu < D; ++mu) acc[mu] = F::accumulate(acc[mu], scr[mu * 32]);
                hsum = F::add(hsum, scr[D * 32]);
            }
            if (ta & LT_PART) {
                E* scr = sc + (C::SC_SCR + (ta >> 12 & 15u) * (D + 1)) * 32;
#pragma unroll
                for (int mu = 0; mu < D; ++mu) scr[mu * 32] = F::reduce(acc[mu]);
                scr[D * 32] = hsum;
                continue;
            }
            // ---- finish: boundary term of the (P-Q) sum, propagator, store, U and V ---------------
            const E nhh = F::neg(F::mul(hsum, F::half()));          // -(sum_k h_k)/2
            if constexpr (F::kExact) {
                // one product per component: the ALU adds are cheaper than a second IMAD.WIDE
                E lh[D];
#pragma unroll
                for (int mu = 0; mu < D; ++mu) lh[mu] = F::add(l[mu], h[mu]);
#pragma unroll
                for (int mu = 0; mu < D; ++mu) acc[mu] = F::mad(nhh, lh[mu], acc[mu]);
            } else {
                // floating point: same operation order as bg_tile.cuh
#pragma unroll
                for (int mu = 0; mu < D; ++mu) {
                    acc[mu] = F::mad(nhh, l[mu], acc[mu]);
                    acc[mu] = F::mad(nhh, h[mu], acc[mu]);
                }
            }
            E v[D];
            if constexpr (!TOP) {
                const E w = si[(C::SC_W + OWN - N) * 32];
#pragma unroll
                for (int mu = 0; mu < D; ++mu) v[mu] = F::mul(F::reduce(acc[mu]), w);
                st_vec<F, D>(ri + OWN * D, v);
                const E c2 = F::reduce(dot_plain<F, D>(x2, v));     // 2 P_{i,j} . J(i..j)
                si[(C::SC_U + OWN) * 32] = F::add(c2, hsum);
                si[(C::SC_V + OWN) * 32] = F::sub(c2, hsum);
            } else {
                // top current: no propagator; amplitude = eps_n . N(1..m)
#pragma unroll
                for (int mu = 0; mu < D; ++mu) v[mu] = F::reduce(acc[mu]);
                E e[D];
                ld_vec<F, D>(rec + (N - 1) * D, e);
                const A nout = dot_neg<F, D>(F::neg(e[0]), e, v);
                if (live) prm.out[pt] = F::canon(F::neg(F::reduce(nout)));
            }
            if (prm.currents && live) {
                E* dst = prm.currents + (pt * M * M + (long long)ci * M + (ci + L - 1)) * D;
#pragma unroll
                for (int mu = 0; mu < D; ++mu) dst[mu] = F::canon(v[mu]);
            }
        }
        if constexpr (!TOP) {
            __syncthreads();
            LevelSweep<F, N, D, W, L + 1>::run(rec, sc, warp, prm, pt, live);
        }
    }
};

template <class F, int N, int D, int W>
__global__ void __launch_bounds__(32 * W) bg_level_kernel(const TileParams<typename F::E> prm)
{
    typedef TileCfg<F, N, D, W> C;
    typedef typename F::E E;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    E* vec = reinterpret_cast<E*>(smem_raw);                  // [32][VSTRIDE]
    E* scal = vec + 32 * C::VSTRIDE;                          // [NSCAL][32]
    uint32_t* stat = reinterpret_cast<uint32_t*>(scal + 32 * C::NSCAL);

    const int lane = threadIdx.x & 31, warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
    const long long tile0 = (long long)blockIdx.x * 32;
    const int valid = (int)min(32LL, prm.batch - tile0);
    const long long pt = tile0 + lane;
    const bool live = lane < valid;

    tile_setup<F, N, D, W>(vec, scal, stat, prm, lane, warp, tile0, valid, pt, live);
    E* rec = vec + (size_t)lane * C::VSTRIDE;
    E* sc = scal + lane;
    LevelSweep<F, N, D, W, 2>::run(rec, sc, warp, prm, pt, live);
}

}  // namespace bg
