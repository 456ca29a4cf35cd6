// bg_unit.cuh -- the tiled Berends-Giele kernel: SURVEY.md 8(a) rows a0-a6 in ONE launch, for
// compile-time (n, d), any field policy, either metric, 1 or 2 lanes per point, and any number
// of state configurations per momentum point.
//
// The level sweep of Eq.(6) is driven per UNIT: a unit = the 3-gluon split
// (i..i+la-1 | i+la..j) together with its c4 = L-la-1 4-gluon splits with the same left factor.
// Its code depends on (L, la) only through c4 and through operand offsets, so there is ONE
// unrolled body per c4, and the offsets of a unit come from a small constexpr table in constant
// memory (warp-uniform loads, [register + uniform register] addressing).  Levels, tasks and units
// are run-time loops; the whole kernel is a few thousand instructions for any n.  Task lists
// (which warp does which units of which current, partial sums, gather tasks, barriers):
// bg_schedule.cuh.  Layout and setup stages: bg_tile.cuh.  Algebra: bg_common.cuh.
#pragma once
#include "bg_common.cuh"
#include "bg_schedule.cuh"
#include "bg_tile.cuh"

namespace bg {

template <class F, int N, int D, int W>
__constant__ LevelProgram<N, W> c_level_program = make_level_program<N, W>();

// BYTE offsets of the operands of unit (L, la), relative to the current's base pointers
// ri = rec + ci*D (vector rows) and si = sc + ci*TP (scalar tables): ready for [register + uniform
// register + immediate] addressing, no per-lane address arithmetic
template <int N>
struct UnitOff {
    static constexpr int MAXC4 = N - 3;                        // c4 = L-la-1 <= M-2
    uint32_t u, v, w;                                          // scalar tables (w: 1/P^2 of the level's currents)
    uint16_t a, b, ps;
    uint16_t own;                                              // per level (same for every la): row of J(i..j)
    uint16_t bm[MAXC4 > 0 ? MAXC4 : 1], c[MAXC4 > 0 ? MAXC4 : 1];
};

template <int N>
struct UnitTable {
    // units packed level-major: (L, la), 2 <= L <= N-1, 1 <= la <= L-1, at index (L-1)(L-2)/2 + la-1
    UnitOff<N> u[(N - 1) * (N - 2) / 2];
    __host__ __device__ static constexpr int index(int L, int la) { return (L - 1) * (L - 2) / 2 + la - 1; }
};

template <class F, int N, int D, int W, int S>
constexpr UnitTable<N> make_unit_table()
{
    typedef TileCfg<F, N, D, W, S> C;
    UnitTable<N> t{};
    constexpr int M = N - 1;
    constexpr int EB = (int)sizeof(typename F::E), TP = C::TP;
    for (int L = 2; L <= M; ++L)
        for (int la = 1; la <= L - 1; ++la) {
            UnitOff<N>& o = t.u[UnitTable<N>::index(L, la)];
            const int ra = lv_rowbase<N>(la), rb = lv_rowbase<N>(L - la) + la;
            o.a = (uint16_t)(ra * D * EB);
            o.b = (uint16_t)(rb * D * EB);
            o.ps = (uint16_t)((C::PS0 + la) * D * EB);
            o.u = (uint32_t)((C::SC_U + ra) * TP * EB);
            o.v = (uint32_t)((C::SC_V + rb) * TP * EB);
            o.own = (uint16_t)(lv_rowbase<N>(L) * D * EB);
            o.w = (uint32_t)((C::SC_W + lv_rowbase<N>(L) - N) * TP * EB);
            for (int lb = 1; lb <= L - la - 1; ++lb) {
                o.bm[lb - 1] = (uint16_t)((lv_rowbase<N>(lb) + la) * D * EB);
                o.c[lb - 1] = (uint16_t)((lv_rowbase<N>(L - la - lb) + la + lb) * D * EB);
            }
        }
    return t;
}

template <class F, int N, int D, int W, int S>
__constant__ UnitTable<N> c_unit_table = make_unit_table<F, N, D, W, S>();

// one unit with C4 4-gluon splits; entry and exit: every acc[] has room for kCapR more products
template <class F, int MET, int N, int D, int S, int C4>
__device__ __forceinline__ void unit_body(const F& f, int mu0, const typename F::E* __restrict__ ri,
                                          const typename F::E* __restrict__ si, const UnitOff<N>& o,
                                          const typename F::E (&x2)[D / S], typename F::A (&acc)[D / S],
                                          typename F::E& hsum)
{
    typedef typename F::E E;
    constexpr int DL = D / S, TP = 32 / S;
    const char* rb_ = reinterpret_cast<const char*>(ri);
    const char* sb_ = reinterpret_cast<const char*>(si);
    E a[DL], b[DL], s[DL], na[DL];
    ld_vec<F, DL>(reinterpret_cast<const E*>(rb_ + o.a), a);
    ld_vec<F, DL>(reinterpret_cast<const E*>(rb_ + o.b), b);
    ld_vec<F, DL>(reinterpret_cast<const E*>(rb_ + o.ps), s);      // PS2_k, k = i+la-1
    const E ua = *reinterpret_cast<const E*>(sb_ + o.u), vb = *reinterpret_cast<const E*>(sb_ + o.v);
    lower_neg<F, MET, DL>(f, mu0, a, na);
    const E h = f.neg(lane_sum<F, S, TP>(f, f.reduce(dot_plain<F, DL>(f, na, b))));   // A.B
    const E xa = lane_sum<F, S, TP>(f, f.reduce(dot_plain<F, DL>(f, x2, a)));         // 2 X.A
    const E xb = lane_sum<F, S, TP>(f, f.reduce(dot_plain<F, DL>(f, x2, b)));         // 2 X.B
    const E cb = f.sub(xa, ua);
    const E ca = f.sub(vb, xb);
    hsum = f.add(hsum, h);
    int room = F::kCapR;
    auto need = [&](int k) {
        if (room < k) {
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) acc[mu] = f.relief(acc[mu]);
            room = F::kCapR;
        }
        room -= k;
    };
    need(2);
#pragma unroll
    for (int mu = 0; mu < DL; ++mu) {
        acc[mu] = f.mad(h, s[mu], acc[mu]);
        acc[mu] = f.mad(cb, b[mu], acc[mu]);
    }
    need(1);
#pragma unroll
    for (int mu = 0; mu < DL; ++mu) acc[mu] = f.mad(ca, a[mu], acc[mu]);
#pragma unroll
    for (int q = 0; q < C4; ++q) {
        // (i..k | k+1..l | l+1..j), l = k+q+1: 2 (A.C) J(k+1..l)
        E bm[DL], c[DL];
        ld_vec<F, DL>(reinterpret_cast<const E*>(rb_ + o.bm[q]), bm);
        ld_vec<F, DL>(reinterpret_cast<const E*>(rb_ + o.c[q]), c);
        const E cc = f.neg(f.dbl(lane_sum<F, S, TP>(f, f.reduce(dot_plain<F, DL>(f, na, c)))));
        need(1);
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) acc[mu] = f.mad(cc, bm[mu], acc[mu]);
    }
    if (room < F::kCapR) {
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) acc[mu] = f.relief(acc[mu]);
    }
}

// dispatch on the (warp-uniform) number of 4-gluon splits
template <class F, int MET, int N, int D, int S, int C4>
struct UnitDispatch {
    __device__ __forceinline__ static void run(const F& f, int mu0, int c4, const typename F::E* __restrict__ ri,
                                               const typename F::E* __restrict__ si, const UnitOff<N>& o,
                                               const typename F::E (&x2)[D / S], typename F::A (&acc)[D / S],
                                               typename F::E& hsum)
    {
        if (c4 == C4) unit_body<F, MET, N, D, S, C4>(f, mu0, ri, si, o, x2, acc, hsum);
        else UnitDispatch<F, MET, N, D, S, C4 - 1>::run(f, mu0, c4, ri, si, o, x2, acc, hsum);
    }
};
template <class F, int MET, int N, int D, int S>
struct UnitDispatch<F, MET, N, D, S, -1> {
    __device__ __forceinline__ static void run(const F&, int, int, const typename F::E*, const typename F::E*,
                                               const UnitOff<N>&, const typename F::E (&)[D / S],
                                               typename F::A (&)[D / S], typename F::E&)
    {
    }
};

// Finish the current (ci, L) whose bracket sum is in acc (room for kCapR more products): boundary
// term of the (P-Q) sum, propagator, store, U and V; for the top current the amplitude instead
// (no propagator).  The ONE copy of this block (every kernel variant of round 1 had its own).
template <class F, int MET, int N, int D, int W, int S>
__device__ __forceinline__ void unit_finish(const F& f, const TileLane<F, N, D, W, S>& t, typename F::E* ri,
                                            typename F::E* si, const typename F::E (&l)[D / S],
                                            const typename F::E (&h)[D / S], const typename F::E (&x2)[D / S],
                                            typename F::A (&acc)[D / S], typename F::E hsum, int ci, int L, int own,
                                            int widx, typename F::E* out, typename F::E* currents)
{
    typedef TileCfg<F, N, D, W, S> C;
    typedef typename F::E E;
    constexpr int M = N - 1, DL = C::DL, TP = C::TP;
    const E nhh = f.neg(f.mul(hsum, f.half()));                 // -(sum_k h_k)/2
    if constexpr (F::kExact) {
        // one product per component: the two ALU instructions of the add are cheaper than a
        // second IMAD.WIDE (the multiplier pipe is the binding one)
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) acc[mu] = f.mad(nhh, f.add(l[mu], h[mu]), acc[mu]);
    } else {
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) {
            acc[mu] = f.mad(nhh, l[mu], acc[mu]);
            acc[mu] = f.mad(nhh, h[mu], acc[mu]);
        }
    }
    E v[DL];
    if (L < M) {
        const E w = *reinterpret_cast<const E*>(reinterpret_cast<const char*>(si) + widx);
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) v[mu] = f.mul(f.reduce(acc[mu]), w);
        st_vec<F, DL>(reinterpret_cast<E*>(reinterpret_cast<char*>(ri) + own), v);
        const E c2 = lane_sum<F, S, TP>(f, f.reduce(dot_plain<F, DL>(f, x2, v)));    // 2 P_{i,j} . J(i..j)
        const int urow = own / (D * (int)sizeof(E));
        si[(C::SC_U + urow) * TP] = f.add(c2, hsum);
        si[(C::SC_V + urow) * TP] = f.sub(c2, hsum);
    } else {
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) v[mu] = f.reduce(acc[mu]);
        E e[DL], ne[DL];
        ld_vec<F, DL>(t.rec() + (N - 1) * D, e);
        lower_neg<F, MET, DL>(f, t.mu0, e, ne);
        const E nout = lane_sum<F, S, TP>(f, f.reduce(dot_plain<F, DL>(f, ne, v)));  // -(eps_n . N)
        if (t.live && t.half == 0) *out = f.to_output(f.neg(nout));
    }
    if (currents && t.live) {
        E* dst = currents + (t.pt * M * M + (long long)ci * M + (ci + L - 1)) * D + t.mu0;
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) dst[mu] = f.to_output(v[mu]);
    }
}

// a4-a6 for one state configuration of one tile: the level sweep L = 2..m (Eq.(6)), amplitude, store.
template <class F, int MET, int N, int D, int W, int S>
__device__ __forceinline__ void unit_sweep_body(const F& f, const TileLane<F, N, D, W, S>& t, const int warp,
                                                typename F::E* out, typename F::E* currents)
{
    typedef TileCfg<F, N, D, W, S> C;
    typedef typename F::E E;
    typedef typename F::A A;
    constexpr int M = N - 1, DL = C::DL, TP = C::TP;
    const LevelProgram<N, W>& tb = c_level_program<F, N, D, W>;
    const UnitTable<N>& ut = c_unit_table<F, N, D, W, S>;
    E* rec = t.rec();
    E* sc = t.sc();
    // ---- a4-a6: level sweep L = 2..m (Eq.(6)), amplitude, store --------------------
#pragma unroll 1
    for (int L = 2; L <= M; ++L) {
        const int lbase = UnitTable<N>::index(L, 1);
        const int own = ut.u[lbase].own, widx = ut.u[lbase].w;
        const int t0 = tb.beg[L][warp], t1 = tb.beg[L][warp + 1];
#pragma unroll 1
        for (int k = t0; k < t1; ++k) {
            const uint32_t ta = tb.task[k].a;
            if (ta & LT_BAR) __syncthreads();
            if (!(ta & (LT_FIN | LT_PART))) continue;
            const int ci = ta & 15u, lo = ta >> 4 & 15u, hi = ta >> 8 & 15u;
            E* ri = rec + ci * D;
            E* si = sc + ci * TP;
            E l[DL], h[DL], x2[DL];
            ld_vec<F, DL>(ri + C::PS0 * D, l);                     // PS2_{i-1}
            ld_vec<F, DL>(ri + (C::PS0 + L) * D, h);               // PS2_j
            lower_diff<F, MET, DL>(f, t.mu0, h, l, x2);            // 2 * covariant P_{i,j}
            A acc[DL];
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) acc[mu] = f.zero();
            E hsum = f.ezero();
#pragma unroll 1
            for (int la = lo + 1; la <= hi; ++la)
                UnitDispatch<F, MET, N, D, S, N - 3>::run(f, t.mu0, L - la - 1, ri, si, ut.u[lbase + la - 1], x2,
                                                          acc, hsum);
            uint32_t mask = tb.task[k].mask;
            if (mask) {                                            // gather task (no units of its own)
                E sum[DL];
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) sum[mu] = f.ezero();
                while (mask) {
                    const int slot = __ffs(mask) - 1;
                    mask &= mask - 1;
                    const E* scr = sc + (C::SC_SCR + slot * (D + 1)) * TP;
#pragma unroll
                    for (int mu = 0; mu < DL; ++mu) sum[mu] = f.add(sum[mu], scr[(t.mu0 + mu) * TP]);
                    hsum = f.add(hsum, scr[D * TP]);
                }
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) acc[mu] = f.widen(sum[mu]);
            }
            if (ta & LT_PART) {
                E* scr = sc + (C::SC_SCR + (ta >> 12 & 63u) * (D + 1)) * TP;
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) scr[(t.mu0 + mu) * TP] = f.reduce(acc[mu]);
                scr[D * TP] = hsum;
                continue;
            }
            unit_finish<F, MET, N, D, W, S>(f, t, ri, si, l, h, x2, acc, hsum, ci, L, own, widx, out,
                                            currents);
        }
        if (L < M) __syncthreads();
    }
}

// MULTI = false: one state configuration and one colour ordering per point, no loops around the sweep (the
// headline path).  MULTI = true adds the loops over orderings and state configurations; it is a separate
// instantiation because ptxas stops using the uniform datapath for the control flow and the table loads of
// the sweep once it sits inside another loop (+12 % executed instructions, measured on cfg3).  (Calling the sweep
// as a __noinline__ function from the loops brings part of the uniform code back but costs more than it saves:
// S = 4 at cfg2's shape 1.00 -> 1.15 ms.)
template <class F, int MET, int N, int D, int W, int S, bool MULTI>
__global__ void __launch_bounds__(32 * W, TileCfg<F, N, D, W, S>::MIN_BLOCKS) bg_unit_kernel(const BgParams<F> prm)
{
    typedef TileCfg<F, N, D, W, S> C;
    typedef TileSetup<F, N, D, W, S> Setup;
    typedef typename F::E E;
    typedef typename F::A A;
    constexpr int M = N - 1, ND = N * D, DL = C::DL, TP = C::TP;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const F f(prm.fld, blockIdx.y);
    TileLane<F, N, D, W, S> t;
    t.vec = reinterpret_cast<E*>(smem_raw);                   // [TP][VSTRIDE]
    t.scal = t.vec + TP * C::VSTRIDE;                         // [NSCAL][TP]
    t.stat = reinterpret_cast<uint32_t*>(t.scal + TP * C::NSCAL);
    const LevelProgram<N, W>& tb = c_level_program<F, N, D, W>;
    const UnitTable<N>& ut = c_unit_table<F, N, D, W, S>;

    // the warp index, broadcast from lane 0 so that everything derived from it (task bounds,
    // task words, branch conditions) is compiled as warp-uniform
    const int lane = threadIdx.x & 31;
    const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
    t.warp = warp;
    t.point = S == 1 ? lane : lane & (TP - 1);
    t.half = S == 1 ? 0 : lane / TP;
    t.mu0 = S == 1 ? 0 : t.half * DL;
    t.q = blockIdx.y;
    t.tile0 = (long long)blockIdx.x * TP;
    t.valid = (int)min((long long)TP, prm.batch - t.tile0);
    t.pt = t.tile0 + t.point;
    t.live = t.point < t.valid;
    const int states = MULTI ? prm.states : 1, n_ord = MULTI ? prm.n_orderings : 1;
    const long long pbase = t.q * prm.batch;                  // first point of this prime's arrays
    const E* gmom = prm.mom + (pbase + t.tile0) * ND;
    const E* gpol = prm.pol + (pbase + t.tile0) * states * ND;
    E* gout = prm.out + (pbase + t.pt) * n_ord * states;
    uint32_t* gstat = prm.status ? prm.status + pbase : nullptr;

    // (a warp-uniform condition first: after a thread-divergent branch in front of the barriers ptxas no longer
    // treats the sweep as convergent and gives up the uniform datapath for its control flow and table loads)
    if (warp == 0 && lane < TP) t.stat[lane] = 0;
    E* rec = t.rec();
    E* sc = t.sc();
#pragma unroll 1
    for (int o = 0; o < n_ord; ++o, gout += states) {
    // colour ordering o (Eq.(5)): the inputs are re-staged in that order (from L2 after the
    // first pass) and everything below runs unchanged
    const unsigned char* perm = MULTI && prm.orderings ? prm.orderings + o * N : nullptr;
    if (o > 0) __syncthreads();                                // the previous sweep is done with the record
    // ---- a0: stage the momenta k_1..k_m (k_n is never used) and the first state configuration ----
    tile_stage<F, N, D, W, S, Setup::PARK, M>(f, t, gmom, ND, perm);
    tile_stage<F, N, D, W, S, 0, N>(f, t, gpol, (long long)states * ND, perm);
    __syncthreads();
    // ---- a1-a3: prefix sums, invariants, propagators (momenta only: once per tile and ordering) ----
    Setup::prefix(f, t);
    Setup::template singles<MET>(f, t, prm.currents);          // first state configuration
    Setup::template propagators<MET>(f, t, gstat);

#pragma unroll 1
    for (int s = 0; s < states; ++s) {
        if (s > 0) {
            __syncthreads();                                   // the previous sweep is done with eps_n
            tile_stage<F, N, D, W, S, 0, N>(f, t, gpol + (long long)s * ND, (long long)states * ND, perm);
            __syncthreads();
            Setup::template singles<MET>(f, t, prm.currents);
            __syncthreads();
        }

        unit_sweep_body<F, MET, N, D, W, S>(f, t, warp, gout + s, prm.currents);
    }
    }
}

}  // namespace bg
