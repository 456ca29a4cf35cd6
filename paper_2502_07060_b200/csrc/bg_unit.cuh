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

// ---- the flat per-warp program ---------------------------------------------------------------------
// The task lists of bg_schedule.cuh (levels -> tasks -> units) are flattened at compile time into ONE list
// of ops per warp; an op is one unit (or a gather / a bare barrier) with every operand offset resolved to a
// byte offset from the lane's record / scalar base, so the sweep is a single run-time loop whose body needs
// two 16-byte constant loads and a few warp-uniform flag tests (round 2 decoded a task word, a unit-table
// entry and a level header per iteration: 4.2 k of the 20.3 k instructions per cfg2 tile).
constexpr uint32_t OP_PAIR = 1u;      // this unit and the next one belong to the same task (see unit_pair_body)
constexpr uint32_t OP_START = 2u;     // first op of a task: form 2 P_{i,j}, clear the bracket sums
constexpr uint32_t OP_UNIT = 4u;      // a 3-gluon split with its c4 4-gluon splits
constexpr uint32_t OP_PART = 8u;      // last op of a later part of a shared current: park the partial sums, raise the flag
constexpr uint32_t OP_FIN = 16u;      // last op of a task: finish the current
constexpr uint32_t OP_GATHER = 32u;   // finisher of a shared current: check the flags, add the parked sums (aux = slots)
constexpr uint32_t OP_LEND = 64u;     // block barrier after the op (end of the level)
constexpr uint32_t OP_TOP = 128u;     // the current is J(1..m): amplitude instead of propagator and store


// what the operand offsets of an op depend on besides n: element size, tile width and the start of the PS2 rows
// and of the U / V tables
struct FlatLayout {
    int D, EB, TP, PS0, SC_U, SC_V;
};

template <int N, int W>
constexpr int flat_count(const LevelProgram<N, W>& p)
{
    constexpr int M = N - 1;
    int n = 0;
    for (int L = 2; L <= M; ++L)
        for (int w = 0; w < W; ++w) {
            int here = 0;
            for (int t = p.beg[L][w]; t < p.beg[L][w + 1]; ++t) {
                const uint32_t a = p.task[t].a;
                here += (int)(a >> 8 & 15u) - (int)(a >> 4 & 15u);          // one op per unit
            }
            n += here ? here : 1;                               // every warp takes the level-end barrier
        }
    return n;
}
template <int N, int W>
constexpr int flat_count_ops() { return flat_count<N, W>(LevelProgramOf<N, W>::value); }
constexpr int flat_count_quads(int n) { return n * (n - 1) * (n - 2) * (n - 3) / 24; }

// the ops of the schedule p for the layout y: op[flat_count(p)], quad[flat_count_quads(N)], beg[W + 1].  Evaluated by
// the compiler for the kernels with a compile-time (n, d), at run time on the host for bg_rt_kernel (bg_api.cu).
template <int N, int W>
constexpr void flat_build(const LevelProgram<N, W>& p, const FlatLayout& y, FlatOp* op, uint32_t* quad, uint16_t* beg)
{
    constexpr int M = N - 1;
    static_assert(M * M <= 256 && N + M * (M - 1) / 2 <= 256, "8-bit fields of FlatOp::w");
    const int D = y.D, EB = y.EB, TP = y.TP, RB = D * EB;
    int no = 0, nq = 0;
    for (int w = 0; w < W; ++w) {
        beg[w] = (uint16_t)no;
        for (int L = 2; L <= M; ++L) {
            const int first = no;
            for (int t = p.beg[L][w]; t < p.beg[L][w + 1]; ++t) {
                const uint32_t a = p.task[t].a, mask = p.task[t].mask;
                const int ci = a & 15u, lo = a >> 4 & 15u, hi = a >> 8 & 15u, slot = a >> 12 & 63u;
                const int own = lv_rowbase<N>(L) + ci;
                const uint32_t endf = ((a & LT_PART) ? OP_PART : mask ? OP_GATHER | OP_FIN : OP_FIN) |
                                      (L == M ? OP_TOP : 0u);
                const uint32_t wfield = (uint32_t)(ci * M + ci + L - 1) | (uint32_t)own << 8 |
                                        (uint32_t)L << 16 | ((a & LT_PART) ? (uint32_t)(32 * slot) << 20 : 0u);
                const uint32_t lh = (uint32_t)((y.PS0 + ci) * RB) | (uint32_t)((y.PS0 + ci + L) * RB) << 16;
                const uint32_t aux = (a & LT_PART) ? (uint32_t)(slot * (D + 1) * TP * EB) : mask;
                for (int la = lo + 1; la <= hi; ++la) {
                    FlatOp& o = op[no++];
                    const int ra = lv_rowbase<N>(la) + ci, rb = lv_rowbase<N>(L - la) + ci + la, c4 = L - la - 1;
                    o.ab = (uint32_t)(ra * RB) | (uint32_t)(rb * RB) << 16;
                    o.pso = (uint32_t)((y.PS0 + ci + la) * RB) | (uint32_t)(own * RB) << 16;
                    o.u = (uint32_t)((y.SC_U + ra) * TP * EB);
                    o.v = (uint32_t)((rb < N ? y.SC_U + rb : y.SC_V + rb - N) * TP * EB);    // V = U for single gluons
                    o.w = wfield;
                    o.lh = lh;
                    o.aux = aux;
                    const uint32_t fl = OP_UNIT | (la == lo + 1 ? OP_START : 0u) | (la == hi ? endf : 0u) |
                                        ((la - lo) % 2 == 1 && la < hi ? OP_PAIR : 0u);
                    o.qcf = (uint32_t)nq | (uint32_t)c4 << 16 | fl << 24;
                    for (int lb = 1; lb <= c4; ++lb)
                        quad[nq++] = (uint32_t)((lv_rowbase<N>(lb) + ci + la) * RB) |
                                     (uint32_t)((lv_rowbase<N>(L - la - lb) + ci + la + lb) * RB) << 16;
                }
            }
            if (no == first) {                                  // nothing to do at this level but the barrier
                op[no] = FlatOp{};
                ++no;
            }
            if (L < M) op[no - 1].qcf |= OP_LEND << 24;
        }
    }
    beg[W] = (uint16_t)no;
}

template <int N, int W>
struct FlatProgram {
    static constexpr int NOPS = flat_count_ops<N, W>();
    static constexpr int NQUAD = flat_count_quads(N);
    FlatOp op[NOPS];
    uint32_t quad[NQUAD > 0 ? NQUAD : 1];     // row J(k+1..l) | row J(l+1..j) << 16 per 4-gluon split
    uint16_t beg[W + 1];                      // ops of warp w: [beg[w], beg[w+1])
};

template <class F, int N, int D, int W, int S>
constexpr FlatProgram<N, W> make_flat_program()
{
    typedef TileCfg<F, N, D, W, S, false> C;    // only what does not depend on KW is used below
    static_assert((long)C::VEC_ROWS * D * sizeof(typename F::E) < 65536, "row offsets are 16-bit");
    FlatProgram<N, W> f{};
    flat_build<N, W>(LevelProgramOf<N, W>::value, FlatLayout{D, (int)sizeof(typename F::E), C::TP, C::PS0, C::SC_U, C::SC_V},
                     f.op, f.quad, f.beg);
    return f;
}

template <class F, int N, int D, int W, int S>
__constant__ FlatProgram<N, W> c_flat_program = make_flat_program<F, N, D, W, S>();

// The finish and the sweep below are written against two small policies, so that the kernels with a compile-time
// (n, d) and the run-time-n kernel (bg_rt.cuh) share them: the LAYOUT (where the scalar tables start, n) and the
// PROGRAM (where the ops come from).  For the compile-time kernels both are empty objects whose members fold.
template <class C>
struct StaticLay {
    __device__ __forceinline__ static constexpr int n() { return C::M + 1; }
    __device__ __forceinline__ static constexpr int sc_u() { return C::SC_U; }
    __device__ __forceinline__ static constexpr int sc_v() { return C::SC_V; }
    __device__ __forceinline__ static constexpr int sc_w() { return C::SC_W; }
    __device__ __forceinline__ static constexpr int sc_scr() { return C::SC_SCR; }
};
template <class F, int N, int D, int W, int S>
struct StaticProg {
    typedef const FlatOp& Op;
    __device__ __forceinline__ Op op(int k) const { return c_flat_program<F, N, D, W, S>.op[k]; }
    __device__ __forceinline__ const uint32_t* quad() const { return c_flat_program<F, N, D, W, S>.quad; }
    __device__ __forceinline__ int beg(int w) const { return c_flat_program<F, N, D, W, S>.beg[w]; }
};

// the 4-gluon split (i..k | k+1..l | l+1..j): acc -= 2 (A.C) J(k+1..l); na = -g A
template <class F, int D, int S>
__device__ __forceinline__ void unit_quad(const F& f, const char* __restrict__ rb_, uint32_t bc,
                                          const typename F::E (&na)[D / S], typename F::A (&acc)[D / S])
{
    typedef typename F::E E;
    constexpr int DL = D / S, TP = 32 / S;
    E bm[DL], c[DL];
    ld_vec<F, DL>(reinterpret_cast<const E*>(rb_ + (bc & 0xffffu)), bm);
    ld_vec<F, DL>(reinterpret_cast<const E*>(rb_ + (bc >> 16)), c);
    const E ncc = f.dbl(lane_sum<F, S, TP>(f, f.reduce(dot_plain<F, DL>(f, na, c))));       // -2 A.C
#pragma unroll
    for (int mu = 0; mu < DL; ++mu) acc[mu] = f.mad(ncc, bm[mu], acc[mu]);
}

// the 3-gluon split (A | B) of a unit, SUBTRACTED from acc (nx2 = -2 covariant X, nhsum = -sum_k h_k); returns
// na = -g A for the unit's 4-gluon splits.  Entry: room for kCapR products; exit: room for one more.
template <class F, int MET, int D, int S>
__device__ __forceinline__ void unit_split3(const F& f, int mu0, const char* __restrict__ rb_,
                                            const char* __restrict__ sb_, const FlatOp& o,
                                            const typename F::E (&nx2)[D / S], typename F::A (&acc)[D / S],
                                            typename F::E& nhsum, typename F::E (&na)[D / S])
{
    typedef typename F::E E;
    constexpr int DL = D / S, TP = 32 / S;
    static_assert(F::kCapR >= 2, "the relief pattern assumes room for two products after relief()");
    E a[DL], b[DL], s[DL];
    ld_vec<F, DL>(reinterpret_cast<const E*>(rb_ + (o.ab & 0xffffu)), a);
    ld_vec<F, DL>(reinterpret_cast<const E*>(rb_ + (o.ab >> 16)), b);
    ld_vec<F, DL>(reinterpret_cast<const E*>(rb_ + (o.pso & 0xffffu)), s);      // PS2_k, k = i+la-1
    const E ua = *reinterpret_cast<const E*>(sb_ + o.u), vb = *reinterpret_cast<const E*>(sb_ + o.v);
    lower_neg<F, MET, DL>(f, mu0, a, na);
    const E nh = lane_sum<F, S, TP>(f, f.reduce(dot_plain<F, DL>(f, na, b)));          // -A.B
    E ncb, nca;                                                                        // U_A - 2X.A, 2X.B - V_B
    if constexpr (S == 1) {
        ncb = f.reduce(dot_plain_from<F, DL>(f, ua, nx2, a));
        nca = f.neg(f.reduce(dot_plain_from<F, DL>(f, vb, nx2, b)));
    } else {
        ncb = f.add(ua, lane_sum<F, S, TP>(f, f.reduce(dot_plain<F, DL>(f, nx2, a))));
        nca = f.neg(f.add(vb, lane_sum<F, S, TP>(f, f.reduce(dot_plain<F, DL>(f, nx2, b)))));
    }
    nhsum = f.add(nhsum, nh);
#pragma unroll
    for (int mu = 0; mu < DL; ++mu) {
        acc[mu] = f.mad(nh, s[mu], acc[mu]);
        acc[mu] = f.mad(ncb, b[mu], acc[mu]);
    }
    if (F::kExact) {
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) acc[mu] = f.relief(acc[mu]);
    }
#pragma unroll
    for (int mu = 0; mu < DL; ++mu) acc[mu] = f.mad(nca, a[mu], acc[mu]);     // room for one more product
}

// one unit: the 3-gluon split (A | B) and its c4 4-gluon splits; entry and exit: every acc[] has room for kCapR
// more products.  The 4-gluon splits are a run-time loop over pairs (the relief pattern of a pair is static), so
// there is ONE body for every c4 and the kernel stays inside the instruction cache for any n.
template <class F, int MET, int N, int D, int S>
__device__ __forceinline__ void unit_body(const F& f, int mu0, const typename F::E* __restrict__ rec,
                                          const typename F::E* __restrict__ sc, const FlatOp& o,
                                          const uint32_t* __restrict__ quad, const typename F::E (&nx2)[D / S],
                                          typename F::A (&acc)[D / S], typename F::E& nhsum)
{
    typedef typename F::E E;
    constexpr int DL = D / S;
    const char* rb_ = reinterpret_cast<const char*>(rec);
    const char* sb_ = reinterpret_cast<const char*>(sc);
    E na[DL];
    unit_split3<F, MET, D, S>(f, mu0, rb_, sb_, o, nx2, acc, nhsum, na);
    auto relieve = [&]() {
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) acc[mu] = f.relief(acc[mu]);
    };
    const int c4 = o.qcf >> 16 & 0xffu;
    const uint32_t* qd = quad + (o.qcf & 0xffffu);
    int q = 0;
#pragma unroll 1
    for (; q + 2 <= c4; q += 2) {
        unit_quad<F, D, S>(f, rb_, qd[q], na, acc);
        if (F::kExact) relieve();
        unit_quad<F, D, S>(f, rb_, qd[q + 1], na, acc);                      // room for one more product again
    }
    if (q < c4) {
        unit_quad<F, D, S>(f, rb_, qd[q], na, acc);
    }
    if (F::kExact) relieve();
}

// Two consecutive units (i..k | ..) and (i..k+1 | ..) of one current together: their 4-gluon splits with the same
// right factor C = J(l+1..j) share ONE load of C (the 4-gluon split q >= 1 of the first unit and q - 1 of the second),
// 1.5 instead of 2 vector loads per split.  Used where shared-memory traffic binds (complex128: a 16-byte element
// per lane makes every vector load 4 wavefronts per warp); same arithmetic, other order of the sums.
template <class F, int MET, int N, int D, int S>
__device__ __forceinline__ void unit_pair_body(const F& f, int mu0, const typename F::E* __restrict__ rec,
                                               const typename F::E* __restrict__ sc, const FlatOp& o1,
                                               const FlatOp& o2, const uint32_t* __restrict__ quad,
                                               const typename F::E (&nx2)[D / S], typename F::A (&acc)[D / S],
                                               typename F::E& nhsum)
{
    typedef typename F::E E;
    constexpr int DL = D / S, TP = 32 / S;
    const char* rb_ = reinterpret_cast<const char*>(rec);
    const char* sb_ = reinterpret_cast<const char*>(sc);
    auto relieve = [&]() {
        if (F::kExact) {
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) acc[mu] = f.relief(acc[mu]);
        }
    };
    E na1[DL], na2[DL];
    unit_split3<F, MET, D, S>(f, mu0, rb_, sb_, o1, nx2, acc, nhsum, na1);
    relieve();
    unit_split3<F, MET, D, S>(f, mu0, rb_, sb_, o2, nx2, acc, nhsum, na2);
    const int c4 = o1.qcf >> 16 & 0xffu;                       // the second unit has c4 - 1
    const uint32_t* qd1 = quad + (o1.qcf & 0xffffu);
    const uint32_t* qd2 = quad + (o2.qcf & 0xffffu);
    if (c4 > 0) unit_quad<F, D, S>(f, rb_, qd1[0], na1, acc);   // (k+1 | k+2..j): no partner
    relieve();
#pragma unroll 1
    for (int q = 1; q < c4; ++q) {
        const uint32_t bc1 = qd1[q], bc2 = qd2[q - 1];
        E c[DL], m1[DL], m2[DL];
        ld_vec<F, DL>(reinterpret_cast<const E*>(rb_ + (bc1 >> 16)), c);
        ld_vec<F, DL>(reinterpret_cast<const E*>(rb_ + (bc1 & 0xffffu)), m1);
        ld_vec<F, DL>(reinterpret_cast<const E*>(rb_ + (bc2 & 0xffffu)), m2);
        const E n1 = f.dbl(lane_sum<F, S, TP>(f, f.reduce(dot_plain<F, DL>(f, na1, c))));    // -2 A1.C
        const E n2 = f.dbl(lane_sum<F, S, TP>(f, f.reduce(dot_plain<F, DL>(f, na2, c))));    // -2 A2.C
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) {
            acc[mu] = f.mad(n1, m1[mu], acc[mu]);
            acc[mu] = f.mad(n2, m2[mu], acc[mu]);
        }
        relieve();
    }
}

// Finish the current whose bracket sum is in acc, NEGATED (room for kCapR more products): boundary term of the
// (P-Q) sum, propagator (the table holds -1/P^2), store, U and V; for the top current the amplitude instead (no
// propagator).  nx2 = -2 covariant P_{i,j}, nhsum = -sum_k h_k.
// t: the lane's mu0, half, live, pt.
template <class F, int MET, int D, int S, class Lay, class Lane>
__device__ __forceinline__ void unit_finish(const F& f, const Lay& lay, const Lane& t, typename F::E* rec,
                                            typename F::E* sc, const FlatOp& o, bool top,
                                            const typename F::E (&nx2)[D / S], typename F::A (&acc)[D / S],
                                            typename F::E nhsum, typename F::E* out, typename F::E* currents)
{
    typedef typename F::E E;
    constexpr int DL = D / S, TP = 32 / S;
    const int N = lay.n(), M = N - 1;
    char* rb_ = reinterpret_cast<char*>(rec);
    E l[DL], h[DL];
    ld_vec<F, DL>(reinterpret_cast<const E*>(rb_ + (o.lh & 0xffffu)), l);     // PS2_{i-1}
    ld_vec<F, DL>(reinterpret_cast<const E*>(rb_ + (o.lh >> 16)), h);         // PS2_j
    const E nhh = f.neg(f.mul(nhsum, f.half()));                // +(sum_k h_k)/2: minus the boundary coefficient
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
    if (!top) {
        const uint32_t own = o.pso >> 16, urow = o.w >> 8 & 0xffu;
        const E w = sc[(lay.sc_w() + urow - N) * TP];           // -1/P^2
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) v[mu] = f.mul(f.reduce(acc[mu]), w);
        st_vec<F, DL>(reinterpret_cast<E*>(rb_ + own), v);
        const E nc2 = lane_sum<F, S, TP>(f, f.reduce(dot_plain<F, DL>(f, nx2, v)));  // -2 P_{i,j} . J(i..j)
        sc[(lay.sc_u() + urow) * TP] = f.canon(f.neg(f.add(nc2, nhsum)));            // U = 2 P.J + sum_k h_k
        sc[(lay.sc_v() + urow - N) * TP] = f.sub(nhsum, nc2);                        // V = 2 P.J - sum_k h_k
        if (currents && t.live) {
            E* dst = currents + (t.pt * M * M + (long long)(o.w & 0xffu)) * D + t.mu0;
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) dst[mu] = f.to_output(v[mu]);
        }
    } else {
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) v[mu] = f.reduce(acc[mu]);
        E e[DL], ne[DL];
        ld_vec<F, DL>(rec + (N - 1) * D, e);
        lower_neg<F, MET, DL>(f, t.mu0, e, ne);
        const E o_ = lane_sum<F, S, TP>(f, f.reduce(dot_plain<F, DL>(f, ne, v)));    // -(eps_n . v) = eps_n . N
        if (t.live && t.half == 0) *out = f.to_output(o_);
        if (currents && t.live) {                               // v = -N(1..m)
            E* dst = currents + (t.pt * M * M + (long long)(o.w & 0xffu)) * D + t.mu0;
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) dst[mu] = f.to_output(f.neg(v[mu]));
        }
    }
}

// a4-a6 for one state configuration of one tile: the level sweep L = 2..m (Eq.(6)), amplitude, store.
// rec, sc: the lane's record and scalar column; flags: the lane's parked flags, [slot * 32].
template <class F, int MET, int D, int S, class Lay, class Prog, class Lane>
__device__ __forceinline__ void unit_sweep_body(const F& f, const Lay& lay, const Prog& prog, const Lane& t,
                                                const int warp, typename F::E* rec, typename F::E* sc,
                                                uint32_t* flags, const uint32_t epoch0, typename F::E* out,
                                                typename F::E* currents)
{
    typedef typename F::E E;
    typedef typename F::A A;
    constexpr int DL = D / S, TP = 32 / S, N = 0;              // (N: unused template argument of the unit bodies)
    constexpr bool kPairs = !F::kExact;                         // unit pairs where shared-memory traffic binds
    char* rb_ = reinterpret_cast<char*>(rec);
    char* sb_ = reinterpret_cast<char*>(sc);
    E nx2[DL];
    A acc[DL];
    E nhsum = f.ezero();
#pragma unroll
    for (int mu = 0; mu < DL; ++mu) { nx2[mu] = f.ezero(); acc[mu] = f.zero(); }
    const int k0 = prog.beg(warp), k1 = prog.beg(warp + 1);
#pragma unroll 1
    for (int k = k0; k < k1; ++k) {
        typename Prog::Op o = prog.op(k);
        const uint32_t fl = o.qcf >> 24;
        if (fl & OP_START) {
            E l[DL], h[DL];
            ld_vec<F, DL>(reinterpret_cast<const E*>(rb_ + (o.lh & 0xffffu)), l);     // PS2_{i-1}
            ld_vec<F, DL>(reinterpret_cast<const E*>(rb_ + (o.lh >> 16)), h);         // PS2_j
            lower_diff<F, MET, DL>(f, t.mu0, l, h, nx2);                              // -2 * covariant P_{i,j}
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) acc[mu] = f.zero();
            nhsum = f.ezero();
        }
        if constexpr (kPairs) {
            if (fl & OP_PAIR) {
                typename Prog::Op o2 = prog.op(k + 1);
                unit_pair_body<F, MET, N, D, S>(f, t.mu0, rec, sc, o, o2, prog.quad(), nx2, acc, nhsum);
                ++k;                                            // the second unit carries the task's end flags
            } else if (fl & OP_UNIT) {
                unit_body<F, MET, N, D, S>(f, t.mu0, rec, sc, o, prog.quad(), nx2, acc, nhsum);
            }
        } else if (fl & OP_UNIT) {
            unit_body<F, MET, N, D, S>(f, t.mu0, rec, sc, o, prog.quad(), nx2, acc, nhsum);
        }
        typename Prog::Op oe = prog.op(k);                     // the op that carries the task's end flags
        const uint32_t fle = oe.qcf >> 24;
        if (fle & OP_PART) {
            // a later part of a current shared between warps: park the partial sums, tell the finisher.
            // (a byte offset from the table, not slot * (D + 1): a run-time multiply here makes ptxas give up the
            // uniform datapath for the whole sweep, +4.5 % at cfg2)
            E* scr = reinterpret_cast<E*>(sb_ + lay.sc_scr() * TP * (int)sizeof(E) + oe.aux);
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) scr[(t.mu0 + mu) * TP] = f.reduce(acc[mu]);
            scr[D * TP] = nhsum;
            // the lane that reads a parked value is this lane of the finishing warp: a per-lane flag, raised after
            // the values (fence), tells it that they are there; `epoch` is unique per sweep and level
            __threadfence_block();
            *reinterpret_cast<volatile uint32_t*>(flags + (oe.w >> 20)) = epoch0 + (oe.w >> 16 & 15u);
        }
        if (fle & OP_GATHER) {
            // the finisher (owner of the first units, this is its last task of the level): the other parts were
            // first tasks of their warps and are parked by now
            const uint32_t epoch = epoch0 + (oe.w >> 16 & 15u);
            for (uint32_t m2 = oe.aux; m2; m2 &= m2 - 1) {
                const volatile uint32_t* fl_ = flags + 32 * (__ffs(m2) - 1);
                while (!__all_sync(0xffffffffu, *fl_ == epoch)) {}    // warp-uniform exit
            }
            __threadfence_block();
            uint32_t mask = oe.aux;
            E sum[DL];
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) sum[mu] = f.ezero();
            while (mask) {
                const int slot = __ffs(mask) - 1;
                mask &= mask - 1;
                const E* scr = sc + (lay.sc_scr() + slot * (D + 1)) * TP;
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) sum[mu] = f.add(sum[mu], scr[(t.mu0 + mu) * TP]);
                nhsum = f.add(nhsum, scr[D * TP]);
            }
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) acc[mu] = f.addw(acc[mu], sum[mu]);   // one of the kCapR products of room
        }
        if (fle & OP_FIN)
            unit_finish<F, MET, D, S>(f, lay, t, rec, sc, oe, (fle & OP_TOP) != 0, nx2, acc, nhsum, out, currents);
        if (fle & OP_LEND) __syncthreads();
    }
}

// MULTI = false: one state configuration and one colour ordering per point, no loops around the sweep (the
// headline path).  MULTI = true adds the loops over orderings and state configurations; it is a separate
// instantiation because ptxas stops using the uniform datapath for the control flow and the table loads of
// the sweep once it sits inside another loop (+12 % executed instructions, measured on cfg3).  (Calling the sweep
// as a __noinline__ function from the loops brings part of the uniform code back but costs more than it saves:
// S = 4 at cfg2's shape 1.00 -> 1.15 ms.)
template <class F, int MET, int N, int D, int W, int S, bool MULTI>
__global__ void __launch_bounds__(32 * W, TileCfg<F, N, D, W, S, MULTI>::MIN_BLOCKS) bg_unit_kernel(const BgParams<F> prm)
{
    constexpr bool KW = MULTI;
    typedef TileCfg<F, N, D, W, S, KW> C;
    typedef TileSetup<F, N, D, W, S, KW> Setup;
    typedef typename F::E E;
    typedef typename F::A A;
    constexpr int M = N - 1, ND = N * D, DL = C::DL, TP = C::TP;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const F f(prm.fld, blockIdx.y);
    TileLane<F, N, D, W, S, KW> t;
    t.vec = reinterpret_cast<E*>(smem_raw);                   // [TP][VSTRIDE]
    t.scal = t.vec + TP * C::VSTRIDE;                         // [NSCAL][TP]
    t.stat = reinterpret_cast<uint32_t*>(t.scal + TP * C::NSCAL);
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
#pragma unroll 1
    for (int sl = warp; sl < C::NSLOTS; sl += W) t.stat[TP + 32 * sl + lane] = 0;    // parked flags (epochs start at 1)
    E* rec = t.rec();
    E* sc = t.sc();
#pragma unroll 1
    for (int o = 0; o < n_ord; ++o, gout += states) {
    // colour ordering o (Eq.(5)): the inputs are re-staged in that order (from L2 after the
    // first pass) and everything below runs unchanged
    const unsigned char* perm = MULTI && prm.orderings ? prm.orderings + o * N : nullptr;
    if (o > 0) __syncthreads();                                // the previous sweep is done with the record
    // ---- a0: stage the momenta k_1..k_m (k_n is never used) and the first state configuration ----
    tile_stage<F, N, D, W, S, KW, Setup::PARK, M>(f, t, gmom, ND, perm);
    tile_stage<F, N, D, W, S, KW, 0, N>(f, t, gpol, (long long)states * ND, perm);
    __syncthreads();
    // ---- a1-a3: prefix sums, invariants, propagators (momenta only: once per tile and ordering) ----
    Setup::prefix(f, t);
    Setup::template singles<MET>(f, t, prm.currents);          // first state configuration
    Setup::template propagators<MET>(f, t, gstat);

#pragma unroll 1
    for (int s = 0; s < states; ++s) {
        if (s > 0) {
            __syncthreads();                                   // the previous sweep is done with eps_n
            tile_stage<F, N, D, W, S, KW, 0, N>(f, t, gpol + (long long)s * ND, (long long)states * ND, perm);
            __syncthreads();
            Setup::template singles<MET>(f, t, prm.currents);
            __syncthreads();
        }

        unit_sweep_body<F, MET, D, S>(f, StaticLay<C>(), StaticProg<F, N, D, W, S>(), t, warp, rec, sc,
                                      t.stat + TP + lane, (uint32_t)(o * states + s) * 16u, gout + s, prm.currents);
    }
    }
}

}  // namespace bg
