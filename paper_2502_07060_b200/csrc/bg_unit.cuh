// bg_unit.cuh -- the Berends-Giele level sweep driven per UNIT, with one straight-line body per
// number of 4-gluon splits.
//
// Between bg_tile.cuh (a loop over single splittings: small code, ~22 instructions of decode per
// splitting) and bg_level.cuh (the code of every (level, left length) pair unrolled: no decode,
// but 90-230 KB of SASS and instruction-cache misses once the warps of an SM are spread over
// the levels): a unit = the 3-gluon split (i..i+la-1 | i+la..j) together with its c4 = L-la-1
// 4-gluon splits with the same left factor (Eq.(6)).  Its code depends on (L, la)
// only through c4 and through operand offsets, so there is ONE unrolled body per c4, and the
// offsets of a unit come from a small constexpr table in constant memory (warp-uniform loads,
// [register + uniform register] addressing).  Levels, tasks and units are run-time loops; the
// whole kernel is a few thousand instructions for any n.  Task lists (which warp does which
// units of which current, partial sums, gather tasks, barriers) are those of bg_level.cuh.
#pragma once
#include "bg_field.cuh"
#include "bg_recursion.cuh"
#include "bg_tables.cuh"
#include "bg_tile.cuh"
#include "bg_level.cuh"

namespace bg {

// BYTE offsets of the operands of unit (L, la), relative to the current's base pointers
// ri = rec + ci*D (vector rows) and si = sc + ci*32 (scalar tables): ready for [register + uniform
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

template <class F, int N, int D, int W>
constexpr UnitTable<N> make_unit_table()
{
    typedef TileCfg<F, N, D, W> C;
    UnitTable<N> t{};
    constexpr int M = N - 1;
    for (int L = 2; L <= M; ++L)
        for (int la = 1; la <= L - 1; ++la) {
            UnitOff<N>& o = t.u[UnitTable<N>::index(L, la)];
            const int ra = lv_rowbase<N>(la), rb = lv_rowbase<N>(L - la) + la;
            constexpr int EB = (int)sizeof(typename F::E);
            o.a = (uint16_t)(ra * D * EB);
            o.b = (uint16_t)(rb * D * EB);
            o.ps = (uint16_t)((C::PS0 + la) * D * EB);
            o.u = (uint32_t)((C::SC_U + ra) * 32 * EB);
            o.v = (uint32_t)((C::SC_V + rb) * 32 * EB);
            o.own = (uint16_t)(lv_rowbase<N>(L) * D * EB);
            o.w = (uint32_t)((C::SC_W + lv_rowbase<N>(L) - N) * 32 * EB);
            for (int lb = 1; lb <= L - la - 1; ++lb) {
                o.bm[lb - 1] = (uint16_t)((lv_rowbase<N>(lb) + la) * D * EB);
                o.c[lb - 1] = (uint16_t)((lv_rowbase<N>(L - la - lb) + la + lb) * D * EB);
            }
        }
    return t;
}

template <class F, int N, int D, int W>
__constant__ UnitTable<N> c_unit_table = make_unit_table<F, N, D, W>();

// one unit with C4 4-gluon splits; entry and exit: every acc[] has room for kCapR more products
template <class F, int N, int D, int C4>
__device__ __forceinline__ void unit_body(const typename F::E* __restrict__ ri, const typename F::E* __restrict__ si,
                                          const UnitOff<N>& o, const typename F::E (&x2)[D],
                                          typename F::A (&acc)[D], typename F::E& hsum)
{
    typedef typename F::E E;
    const char* rb_ = reinterpret_cast<const char*>(ri);
    const char* sb_ = reinterpret_cast<const char*>(si);
    E a[D], b[D], s[D];
    ld_vec<F, D>(reinterpret_cast<const E*>(rb_ + o.a), a);
    ld_vec<F, D>(reinterpret_cast<const E*>(rb_ + o.b), b);
    ld_vec<F, D>(reinterpret_cast<const E*>(rb_ + o.ps), s);       // PS2_k, k = i+la-1
    const E ua = *reinterpret_cast<const E*>(sb_ + o.u), vb = *reinterpret_cast<const E*>(sb_ + o.v);
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
    for (int q = 0; q < C4; ++q) {
        // (i..k | k+1..l | l+1..j), l = k+q+1: 2 (A.C) J(k+1..l)
        E bm[D], c[D];
        ld_vec<F, D>(reinterpret_cast<const E*>(rb_ + o.bm[q]), bm);
        ld_vec<F, D>(reinterpret_cast<const E*>(rb_ + o.c[q]), c);
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

// dispatch on the (warp-uniform) number of 4-gluon splits
template <class F, int N, int D, int C4>
struct UnitDispatch {
    __device__ __forceinline__ static void run(int c4, const typename F::E* __restrict__ ri,
                                               const typename F::E* __restrict__ si, const UnitOff<N>& o,
                                               const typename F::E (&x2)[D], typename F::A (&acc)[D],
                                               typename F::E& hsum)
    {
        if (c4 == C4) unit_body<F, N, D, C4>(ri, si, o, x2, acc, hsum);
        else UnitDispatch<F, N, D, C4 - 1>::run(c4, ri, si, o, x2, acc, hsum);
    }
};
template <class F, int N, int D>
struct UnitDispatch<F, N, D, -1> {
    __device__ __forceinline__ static void run(int, const typename F::E*, const typename F::E*, const UnitOff<N>&,
                                               const typename F::E (&)[D], typename F::A (&)[D], typename F::E&)
    {
    }
};

template <class F, int N, int D, int W>
__global__ void __launch_bounds__(32 * W) bg_unit_kernel(const TileParams<typename F::E> prm)
{
    typedef TileCfg<F, N, D, W> C;
    typedef typename F::E E;
    typedef typename F::A A;
    constexpr int M = N - 1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    E* vec = reinterpret_cast<E*>(smem_raw);                  // [32][VSTRIDE]
    E* scal = vec + 32 * C::VSTRIDE;                          // [NSCAL][32]
    uint32_t* stat = reinterpret_cast<uint32_t*>(scal + 32 * C::NSCAL);
    const LevelProgram<N, W>& tb = c_level_program<F, N, D, W>;
    const UnitTable<N>& ut = c_unit_table<F, N, D, W>;

    const int lane = threadIdx.x & 31, warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
    const long long tile0 = (long long)blockIdx.x * 32;
    const int valid = (int)min(32LL, prm.batch - tile0);
    const long long pt = tile0 + lane;
    const bool live = lane < valid;

    tile_setup<F, N, D, W>(vec, scal, stat, prm, lane, warp, tile0, valid, pt, live);
    E* rec = vec + (size_t)lane * C::VSTRIDE;
    E* sc = scal + lane;

#pragma unroll 1
    for (int L = 2; L <= M; ++L) {
        const bool top = L == M;
        const int lbase = UnitTable<N>::index(L, 1);
        const int own = ut.u[lbase].own, widx = ut.u[lbase].w;
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
#pragma unroll 1
            for (int la = lo + 1; la <= hi; ++la)
                UnitDispatch<F, N, D, N - 3>::run(L - la - 1, ri, si, ut.u[lbase + la - 1], x2, acc, hsum);
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
#pragma unroll
                for (int mu = 0; mu < D; ++mu) acc[mu] = F::mad(nhh, F::add(l[mu], h[mu]), acc[mu]);
            } else {
#pragma unroll
                for (int mu = 0; mu < D; ++mu) {
                    acc[mu] = F::mad(nhh, l[mu], acc[mu]);
                    acc[mu] = F::mad(nhh, h[mu], acc[mu]);
                }
            }
            E v[D];
            if (!top) {
                const E w = *reinterpret_cast<const E*>(reinterpret_cast<const char*>(si) + widx);
#pragma unroll
                for (int mu = 0; mu < D; ++mu) v[mu] = F::mul(F::reduce(acc[mu]), w);
                st_vec<F, D>(reinterpret_cast<E*>(reinterpret_cast<char*>(ri) + own), v);
                const E c2 = F::reduce(dot_plain<F, D>(x2, v));     // 2 P_{i,j} . J(i..j)
                const int urow = own / (D * (int)sizeof(E));
                si[(C::SC_U + urow) * 32] = F::add(c2, hsum);
                si[(C::SC_V + urow) * 32] = F::sub(c2, hsum);
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
        if (L < M) __syncthreads();
    }
}

}  // namespace bg
