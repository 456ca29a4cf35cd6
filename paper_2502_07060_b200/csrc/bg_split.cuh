// bg_split.cuh -- the table-driven tiled Berends-Giele kernel with S = 2 lanes per point.
//
// For shapes whose per-point record is large (complex128 at n = 12 needs 11 KB per point) a
// 32-point tile does not fit an SM's shared memory, and the one-thread-per-point kernel is
// left with a single half-empty warp per SM.  Here a tile holds TP = 32/S points and the S
// lanes (l, l + TP) of every warp share one point: each owns DL = D/S of the d vector
// components.  Everything that is linear in a vector (the axpy updates of Eq.(6)'s bracket,
// PAPER.md:95, loads, stores) is simply done on the lane's own components; a Minkowski
// product is the sum of the two lanes' partial products, exchanged with one
// warp shuffle.  Scalars (U, V, 1/P^2, sum_k h_k) are computed redundantly by both lanes.
// Control flow stays uniform across the warp, shared-memory accesses stay conflict-free
// (same record stride rule as bg_tile.cuh), and the work lists are the ones of bg_tables.cuh.
//
// Algebra, layout of the per-point record and the scratch/gather scheme: see bg_tile.cuh.
#pragma once
#include "bg_field.cuh"
#include "bg_recursion.cuh"
#include "bg_tables.cuh"
#include "bg_tile.cuh"

namespace bg {

template <class F, int N, int D, int W, int S>
struct SplitCfg {
    typedef TileCfg<F, N, D, W> T;
    typedef typename F::E E;
    static_assert(S == 2 && D % S == 0, "two lanes per point, even d");
    static constexpr int TP = 32 / S;                         // points per tile
    static constexpr int DL = D / S;                          // components per lane
    static constexpr size_t SMEM_BYTES = (size_t)TP * (T::VSTRIDE + T::NSCAL) * sizeof(E) + TP * sizeof(uint32_t);
};

// same work lists as bg_tile.cuh, scalar columns TP wide
template <class F, int N, int D, int W, int S>
__constant__ TileProgram<N, W> c_split_program = make_tile_program<N, W>(
    D * (int)sizeof(typename F::E), TileCfg<F, N, D, W>::PS0, TileCfg<F, N, D, W>::SC_U, TileCfg<F, N, D, W>::SC_V,
    SplitCfg<F, N, D, W, S>::TP * (int)sizeof(typename F::E));

// x or -x, per lane (the time component's metric sign lives in the lane that owns it)
__device__ __forceinline__ uint32_t cneg(uint32_t x, bool f) { return x ^ (f ? kP : 0u); }
__device__ __forceinline__ double2 cneg(double2 x, bool f)
{
    const double s = f ? -1.0 : 1.0;
    return make_double2(x.x * s, x.y * s);
}

// sum of the two lanes' values
template <class F, int TP>
__device__ __forceinline__ uint32_t pair_sum(uint32_t x)
{
    return F::add(x, __shfl_xor_sync(0xffffffffu, x, TP));
}
template <class F, int TP>
__device__ __forceinline__ double2 pair_sum(double2 x)
{
    return make_double2(x.x + __shfl_xor_sync(0xffffffffu, x.x, TP), x.y + __shfl_xor_sync(0xffffffffu, x.y, TP));
}

// MINUS the Minkowski product of two vectors held as (lane 0: components 0..DL-1, lane 1: the
// rest); t0 = this lane owns the time component.  Returns the full value in both lanes.
template <class F, int DL, int TP>
__device__ __forceinline__ typename F::E split_dot_neg(bool t0, const typename F::E (&x)[DL],
                                                       const typename F::E (&y)[DL])
{
    return pair_sum<F, TP>(F::reduce(dot_neg<F, DL>(cneg(x[0], t0), x, y)));
}
template <class F, int DL, int TP>
__device__ __forceinline__ typename F::E split_dot_plain(const typename F::E (&x)[DL], const typename F::E (&y)[DL])
{
    return pair_sum<F, TP>(F::reduce(dot_plain<F, DL>(x, y)));
}

// Finish the current stored at `own`; same steps as tile_finish (bg_tile.cuh).
template <class F, int N, int D, int W, int S>
__device__ __forceinline__ void split_finish(typename F::E* __restrict__ rec, typename F::E* __restrict__ sc,
                                             typename F::A (&acc)[D / S], typename F::E hsum, int own, int lo,
                                             int hi, bool top, bool t0, int half,
                                             const TileParams<typename F::E>& prm, long long pt, bool live)
{
    typedef TileCfg<F, N, D, W> C;
    typedef SplitCfg<F, N, D, W, S> SC;
    typedef typename F::E E;
    constexpr int DL = SC::DL, TP = SC::TP;
    E l[DL], h[DL];
    ld_vec<F, DL>(rec + (C::PS0 + lo) * D, l);
    ld_vec<F, DL>(rec + (C::PS0 + hi) * D, h);
    const E nhh = F::neg(F::mul(hsum, F::half()));               // -(sum_k h_k)/2
#pragma unroll
    for (int mu = 0; mu < DL; ++mu) {
        acc[mu] = F::relief(acc[mu]);
        acc[mu] = F::mad(nhh, l[mu], acc[mu]);
        acc[mu] = F::mad(nhh, h[mu], acc[mu]);
    }
    E v[DL];
    if (!top) {
        const E w = sc[(C::SC_W + own - N) * TP];
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) v[mu] = F::mul(F::reduce(acc[mu]), w);
        st_vec<F, DL>(rec + own * D, v);
        E x2[DL];
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) x2[mu] = F::sub(l[mu], h[mu]);
        x2[0] = cneg(x2[0], t0);                                  // 2 * covariant P_{i,j}
        const E c2 = split_dot_plain<F, DL, TP>(x2, v);          // 2 P_{i,j} . J(i..j)
        sc[(C::SC_U + own) * TP] = F::add(c2, hsum);
        sc[(C::SC_V + own) * TP] = F::sub(c2, hsum);
    } else {
        // top current: no propagator; amplitude = eps_n . N(1..m)
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) v[mu] = F::reduce(acc[mu]);
        E e[DL];
        ld_vec<F, DL>(rec + (N - 1) * D, e);
        const E nout = split_dot_neg<F, DL, TP>(t0, e, v);
        if (live && half == 0) prm.out[pt] = F::canon(F::neg(nout));
    }
    if (prm.currents && live) {
        constexpr int M = C::M;
        E* dst = prm.currents + (pt * M * M + (long long)lo * M + (hi - 1)) * D + half * DL;
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) dst[mu] = F::canon(v[mu]);
    }
}

// a0-a3 for one 16-point tile (stage, doubled prefix sums, single-gluon U/V, invariants, batch-inverted
// propagators); ends with a block barrier.  Shared by bg_split_kernel and bg_level2_kernel.
template <class F, int N, int D, int W, int S>
__device__ __forceinline__ void split_setup(typename F::E* __restrict__ vec, typename F::E* __restrict__ scal,
                                            uint32_t* __restrict__ stat, const TileParams<typename F::E>& prm,
                                            int warp, int point, int half, bool t0, long long tile0, int valid,
                                            long long pt, bool live)
{
    typedef TileCfg<F, N, D, W> C;
    typedef SplitCfg<F, N, D, W, S> SC;
    typedef typename F::E E;
    typedef typename F::A A;
    constexpr int M = C::M, U = C::U, ND = N * D, TP = SC::TP, DL = SC::DL;
    // ---- a0: stage the tile (coalesced, one vector unit per thread and step) ---------------------
    {
        typedef typename VecType<F, U>::type V;
        constexpr int UPP = ND / U;                            // units per point
        const V* gp = reinterpret_cast<const V*>(prm.pol + tile0 * ND);
        const V* gm = reinterpret_cast<const V*>(prm.mom + tile0 * ND);
        const int total = valid * UPP;
        for (int g = threadIdx.x; g < total; g += 32 * W) {
            const int p = g / UPP, q = g - p * UPP;
            V* r = reinterpret_cast<V*>(vec + (size_t)p * C::VSTRIDE);
            r[q] = load_unit<F>(gp[g]);
            if (q < M * D / U) r[(C::PS0 + 1) * D / U + q] = load_unit<F>(gm[g]);         // k_n is never used
        }
        if (threadIdx.x < TP) stat[threadIdx.x] = 0;
    }
    __syncthreads();

    E* recf = vec + (size_t)point * C::VSTRIDE;               // the point's record, all components
    E* rec = recf + half * DL;                                // ... this lane's components
    E* sc = scal + point;

    // ---- a1: doubled prefix sums PS2_c and the single-gluon U = V = 2 k_i . eps_i ------------------
    if (warp == 0) {
        E run[DL];
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) run[mu] = F::ezero();
        st_vec<F, DL>(rec + C::PS0 * D, run);
#pragma unroll 1
        for (int c = 1; c <= M; ++c) {
            E k[DL], e[DL];
            ld_vec<F, DL>(rec + (C::PS0 + c) * D, k);
            ld_vec<F, DL>(rec + (c - 1) * D, e);
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) k[mu] = F::dbl(k[mu]);
            const E u = F::neg(split_dot_neg<F, DL, TP>(t0, k, e));                  // 2 k.eps
            sc[(C::SC_U + c - 1) * TP] = u;
            sc[(C::SC_V + c - 1) * TP] = u;
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) run[mu] = F::add(run[mu], k[mu]);
            st_vec<F, DL>(rec + (C::PS0 + c) * D, run);
            if (prm.currents && live) {
                E* dst = prm.currents + (pt * M * M + (long long)(c - 1) * M + (c - 1)) * D + half * DL;
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) dst[mu] = F::canon(e[mu]);
            }
        }
    }
    __syncthreads();

    // ---- a2 + a3: invariants and propagators.  The R proper ranges are dealt round-robin to the
    //      W*S half-warps (each lane works on whole vectors here); every half-warp batch-inverts
    //      its own share with Montgomery's trick.
    {
        constexpr int VW = W * S;
        const int vw = warp * S + half;
        E* Wt = sc + C::SC_W * TP;
        uint32_t status = 0;
#pragma unroll 1
        for (int r = vw; r < C::R; r += VW) {
            int L = 2, i = r;
            while (i >= M - L + 1) { i -= M - L + 1; ++L; }
            E lo[D], hi[D], x[D];
            ld_vec<F, D>(recf + (C::PS0 + i) * D, lo);
            ld_vec<F, D>(recf + (C::PS0 + i + L) * D, hi);
#pragma unroll
            for (int mu = 0; mu < D; ++mu) x[mu] = F::sub(hi[mu], lo[mu]);
            const A ns = dot_neg<F, D>(F::neg(x[0]), x, x);                  // -(2P).(2P)
            Wt[r * TP] = F::canon(F::neg(F::reduce(ns)));
        }
        if constexpr (F::kExact) {
            E* tmp = sc + (C::SC_U + N) * TP;
            E c = F::one();
#pragma unroll 1
            for (int r = vw; r < C::R; r += VW) {
                tmp[r * TP] = c;
                const E s = Wt[r * TP];
                const bool z = F::is_zero(s);
                if (z) status |= 1u;
                c = F::mul(c, z ? F::one() : s);
            }
            E u = F::inv(c);
            u = F::dbl(F::dbl(u));
            int rl = vw + ((C::R - 1 - vw) / VW) * VW;                      // last r of this half-warp
            if (vw >= C::R) rl = -1;
#pragma unroll 1
            for (int r = rl; r >= 0; r -= VW) {
                const E s = Wt[r * TP];
                const bool z = F::is_zero(s);
                Wt[r * TP] = z ? F::ezero() : F::mul(u, tmp[r * TP]);
                u = F::mul(u, z ? F::one() : s);
            }
        } else {
#pragma unroll 1
            for (int r = vw; r < C::R; r += VW) {
                const E s = Wt[r * TP];
                if (F::is_zero(s)) status |= 1u;
                Wt[r * TP] = F::dbl(F::dbl(F::inv(s)));
            }
        }
        if (prm.status && status) atomicOr(&stat[point], status);
    }
    __syncthreads();
    if (prm.status && warp == 0 && half == 0 && live) prm.status[pt] = stat[point];

}

template <class F, int N, int D, int W, int S>
__global__ void __launch_bounds__(32 * W) bg_split_kernel(const TileParams<typename F::E> prm)
{
    typedef TileCfg<F, N, D, W> C;
    typedef SplitCfg<F, N, D, W, S> SC;
    typedef typename F::E E;
    typedef typename F::A A;
    constexpr int M = C::M, U = C::U, ND = N * D, TP = SC::TP, DL = SC::DL;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    E* vec = reinterpret_cast<E*>(smem_raw);                  // [TP][VSTRIDE]
    E* scal = vec + TP * C::VSTRIDE;                          // [NSCAL][TP]
    uint32_t* stat = reinterpret_cast<uint32_t*>(scal + TP * C::NSCAL);
    const TileProgram<N, W>& tb = c_split_program<F, N, D, W, S>;

    const int lane = threadIdx.x & 31, warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
    const int point = lane & (TP - 1), half = lane / TP;
    const bool t0 = half == 0;                                 // this lane owns the time component
    const long long tile0 = (long long)blockIdx.x * TP;
    const int valid = (int)min((long long)TP, prm.batch - tile0);
    const long long pt = tile0 + point;
    const bool live = point < valid;

    split_setup<F, N, D, W, S>(vec, scal, stat, prm, warp, point, half, t0, tile0, valid, pt, live);
    E* rec = vec + (size_t)point * C::VSTRIDE + half * DL;   // this lane's components of the point's record
    E* sc = scal + point;

    // ---- a4-a6: level sweep L = 2..m (Eq.(6)), amplitude, store ----------------------
#pragma unroll 1
    for (int L = 2; L <= M; ++L) {
        // phase A: this warp's chunk of the level's splittings
        const int ibeg = tb.beg[L][warp], iend = tb.beg[L][warp + 1];
        A acc[DL];
        E a[DL], x2[DL];
        E hsum = F::ezero();
        int room = 0;
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) { acc[mu] = F::zero(); a[mu] = F::ezero(); x2[mu] = F::ezero(); }
#pragma unroll 1
        for (int it = ibeg; it < iend; ++it) {
            const uint32_t fl = tb.flags[it];
            const TileOff o = tb.off[it];
            const char* recb = reinterpret_cast<const char*>(rec);
            const char* scb = reinterpret_cast<const char*>(sc);
            if (fl & IT_SEG_START) {
                const uint32_t sg = tb.seg[it];
                E l[DL], h[DL];
                ld_vec<F, DL>(rec + (C::PS0 + (sg & 255)) * D, l);
                ld_vec<F, DL>(rec + (C::PS0 + (sg >> 8 & 255)) * D, h);
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) x2[mu] = F::sub(l[mu], h[mu]);
                x2[0] = cneg(x2[0], t0);                             // 2 * covariant P_{i,j}
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) acc[mu] = F::zero();
                hsum = F::ezero();
                room = F::kCap0;
            }
            if (fl & IT_LOAD_A) ld_vec<F, DL>(reinterpret_cast<const E*>(recb + o.a), a);
            if (!(fl & IT_KIND4)) {
                // ---- 3-gluon split (i..k | k+1..j) -------------------------------------------------
                E b[DL], s[DL];
                ld_vec<F, DL>(reinterpret_cast<const E*>(recb + o.b), b);
                ld_vec<F, DL>(reinterpret_cast<const E*>(recb + o.c), s);
                const E ua = *reinterpret_cast<const E*>(scb + (o.uv & 0xffffu));
                const E vb = *reinterpret_cast<const E*>(scb + (o.uv >> 16));
                const E h = F::neg(split_dot_neg<F, DL, TP>(t0, a, b));           // A.B
                const E xa = split_dot_plain<F, DL, TP>(x2, a);                   // 2 X.A
                const E xb = split_dot_plain<F, DL, TP>(x2, b);                   // 2 X.B
                const E cb = F::sub(xa, ua);
                const E ca = F::sub(vb, xb);
                hsum = F::add(hsum, h);
                if (room < 2) {
#pragma unroll
                    for (int mu = 0; mu < DL; ++mu) acc[mu] = F::relief(acc[mu]);
                    room = F::kCapR;
                }
                room -= 2;
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) {
                    acc[mu] = F::mad(h, s[mu], acc[mu]);
                    acc[mu] = F::mad(cb, b[mu], acc[mu]);
                }
                if (room < 1) {
#pragma unroll
                    for (int mu = 0; mu < DL; ++mu) acc[mu] = F::relief(acc[mu]);
                    room = F::kCapR;
                }
                room -= 1;
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) acc[mu] = F::mad(ca, a[mu], acc[mu]);
            } else {
                // ---- 4-gluon split (i..k | k+1..l | l+1..j): 2 (A.C) J(k+1..l) ------------------------
                E bm[DL], c[DL];
                ld_vec<F, DL>(reinterpret_cast<const E*>(recb + o.b), bm);
                ld_vec<F, DL>(reinterpret_cast<const E*>(recb + o.c), c);
                const E cc = F::neg(F::dbl(split_dot_neg<F, DL, TP>(t0, a, c)));      // 2 A.C
                if (room < 1) {
#pragma unroll
                    for (int mu = 0; mu < DL; ++mu) acc[mu] = F::relief(acc[mu]);
                    room = F::kCapR;
                }
                room -= 1;
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) acc[mu] = F::mad(cc, bm[mu], acc[mu]);
            }
            if (fl & IT_SEG_END) {
                const uint32_t sg = tb.seg[it];
                if (fl & IT_COMPLETE) {
                    split_finish<F, N, D, W, S>(rec, sc, acc, hsum, sg >> 16 & 255, sg & 255, sg >> 8 & 255, L == M,
                                                t0, half, prm, pt, live);
                } else {
                    E* scr = sc + (C::SC_SCR + (sg >> 24) * (D + 1) + half * DL) * TP;
#pragma unroll
                    for (int mu = 0; mu < DL; ++mu) scr[mu * TP] = F::reduce(acc[mu]);
                    sc[(C::SC_SCR + (sg >> 24) * (D + 1) + D) * TP] = hsum;
                }
            }
        }
        // phase B: currents whose splittings were shared between warps
        const int nj = tb.njobs[L];
        if (nj) {
            __syncthreads();
#pragma unroll 1
            for (int j = warp; j < nj; j += W) {
                uint32_t mask = tb.job_mask[L][j];
                const uint32_t wy = tb.job_seg[L][j];
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) acc[mu] = F::zero();
                hsum = F::ezero();
                while (mask) {
                    const int slot = __ffs(mask) - 1;
                    mask &= mask - 1;
                    const E* scr = sc + (C::SC_SCR + slot * (D + 1) + half * DL) * TP;
#pragma unroll
                    for (int mu = 0; mu < DL; ++mu) acc[mu] = F::accumulate(acc[mu], scr[mu * TP]);
                    hsum = F::add(hsum, sc[(C::SC_SCR + slot * (D + 1) + D) * TP]);
                }
                split_finish<F, N, D, W, S>(rec, sc, acc, hsum, wy >> 16 & 255, wy & 255, wy >> 8 & 255, L == M,
                                            t0, half, prm, pt, live);
            }
        }
        if (L < M) __syncthreads();
    }
}

}  // namespace bg
