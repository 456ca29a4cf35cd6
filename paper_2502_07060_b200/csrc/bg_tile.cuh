// bg_tile.cuh -- the Berends-Giele level sweep for compile-time (n, d): the fast path.
//
// Mapping: a thread block owns one TILE of 32 phase-space points and has W
// warps.  In every warp, lane l works on point l of the tile, so all arithmetic and all
// control flow are uniform across a warp and every shared-memory access is conflict-free
// by construction (per-point vector records with an odd stride; scalar tables [index][lane]).
// The W warps split the WORK of a level: the flattened list of splittings of the level
// (bg_tables.cuh) is cut into W chunks of equal weight.  A current whose splittings all
// fall into one chunk is finished by that warp; one that straddles a chunk boundary has its
// partial sums parked in shared scratch and is finished by a gather job after a barrier.
//
// The code is a short loop over table items (read from constant memory with warp-uniform
// indices); nothing is unrolled over splittings, so the kernel stays resident in the
// instruction cache.
//
// Per point the tile holds
//   vector record:  rows [0,n)        eps_1..eps_n verbatim from the caller's array
//                   rows [n, n+R)     multi-gluon currents J(i..j), level-major, top excluded
//                   rows PS0 + c      doubled prefix sums PS2_c = 2 (k_1+..+k_c), c = 0..m
//                                     (Eq.(7))
//   scalar tables:  U, V per row      U = 2 P.J + S,  V = 2 P.J - S   (P own momentum)
//                   Wt per proper multi-gluon range: 1/P^2 (batch-inverted)
//                   scratch           partial sums of segments, 2 slots per warp
//
// Algebra (i-free V3, V4 of Eq.(7); DESIGN.md §6 "factored form"): for the
// current (i..j) with own momentum X = P_{i,j} and a split A = J(i..k), B = J(k+1..j):
//   bracket^mu = sum_k [ h_k PS2_k^mu + (2X.A - U_A) B^mu + (V_B - 2X.B) A^mu ]
//              - (sum_k h_k)/2 (PS2_{i-1} + PS2_j)^mu
//              + sum_{k<l} 2 (A_k . C_l) J(k+1..l)^mu ,        h_k = A.B
// Exact over F_p, hence bit-identical to the literal evaluation.
#pragma once
#include "bg_field.cuh"
#include "bg_recursion.cuh"   // ld_vec / st_vec / dot helpers, VecWidth
#include "bg_tables.cuh"

namespace bg {

template <class F, int N, int D, int W>
struct TileCfg {
    typedef typename F::E E;
    static constexpr int M = N - 1;
    static constexpr int U = VecWidth<F, D>::value;           // elements per vector unit
    static constexpr int R = M * (M - 1) / 2 - 1;             // proper multi-gluon ranges
    static constexpr int J_ROWS = N + R;
    static constexpr int PS0 = J_ROWS;                        // PS2 rows 0..M
    static constexpr int VEC_ROWS = J_ROWS + M + 1;
    static constexpr int VEC_ELEMS = VEC_ROWS * D;
    static constexpr int VSTRIDE = (VEC_ELEMS / U % 2 == 1 ? VEC_ELEMS / U : VEC_ELEMS / U + 1) * U;
    static constexpr int SC_U = 0, SC_V = J_ROWS, SC_W = 2 * J_ROWS, SC_SCR = 2 * J_ROWS + R;
    static constexpr int NSLOTS = 2 * W;
    static constexpr int NSCAL = SC_SCR + NSLOTS * (D + 1);
    static constexpr int THREADS = 32 * W;
    static constexpr size_t SMEM_BYTES = (size_t)32 * (VSTRIDE + NSCAL) * sizeof(E) + 32 * sizeof(uint32_t);
};

// the work lists of one (field, N, D, W) instance, in constant memory
template <class F, int N, int D, int W>
__constant__ TileProgram<N, W> c_tile_program = make_tile_program<N, W>(
    D * (int)sizeof(typename F::E), TileCfg<F, N, D, W>::PS0, TileCfg<F, N, D, W>::SC_U, TileCfg<F, N, D, W>::SC_V,
    32 * (int)sizeof(typename F::E));

// proper multi-gluon range r (level-major) -> lo | hi << 8 with P_{i,j} = PS_hi - PS_lo
template <int N>
struct TileRanges {
    uint16_t lohi[(N - 1) * (N - 2) / 2];
};
template <int N>
constexpr TileRanges<N> make_tile_ranges()
{
    TileRanges<N> t{};
    int r = 0;
    for (int L = 2; L <= N - 2; ++L)
        for (int i = 0; i + L <= N - 1; ++i) t.lohi[r++] = (uint16_t)(i | (i + L) << 8);
    return t;
}
template <int N>
__constant__ TileRanges<N> c_tile_ranges = make_tile_ranges<N>();

template <class E>
struct TileParams {
    const E* mom;         // [batch][n][D]
    const E* pol;         // [batch][n][D]
    E* out;               // [batch]
    E* currents;          // NULL or [batch][m][m][D]
    uint32_t* status;     // NULL or [batch]
    long long batch;
};

// Finish the current stored at `own` (P_{i,j} = (PS2_hi - PS2_lo)/2): boundary term of the
// (P-Q) sum, propagator, store, U and V; for the top current the amplitude instead.
template <class F, int N, int D, int W>
__device__ __forceinline__ void tile_finish(typename F::E* __restrict__ rec, typename F::E* __restrict__ sc,
                                            typename F::A (&acc)[D], typename F::E hsum, int own, int lo,
                                            int hi, bool top, const TileParams<typename F::E>& prm,
                                            long long pt, bool live)
{
    typedef TileCfg<F, N, D, W> C;
    typedef typename F::E E;
    typedef typename F::A A;
    E l[D], h[D];
    ld_vec<F, D>(rec + (C::PS0 + lo) * D, l);
    ld_vec<F, D>(rec + (C::PS0 + hi) * D, h);
    const E nhh = F::neg(F::mul(hsum, F::half()));               // -(sum_k h_k)/2
    if constexpr (F::kExact) {
        // one product per component: the two ALU instructions of the add are cheaper than a
        // second IMAD.WIDE (the multiplier pipe is the binding one)
#pragma unroll
        for (int mu = 0; mu < D; ++mu) {
            acc[mu] = F::relief(acc[mu]);
            acc[mu] = F::mad(nhh, F::add(l[mu], h[mu]), acc[mu]);
        }
    } else {
#pragma unroll
        for (int mu = 0; mu < D; ++mu) {
            acc[mu] = F::mad(nhh, l[mu], acc[mu]);
            acc[mu] = F::mad(nhh, h[mu], acc[mu]);
        }
    }
    E v[D];
    if (!top) {
        const E w = sc[(C::SC_W + own - N) * 32];
#pragma unroll
        for (int mu = 0; mu < D; ++mu) v[mu] = F::mul(F::reduce(acc[mu]), w);
        st_vec<F, D>(rec + own * D, v);
        E x2[D];
        x2[0] = F::sub(h[0], l[0]);
#pragma unroll
        for (int mu = 1; mu < D; ++mu) x2[mu] = F::sub(l[mu], h[mu]);
        const E c2 = F::reduce(dot_plain<F, D>(x2, v));          // 2 P_{i,j} . J(i..j)
        sc[(C::SC_U + own) * 32] = F::add(c2, hsum);
        sc[(C::SC_V + own) * 32] = F::sub(c2, hsum);
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
        constexpr int M = C::M;
        E* dst = prm.currents + (pt * M * M + (long long)lo * M + (hi - 1)) * D;
#pragma unroll
        for (int mu = 0; mu < D; ++mu) dst[mu] = F::canon(v[mu]);
    }
}

// a0-a3 for one tile: stage the inputs, doubled prefix sums, single-gluon U/V, invariants and
// batch-inverted propagators.  Ends with a block barrier; shared by bg_tile_kernel and
// bg_level_kernel (bg_level.cuh).
template <class F, int N, int D, int W>
__device__ __forceinline__ void tile_setup(typename F::E* __restrict__ vec, typename F::E* __restrict__ scal,
                                           uint32_t* __restrict__ stat, const TileParams<typename F::E>& prm,
                                           int lane, int warp, long long tile0, int valid, long long pt, bool live)
{
    typedef TileCfg<F, N, D, W> C;
    typedef typename F::E E;
    typedef typename F::A A;
    constexpr int M = C::M, U = C::U, ND = N * D;
    constexpr bool kParPrefix = W > 1 && C::R >= M;          // room to park the momenta in the multi-gluon rows
    // ---- a0: stage the tile (coalesced, one vector unit per thread and step) ---------------------
    {
        typedef typename VecType<F, U>::type V;
        constexpr int UPP = ND / U;                            // units per point
        const V* gp = reinterpret_cast<const V*>(prm.pol + tile0 * ND);
        const V* gm = reinterpret_cast<const V*>(prm.mom + tile0 * ND);
        const int total = valid * UPP;
#pragma unroll 4
        for (int g = threadIdx.x; g < total; g += 32 * W) {
            const int p = g / UPP, q = g - p * UPP;
            V* r = reinterpret_cast<V*>(vec + (size_t)p * C::VSTRIDE);
            r[q] = load_unit<F>(__ldg(gp + g));
            // k_n is never used.  With several warps the momenta are parked in the rows of the
            // multi-gluon currents (free until the level sweep), so that the prefix sums below can
            // be formed by all warps at once without overwriting their own input.
            if (q < M * D / U) r[(kParPrefix ? N : C::PS0 + 1) * D / U + q] = load_unit<F>(__ldg(gm + g));
        }
        if (warp == 0) stat[lane] = 0;
    }
    __syncthreads();

    E* rec = vec + (size_t)lane * C::VSTRIDE;
    E* sc = scal + lane;

    // ---- a1: doubled prefix sums PS2_c = 2 (k_1 + .. + k_c)  (Eq.(7)) and the
    //      single-gluon U = V = 2 k_i . eps_i  (zero for transverse states; kept for any input)
    if constexpr (kParPrefix) {
        // row c is formed by warp (c-1) mod W from the parked momenta (same left-to-right order
        // of additions as the running sum, so the floating-point result is the same)
        if (warp == 0) {
            E z[D];
#pragma unroll
            for (int mu = 0; mu < D; ++mu) z[mu] = F::ezero();
            st_vec<F, D>(rec + C::PS0 * D, z);
        }
#pragma unroll 1
        for (int c = warp + 1; c <= M; c += W) {
            E run[D], k[D], e[D];
            ld_vec<F, D>(rec + N * D, run);
#pragma unroll 1
            for (int l = 2; l <= c; ++l) {
                ld_vec<F, D>(rec + (N + l - 1) * D, k);
#pragma unroll
                for (int mu = 0; mu < D; ++mu) run[mu] = F::add(run[mu], k[mu]);
            }
            ld_vec<F, D>(rec + (N + c - 1) * D, k);
            ld_vec<F, D>(rec + (c - 1) * D, e);
#pragma unroll
            for (int mu = 0; mu < D; ++mu) { k[mu] = F::dbl(k[mu]); run[mu] = F::dbl(run[mu]); }
            const E u = F::neg(F::reduce(dot_neg<F, D>(F::neg(k[0]), k, e)));       // 2 k.eps
            sc[(C::SC_U + c - 1) * 32] = u;
            sc[(C::SC_V + c - 1) * 32] = u;
            st_vec<F, D>(rec + (C::PS0 + c) * D, run);
            if (prm.currents && live) {
                E* dst = prm.currents + (pt * M * M + (long long)(c - 1) * M + (c - 1)) * D;
#pragma unroll
                for (int mu = 0; mu < D; ++mu) dst[mu] = F::canon(e[mu]);
            }
        }
    } else if (warp == 0) {
        E run[D];
#pragma unroll
        for (int mu = 0; mu < D; ++mu) run[mu] = F::ezero();
        st_vec<F, D>(rec + C::PS0 * D, run);
#pragma unroll 1
        for (int c = 1; c <= M; ++c) {
            E k[D], e[D];
            ld_vec<F, D>(rec + (C::PS0 + c) * D, k);
            ld_vec<F, D>(rec + (c - 1) * D, e);
#pragma unroll
            for (int mu = 0; mu < D; ++mu) k[mu] = F::dbl(k[mu]);
            const E u = F::neg(F::reduce(dot_neg<F, D>(F::neg(k[0]), k, e)));       // 2 k.eps
            sc[(C::SC_U + c - 1) * 32] = u;
            sc[(C::SC_V + c - 1) * 32] = u;
#pragma unroll
            for (int mu = 0; mu < D; ++mu) run[mu] = F::add(run[mu], k[mu]);
            st_vec<F, D>(rec + (C::PS0 + c) * D, run);
            if (prm.currents && live) {
                E* dst = prm.currents + (pt * M * M + (long long)(c - 1) * M + (c - 1)) * D;
#pragma unroll
                for (int mu = 0; mu < D; ++mu) dst[mu] = F::canon(e[mu]);
            }
        }
    }
    __syncthreads();

    // ---- a2 + a3: invariants 4 P_{i,j}^2 and propagators 1/P^2 = 4/(4P^2).  The R proper ranges
    //      are dealt round-robin to the warps (r = warp, warp+W, ..); every warp batch-inverts its
    //      own share with Montgomery's trick: ONE field inversion per warp and point.
    {
        E* Wt = sc + C::SC_W * 32;
        uint32_t status = 0;
#pragma unroll 1
        for (int r = warp; r < C::R; r += W) {
            // range r -> (i, i+L) from the constant table: level-major, level L has M-L+1 ranges
            const uint32_t rg = c_tile_ranges<N>.lohi[r];
            E lo[D], hi[D], x[D];
            ld_vec<F, D>(rec + (C::PS0 + (rg & 255u)) * D, lo);
            ld_vec<F, D>(rec + (C::PS0 + (rg >> 8)) * D, hi);
#pragma unroll
            for (int mu = 0; mu < D; ++mu) x[mu] = F::sub(hi[mu], lo[mu]);
            const A ns = dot_neg<F, D>(F::neg(x[0]), x, x);                  // -(2P).(2P)
            Wt[r * 32] = F::canon(F::neg(F::reduce(ns)));
        }
        if constexpr (F::kExact) {
            // zero-safe (inv(0) := 0, bg.h); prefix products parked in the not-yet-used U slots
            // of the multi-gluon currents
            E* tmp = sc + (C::SC_U + N) * 32;
            E c = F::one();
#pragma unroll 1
            for (int r = warp; r < C::R; r += W) {
                tmp[r * 32] = c;
                const E s = Wt[r * 32];
                const bool z = F::is_zero(s);
                if (z) status |= 1u;
                c = F::mul(c, z ? F::one() : s);
            }
            E u = F::inv(c);
            u = F::dbl(F::dbl(u));
            int rl = warp + ((C::R - 1 - warp) / W) * W;                    // last r of this warp
            if (warp >= C::R) rl = -1;
#pragma unroll 1
            for (int r = rl; r >= 0; r -= W) {
                const E s = Wt[r * 32];
                const bool z = F::is_zero(s);
                Wt[r * 32] = z ? F::ezero() : F::mul(u, tmp[r * 32]);
                u = F::mul(u, z ? F::one() : s);
            }
        } else {
#pragma unroll 1
            for (int r = warp; r < C::R; r += W) {
                const E s = Wt[r * 32];
                if (F::is_zero(s)) status |= 1u;
                Wt[r * 32] = F::dbl(F::dbl(F::inv(s)));
            }
        }
        if (prm.status && status) atomicOr(&stat[lane], status);
    }
    __syncthreads();
    if (prm.status && warp == 0 && live) prm.status[pt] = stat[lane];

}

template <class F, int N, int D, int W>
__global__ void __launch_bounds__(32 * W) bg_tile_kernel(const TileParams<typename F::E> prm)
{
    typedef TileCfg<F, N, D, W> C;
    typedef typename F::E E;
    typedef typename F::A A;
    constexpr int M = C::M, U = C::U, ND = N * D;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    E* vec = reinterpret_cast<E*>(smem_raw);                  // [32][VSTRIDE]
    E* scal = vec + 32 * C::VSTRIDE;                          // [NSCAL][32]
    uint32_t* stat = reinterpret_cast<uint32_t*>(scal + 32 * C::NSCAL);
    const TileProgram<N, W>& tb = c_tile_program<F, N, D, W>;

    // the warp index, broadcast from lane 0 so that everything derived from it (chunk bounds,
    // item words, branch conditions) is compiled as warp-uniform
    const int lane = threadIdx.x & 31, warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
    const long long tile0 = (long long)blockIdx.x * 32;
    const int valid = (int)min(32LL, prm.batch - tile0);
    const long long pt = tile0 + lane;
    const bool live = lane < valid;

    tile_setup<F, N, D, W>(vec, scal, stat, prm, lane, warp, tile0, valid, pt, live);
    E* rec = vec + (size_t)lane * C::VSTRIDE;
    E* sc = scal + lane;

    // ---- a4-a6: level sweep L = 2..m (Eq.(6)), amplitude, store ----------------------
#pragma unroll 1
    for (int L = 2; L <= M; ++L) {
        // phase A: this warp's chunk of the level's splittings
        const int ibeg = tb.beg[L][warp], iend = tb.beg[L][warp + 1];
        A acc[D];
        E a[D], x2[D];
        E hsum = F::ezero(), na0 = F::ezero();
        int room = 0;
#pragma unroll
        for (int mu = 0; mu < D; ++mu) { acc[mu] = F::zero(); a[mu] = F::ezero(); x2[mu] = F::ezero(); }
#pragma unroll 1
        for (int it = ibeg; it < iend; ++it) {
            const uint32_t fl = tb.flags[it];
            const TileOff o = tb.off[it];
            const char* recb = reinterpret_cast<const char*>(rec);
            const char* scb = reinterpret_cast<const char*>(sc);
            if (fl & IT_SEG_START) {
                const uint32_t sg = tb.seg[it];
                E l[D], h[D];
                ld_vec<F, D>(rec + (C::PS0 + (sg & 255)) * D, l);
                ld_vec<F, D>(rec + (C::PS0 + (sg >> 8 & 255)) * D, h);
                x2[0] = F::sub(h[0], l[0]);                          // 2 * covariant P_{i,j}
#pragma unroll
                for (int mu = 1; mu < D; ++mu) x2[mu] = F::sub(l[mu], h[mu]);
#pragma unroll
                for (int mu = 0; mu < D; ++mu) acc[mu] = F::zero();
                hsum = F::ezero();
                room = F::kCap0;
            }
            if (fl & IT_LOAD_A) {
                ld_vec<F, D>(reinterpret_cast<const E*>(recb + o.a), a);
                na0 = F::neg(a[0]);
            }
            if (!(fl & IT_KIND4)) {
                // ---- 3-gluon split (i..k | k+1..j) -------------------------------------------------
                E b[D], s[D];
                ld_vec<F, D>(reinterpret_cast<const E*>(recb + o.b), b);
                ld_vec<F, D>(reinterpret_cast<const E*>(recb + o.c), s);
                const E ua = *reinterpret_cast<const E*>(scb + (o.uv & 0xffffu));
                const E vb = *reinterpret_cast<const E*>(scb + (o.uv >> 16));
                const E h = F::neg(F::reduce(dot_neg<F, D>(na0, a, b)));          // A.B
                const E xa = F::reduce(dot_plain<F, D>(x2, a));                   // 2 X.A
                const E xb = F::reduce(dot_plain<F, D>(x2, b));                   // 2 X.B
                const E cb = F::sub(xa, ua);
                const E ca = F::sub(vb, xb);
                hsum = F::add(hsum, h);
                if (room < 2) {
#pragma unroll
                    for (int mu = 0; mu < D; ++mu) acc[mu] = F::relief(acc[mu]);
                    room = F::kCapR;
                }
                room -= 2;
#pragma unroll
                for (int mu = 0; mu < D; ++mu) {
                    acc[mu] = F::mad(h, s[mu], acc[mu]);
                    acc[mu] = F::mad(cb, b[mu], acc[mu]);
                }
                if (room < 1) {
#pragma unroll
                    for (int mu = 0; mu < D; ++mu) acc[mu] = F::relief(acc[mu]);
                    room = F::kCapR;
                }
                room -= 1;
#pragma unroll
                for (int mu = 0; mu < D; ++mu) acc[mu] = F::mad(ca, a[mu], acc[mu]);
            } else {
                // ---- 4-gluon split (i..k | k+1..l | l+1..j): 2 (A.C) J(k+1..l) ------------------------
                E bm[D], c[D];
                ld_vec<F, D>(reinterpret_cast<const E*>(recb + o.b), bm);
                ld_vec<F, D>(reinterpret_cast<const E*>(recb + o.c), c);
                const E cc = F::neg(F::dbl(F::reduce(dot_neg<F, D>(na0, a, c))));   // 2 A.C
                if (room < 1) {
#pragma unroll
                    for (int mu = 0; mu < D; ++mu) acc[mu] = F::relief(acc[mu]);
                    room = F::kCapR;
                }
                room -= 1;
#pragma unroll
                for (int mu = 0; mu < D; ++mu) acc[mu] = F::mad(cc, bm[mu], acc[mu]);
            }
            if (fl & IT_SEG_END) {
                const uint32_t sg = tb.seg[it];
                if (fl & IT_COMPLETE) {
                    tile_finish<F, N, D, W>(rec, sc, acc, hsum, sg >> 16 & 255, sg & 255, sg >> 8 & 255, L == M,
                                            prm, pt, live);
                } else {
                    E* scr = sc + (C::SC_SCR + (sg >> 24) * (D + 1)) * 32;
#pragma unroll
                    for (int mu = 0; mu < D; ++mu) scr[mu * 32] = F::reduce(acc[mu]);
                    scr[D * 32] = hsum;
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
                for (int mu = 0; mu < D; ++mu) acc[mu] = F::zero();
                hsum = F::ezero();
                while (mask) {
                    const int slot = __ffs(mask) - 1;
                    mask &= mask - 1;
                    const E* scr = sc + (C::SC_SCR + slot * (D + 1)) * 32;
#pragma unroll
                    for (int mu = 0; mu < D; ++mu) acc[mu] = F::accumulate(acc[mu], scr[mu * 32]);
                    hsum = F::add(hsum, scr[D * 32]);
                }
                tile_finish<F, N, D, W>(rec, sc, acc, hsum, wy >> 16 & 255, wy & 255, wy >> 8 & 255, L == M, prm,
                                        pt, live);
            }
        }
        if (L < M) __syncthreads();
    }
}

}  // namespace bg
