// bg_tile.cuh -- shared-memory layout of a tile of points and the per-tile setup stages (SURVEY.md
// 8(a) rows a0-a3) of the tiled Berends-Giele kernel (bg_unit.cuh).
//
// Mapping: a thread block owns one TILE of TP = 32/S phase-space points and has W
// warps.  With S = 1, lane l of every warp works on point l; with S = 2 the lanes (l, l + 16) of
// every warp share point l and each owns DL = D/2 of the d vector components (for records too
// large for 32 points per SM: complex128 at n = 12 needs 11 KB per point).  Arithmetic and
// control flow are uniform across a warp and every shared-memory access is conflict-free by
// construction (per-point vector records with an odd stride; scalar tables [index][point]).
//
// Per point the tile holds
//   vector record:  rows [0,n)        eps_1..eps_n of the CURRENT state configuration
//                   rows [n, n+R)     multi-gluon currents J(i..j), level-major, top excluded
//                   rows PS0 + c      doubled prefix sums PS2_c = 2 (k_1+..+k_c), c = 0..m
//                                     (Eq.(7))
//   scalar tables:  U, V per row      U = 2 P.J + S,  V = 2 P.J - S   (P own momentum; V = U for single gluons)
//                   1/P^2 per proper multi-gluon range (batch-inverted), parked in the range's U slot
//                   scratch           partial sums of currents shared between warps
//
// PS2, Wt and the status word depend on the momenta only: with S_c > 1 state configurations per
// momentum point (Eq.(4): "the state sum runs over all D_s-dimensional particle
// states") they are formed ONCE per tile and the level sweep is repeated per configuration.
#pragma once
#include "bg_common.cuh"
#include "bg_schedule.cuh"

namespace bg {

template <class F, int N, int D, int W, int S, bool KW>
struct TileCfg {
    typedef typename F::E E;
    static_assert(S == 1 || S == 2, "one or two lanes per point");
    static_assert(D % S == 0, "two lanes per point need an even d");
    static constexpr int M = N - 1;
    static constexpr int TP = 32 / S;                         // points per tile
    static constexpr int DL = D / S;                          // vector components per lane
    static constexpr int U = VecWidth<F, D>::value;           // elements per vector unit
    static constexpr int R = M * (M - 1) / 2 - 1;             // proper multi-gluon ranges
    static constexpr int J_ROWS = N + R;
    static constexpr int PS0 = J_ROWS;                        // PS2 rows 0..M
    static constexpr int VEC_ROWS = J_ROWS + M + 1;
    static constexpr int VEC_ELEMS = VEC_ROWS * D;
    static constexpr int VSTRIDE = (VEC_ELEMS / U % 2 == 1 ? VEC_ELEMS / U : VEC_ELEMS / U + 1) * U;
    // scalar tables [index][point]: U per row; V per multi-gluon row (the single-gluon rows have V = U);
    // 1/P^2 of a proper range lives in the U slot of its current until the current is finished (the finish
    // reads it, then writes U); scratch slots for the partial sums of currents shared between warps
    // (KW: a table of its own instead -- with several state configurations per point the propagators outlive a sweep)
    static constexpr int SC_U = 0, SC_V = J_ROWS, SC_W = KW ? J_ROWS + R : SC_U + N, SC_SCR = J_ROWS + R + (KW ? R : 0);
    __host__ __device__ static constexpr int v_index(int row) { return row < N ? SC_U + row : SC_V + row - N; }
    static constexpr int NSLOTS = LevelProgramOf<N, W>::value.nslots;
    static constexpr int NSCAL = SC_SCR + NSLOTS * (D + 1);
    static constexpr int THREADS = 32 * W;
    // + the status word per point and one "parked" flag per (scratch slot, lane)
    static constexpr size_t SMEM_BYTES = (size_t)TP * (VSTRIDE + NSCAL) * sizeof(E) + (TP + 32 * NSLOTS) * sizeof(uint32_t);
    // resident blocks per SM that shared memory allows (228 KB per SM, 1 KB reserved per block): the register
    // budget of the kernel is set so that registers do not lower it (__launch_bounds__ in bg_unit.cuh)
    static constexpr int SMEM_BLOCKS = (int)(233472 / (SMEM_BYTES + 1024)) < 1 ? 1 : (int)(233472 / (SMEM_BYTES + 1024));
    static constexpr int WARP_BLOCKS = 64 / W;                 // 64 resident warps per SM
    static constexpr int MIN_BLOCKS = SMEM_BLOCKS < WARP_BLOCKS ? (SMEM_BLOCKS > 16 ? 16 : SMEM_BLOCKS)
                                                                : (WARP_BLOCKS > 16 ? 16 : WARP_BLOCKS);
};

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

// the lane's view of its tile
template <class F, int N, int D, int W, int S, bool KW>
struct TileLane {
    typedef TileCfg<F, N, D, W, S, KW> C;
    typedef typename F::E E;
    E* vec;               // [TP][VSTRIDE]
    E* scal;              // [NSCAL][TP]
    uint32_t* stat;       // [TP], then the parked flags [NSLOTS][32]
    int warp, point, half, mu0, valid;
    long long tile0, pt;  // first point of the tile, this lane's point (index within the prime's batch)
    long long q;          // prime index (blockIdx.y)
    bool live;
    __device__ __forceinline__ E* recf() const { return vec + (size_t)point * C::VSTRIDE; }   // all components
    __device__ __forceinline__ E* rec() const { return recf() + mu0; }                        // this lane's components
    __device__ __forceinline__ E* sc() const { return scal + point; }
};

// a0: stage rows of the tile's points from global memory (coalesced, one vector unit per thread and
// step).  src: first element of point tile0's block; a point's block is ND elements, consecutive
// points are `pstride` elements apart; the first ROWS rows go to record rows [ROW0, ROW0 + ROWS).
// perm: NULL, or the colour ordering (Eq.(5)): record row ROW0 + i receives the caller's row perm[i].
template <class F, int N, int D, int W, int S, bool KW, int ROW0, int ROWS>
__device__ __forceinline__ void tile_stage(const F& f, const TileLane<F, N, D, W, S, KW>& t, const typename F::E* src,
                                           long long pstride, const unsigned char* __restrict__ perm)
{
    typedef TileCfg<F, N, D, W, S, KW> C;
    typedef typename VecType<F, C::U>::type V;
    constexpr int U = C::U, row0 = ROW0;
    constexpr int upp = ROWS * D / U;                           // units per point
    constexpr int upr = D / U;                                  // units per row
    const int total = t.valid * upp;
    if (perm == nullptr) {
        // Thread tid moves the units g = tid + j THREADS, j = 0..NIT-1.  (point, unit-in-point) and both
        // addresses advance incrementally (no division, no 64-bit multiply per unit), and ALL loads of
        // a thread are issued before the first store: one global-memory latency per stage instead of
        // one per batch of four (the staging loops were 9 % of the instructions and the
        // long-scoreboard stall of the round-2 profile).
        constexpr int T = 32 * W;
        constexpr int NIT = (C::TP * upp + T - 1) / T;
        constexpr int dp = T / upp, du = T % upp;               // advance of (point, unit) per step
        constexpr int VS = C::VSTRIDE / U;                      // record stride in units
        const int ps = (int)(pstride / U);                      // source stride in units
        const int p0 = threadIdx.x / upp, u0 = threadIdx.x - p0 * upp;
        constexpr int CHUNK = 24 / (int)(sizeof(V) / 4) > 0 ? 24 / (int)(sizeof(V) / 4) : 1;   // <= 24 registers in flight
        const V* s = reinterpret_cast<const V*>(src) + (long long)p0 * ps + u0;
        V* r = reinterpret_cast<V*>(t.vec) + p0 * VS + row0 * D / U + u0;
        int us = u0, ur = u0, gs = threadIdx.x, gr = threadIdx.x;
#pragma unroll
        for (int j0 = 0; j0 < NIT; j0 += CHUNK) {
            V buf[CHUNK];
#pragma unroll
            for (int j = 0; j < CHUNK; ++j) {
                if (j0 + j < NIT) {
                    if (gs < total) buf[j] = __ldg(s);
                    gs += T;
                    us += du;
                    s += dp * ps + du;
                    if (du != 0 && us >= upp) { us -= upp; s += ps - upp; }
                }
            }
#pragma unroll
            for (int j = 0; j < CHUNK; ++j) {
                if (j0 + j < NIT) {
                    if (gr < total) *r = load_unit<F>(f, buf[j]);
                    gr += T;
                    ur += du;
                    r += dp * VS + du;
                    if (du != 0 && ur >= upp) { ur -= upp; r += VS - upp; }
                }
            }
        }
    } else {
#pragma unroll 2
        for (int g = threadIdx.x; g < total; g += 32 * W) {
            const int p = g / upp, u = g - p * upp, row = u / upr, c = u - row * upr;
            V* r = reinterpret_cast<V*>(t.vec + (size_t)p * C::VSTRIDE) + row0 * D / U;
            r[u] = load_unit<F>(f, __ldg(reinterpret_cast<const V*>(src + p * pstride) + min((int)__ldg(perm + row), N - 1) * upr + c));
        }
    }
}

// a1-a3, once per tile: prefix() forms the doubled prefix sums, propagators() the invariants, the
// batch-inverted propagators and the status word; each ends with a block barrier.  On entry the momenta
// k_1..k_m are parked in rows [PARK, PARK + m).  singles() (per state configuration) only needs the
// prefix sums, so the first configuration's runs between the two without a barrier of its own.
template <class F, int N, int D, int W, int S, bool KW>
struct TileSetup {
    typedef TileCfg<F, N, D, W, S, KW> C;
    typedef typename F::E E;
    typedef typename F::A A;
    static constexpr int M = C::M, DL = C::DL, TP = C::TP;
    // With several warps the momenta are parked in the rows of the multi-gluon currents (free until
    // the level sweep), so that the prefix sums can be formed by all warps at once without
    // overwriting their own input; otherwise in the PS2 rows themselves (running sum by warp 0).
    static constexpr bool kParPrefix = W > 1 && C::R >= M;
    static constexpr int PARK = kParPrefix ? N : C::PS0 + 1;

    __device__ __forceinline__ static void prefix(const F& f, const TileLane<F, N, D, W, S, KW>& t)
    {
        E* rec = t.rec();
        // ---- a1: doubled prefix sums PS2_c = 2 (k_1 + .. + k_c)  (Eq.(7)) ------------
        if constexpr (kParPrefix) {
            // row c is formed by warp (c-1) mod W from the parked momenta (same left-to-right order
            // of additions as the running sum, so the floating-point result is the same)
            if (t.warp == 0) {
                E z[DL];
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) z[mu] = f.ezero();
                st_vec<F, DL>(rec + C::PS0 * D, z);
            }
#pragma unroll 1
            for (int c = t.warp + 1; c <= M; c += W) {
                E run[DL], k[DL];
                ld_vec<F, DL>(rec + PARK * D, run);
#pragma unroll 1
                for (int l = 2; l <= c; ++l) {
                    ld_vec<F, DL>(rec + (PARK + l - 1) * D, k);
#pragma unroll
                    for (int mu = 0; mu < DL; ++mu) run[mu] = f.add(run[mu], k[mu]);
                }
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) run[mu] = f.dbl(run[mu]);
                st_vec<F, DL>(rec + (C::PS0 + c) * D, run);
            }
        } else if (t.warp == 0) {
            E run[DL];
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) run[mu] = f.ezero();
            st_vec<F, DL>(rec + C::PS0 * D, run);
#pragma unroll 1
            for (int c = 1; c <= M; ++c) {
                E k[DL];
                ld_vec<F, DL>(rec + (C::PS0 + c) * D, k);
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) run[mu] = f.add(run[mu], f.dbl(k[mu]));
                st_vec<F, DL>(rec + (C::PS0 + c) * D, run);
            }
        }
        __syncthreads();
    }

    // a2 + a3 (needs the prefix sums; ends with a block barrier)
    template <int MET>
    __device__ __forceinline__ static void propagators(const F& f, const TileLane<F, N, D, W, S, KW>& t,
                                                       uint32_t* status_out)
    {
        E* sc = t.sc();
        // ---- a2 + a3: invariants 4 P_{i,j}^2 and propagators 1/P^2 = 4/(4P^2).  The R proper ranges
        //      are dealt round-robin to the W*S (half-)warps, each lane working on whole vectors here;
        //      every (half-)warp batch-inverts its own share with Montgomery's trick: ONE field
        //      inversion per (half-)warp and point.
        {
            constexpr int VW = W * S;
            const int vw = t.warp * S + t.half;
            const E* recf = t.recf();
            E* Wt = sc + C::SC_W * TP;
            uint32_t status = 0;
#pragma unroll 1
            for (int r = vw; r < C::R; r += VW) {
                const uint32_t rg = c_tile_ranges<N>.lohi[r];
                E lo[D], hi[D], x[D], nx[D];
                ld_vec<F, D>(recf + (C::PS0 + (rg & 255u)) * D, lo);
                ld_vec<F, D>(recf + (C::PS0 + (rg >> 8)) * D, hi);
#pragma unroll
                for (int mu = 0; mu < D; ++mu) x[mu] = f.sub(hi[mu], lo[mu]);
                lower_neg<F, MET, D>(f, 0, x, nx);
                const A ns = dot_plain<F, D>(f, nx, x);                          // -(2P).(2P)
                Wt[r * TP] = f.canon(f.neg(f.reduce(ns)));
            }
            if constexpr (F::kExact) {
                // zero-safe (inv(0) := 0, bg.h); prefix products parked in the not-yet-used V slots
                // of the multi-gluon currents
                E* tmp = sc + C::SC_V * TP;
                E c = f.one();
#pragma unroll 1
                for (int r = vw; r < C::R; r += VW) {
                    tmp[r * TP] = c;
                    const E s = Wt[r * TP];
                    const bool z = f.is_zero(s);
                    if (z) status |= 1u;
                    c = f.mul(c, z ? f.one() : s);
                }
                E u = f.inv(c);
                u = f.neg(f.dbl(f.dbl(u)));                                     // the table holds -1/P^2 (bg_unit.cuh)
                int rl = vw + ((C::R - 1 - vw) / VW) * VW;                      // last r of this (half-)warp
                if (vw >= C::R) rl = -1;
#pragma unroll 1
                for (int r = rl; r >= 0; r -= VW) {
                    const E s = Wt[r * TP];
                    const bool z = f.is_zero(s);
                    Wt[r * TP] = z ? f.ezero() : f.mul(u, tmp[r * TP]);
                    u = f.mul(u, z ? f.one() : s);
                }
            } else {
#pragma unroll 1
                for (int r = vw; r < C::R; r += VW) {
                    const E s = Wt[r * TP];
                    if (f.is_zero(s)) status |= 1u;
                    Wt[r * TP] = f.neg(f.dbl(f.dbl(f.inv(s))));
                }
            }
            if (status_out && status) atomicOr(&t.stat[t.point], status);
        }
        __syncthreads();
        if (status_out && t.warp == 0 && t.half == 0 && t.live) status_out[t.pt] = t.stat[t.point];
    }

    // per state configuration: the single-gluon U = V = 2 k_c . eps_c (zero for transverse states;
    // kept for any input, R4), 2 k_c = PS2_c - PS2_{c-1}.  No barrier inside.
    template <int MET>
    __device__ __forceinline__ static void singles(const F& f, const TileLane<F, N, D, W, S, KW>& t,
                                                   typename F::E* currents)
    {
        E* rec = t.rec();
        E* sc = t.sc();
#pragma unroll 1
        for (int c = t.warp + 1; c <= M; c += W) {
            E lo[DL], hi[DL], k2[DL], e[DL];
            ld_vec<F, DL>(rec + (C::PS0 + c - 1) * D, lo);
            ld_vec<F, DL>(rec + (C::PS0 + c) * D, hi);
            ld_vec<F, DL>(rec + (c - 1) * D, e);
            lower_diff<F, MET, DL>(f, t.mu0, hi, lo, k2);                       // 2 * covariant k_c
            const E u = lane_sum<F, S, TP>(f, f.reduce(dot_plain<F, DL>(f, k2, e)));   // 2 k.eps
            sc[(C::SC_U + c - 1) * TP] = u;
            if (currents && t.live) {
                E* dst = currents + (t.pt * M * M + (long long)(c - 1) * M + (c - 1)) * D + t.mu0;
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) dst[mu] = f.to_output(e[mu]);
            }
        }
    }
};

}  // namespace bg
