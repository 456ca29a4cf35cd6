// bg_rt.cuh -- the tiled Berends-Giele kernel for a RUN-TIME number of gluons (compile-time d): SURVEY.md 8(a)
// rows a0-a6 in one launch for every shape without a compiled bg_unit_kernel instance.
//
// Same tile (32 / S points, W warps, per-point records with an odd stride, scalar tables [index][point]), same
// schedule (bg_schedule.cuh), same flat op program, same unit bodies, finish and sweep as bg_unit_kernel
// (bg_unit.cuh: unit_split3 / unit_body / unit_pair_body / unit_finish / unit_sweep_body, shared through the layout
// and program policies) -- but the layout and the ops are kernel ARGUMENTS: the host builds the schedule at the first
// call for a shape (bg_rt_host.cu) and every launch carries it in its parameter block (RtParams, bg_common.cuh: the
// constant bank, read with uniform loads like the compiled kernels' tables).  Only the per-tile setup (rows a0-a3) is
// restated here with run-time row counts.  The MULTI instantiation loops over K colour orderings and S state
// configurations per point like bg_unit_kernel's (a1-a3 once per ordering, the sweep once per configuration; its
// layout keeps -1/P^2 in a table of its own, because the propagators outlive a sweep); the plain one serves one
// of each.  Shapes whose 16-point tile does not fit shared memory run bg_general_kernel.
//
// Round 2 ran every such shape on bg_general_kernel (one thread per point, at most one warp per block: 0.12 of the
// multiplier peak at n = 13, d = 5 and n = 16, d = 4 against 0.6-0.7 for the compiled shapes).
#pragma once
#include "bg_unit.cuh"

namespace bg {

struct RtLay {
    RtLayout l;
    __device__ __forceinline__ int n() const { return l.n; }
    __device__ __forceinline__ static constexpr int sc_u() { return 0; }
    __device__ __forceinline__ int sc_v() const { return l.sc_v; }
    __device__ __forceinline__ int sc_w() const { return l.sc_w; }
    __device__ __forceinline__ int sc_scr() const { return l.sc_scr; }
};

struct RtProg {                                                 // the tables are a kernel parameter: constant bank
    typedef const FlatOp& Op;
    const RtTables& tab;
    __device__ __forceinline__ Op op(int k) const { return tab.ops[k]; }
    __device__ __forceinline__ const uint32_t* quad() const { return tab.quad; }
    __device__ __forceinline__ int beg(int w) const { return tab.beg[w]; }
};

struct RtLane {
    int mu0, half;
    bool live;
    long long pt;
};

// a0: stage `rows` rows of the tile's points into record rows [row0, row0 + rows), coalesced, one vector unit
// per thread and step.  perm: NULL, or the colour ordering (Eq.(5)): record row row0 + i receives the
// caller's row perm[i] (entries >= n are clamped, bg.h)
template <class F, int D, int W>
__device__ __forceinline__ void rt_stage(const F& f, typename F::E* vec, int vstride, int valid,
                                         const typename F::E* src, long long pstride, int row0, int rows,
                                         const unsigned char* __restrict__ perm = nullptr, int n = 0)
{
    constexpr int U = VecWidth<F, D>::value, upr = D / U;
    typedef typename VecType<F, U>::type V;
    const int upp = rows * upr, total = valid * upp;
    if (perm == nullptr) {
#pragma unroll 4
        for (int g = threadIdx.x; g < total; g += 32 * W) {
            const int p = g / upp, u = g - p * upp;
            V* r = reinterpret_cast<V*>(vec + (size_t)p * vstride) + row0 * upr;
            r[u] = load_unit<F>(f, __ldg(reinterpret_cast<const V*>(src + p * pstride) + u));
        }
    } else {
#pragma unroll 2
        for (int g = threadIdx.x; g < total; g += 32 * W) {
            const int p = g / upp, u = g - p * upp, row = u / upr, c = u - row * upr;
            V* r = reinterpret_cast<V*>(vec + (size_t)p * vstride) + row0 * upr;
            r[u] = load_unit<F>(f, __ldg(reinterpret_cast<const V*>(src + p * pstride) + min((int)__ldg(perm + row), n - 1) * upr + c));
        }
    }
}

template <class F, int MET, int D, int W, int S, bool MULTI>
__global__ void __launch_bounds__(32 * W) bg_rt_kernel(const __grid_constant__ RtParams<F> P)
{
    const BgParams<F>& prm = P.base;
    typedef typename F::E E;
    typedef typename F::A A;
    constexpr int TP = 32 / S, DL = D / S;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const F f(prm.fld, blockIdx.y);
    const RtLayout L = prm.rt;
    const int n = L.n, m = L.m, nd = n * D, PS0 = L.ps0;
    E* vec = reinterpret_cast<E*>(smem_raw);                   // [TP][vstride]
    E* scal = vec + (size_t)TP * L.vstride;                    // [nscal][TP]
    uint32_t* stat = reinterpret_cast<uint32_t*>(scal + (size_t)TP * L.nscal);   // [TP], then parked flags [nslots][32]
    const int lane = threadIdx.x & 31;
    const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
    const int point = S == 1 ? lane : lane & (TP - 1);
    RtLane t;
    t.half = S == 1 ? 0 : lane / TP;
    t.mu0 = S == 1 ? 0 : t.half * DL;
    const long long tile0 = (long long)blockIdx.x * TP;
    const int valid = (int)min((long long)TP, prm.batch - tile0);
    t.pt = tile0 + point;
    t.live = point < valid;
    const int states = MULTI ? prm.states : 1, n_ord = MULTI ? prm.n_orderings : 1;
    const long long pbase = (long long)blockIdx.y * prm.batch; // first point of this prime's arrays
    const E* gmom = prm.mom + (pbase + tile0) * nd;
    const E* gpol = prm.pol + (pbase + tile0) * states * nd;
    E* gout = prm.out + (pbase + t.pt) * n_ord * states;
    E* recf = vec + (size_t)point * L.vstride;                 // the point's record, all components
    E* rec = recf + t.mu0;                                     // this lane's components
    E* sc = scal + point;
    uint32_t* gstat = prm.status ? prm.status + pbase : nullptr;
    RtLay lay;
    lay.l = L;
    const RtProg prog{P.tab};

    // single-gluon U = V = 2 k_c . eps_c (zero for transverse states; kept for any input, R4)
    auto singles = [&]() {
#pragma unroll 1
        for (int c = warp + 1; c <= m; c += W) {
            E lo[DL], hi[DL], k2[DL], e[DL];
            ld_vec<F, DL>(rec + (PS0 + c - 1) * D, lo);
            ld_vec<F, DL>(rec + (PS0 + c) * D, hi);
            ld_vec<F, DL>(rec + (c - 1) * D, e);
            lower_diff<F, MET, DL>(f, t.mu0, hi, lo, k2);                               // 2 * covariant k_c
            sc[(c - 1) * TP] = lane_sum<F, S, TP>(f, f.reduce(dot_plain<F, DL>(f, k2, e)));
            if (prm.currents && t.live) {
                E* dst = prm.currents + (t.pt * m * m + (long long)(c - 1) * m + (c - 1)) * D + t.mu0;
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) dst[mu] = f.to_output(e[mu]);
            }
        }
    };

    if (warp == 0 && lane < TP) stat[lane] = 0;
#pragma unroll 1
    for (int sl = warp; sl < L.nslots; sl += W) stat[TP + 32 * sl + lane] = 0;

#pragma unroll 1
    for (int o = 0; o < n_ord; ++o, gout += states) {
    // colour ordering o (Eq.(5)): the inputs are re-staged in that order, everything below runs unchanged
    const unsigned char* perm = MULTI && prm.orderings ? prm.orderings + o * n : nullptr;
    if (MULTI && o > 0) __syncthreads();                       // the previous sweep is done with the record
    // ---- a0: momenta k_1..k_m into the PS2 rows 1..m (summed in place below), eps_1..eps_n into rows [0, n) ----
    rt_stage<F, D, W>(f, vec, L.vstride, valid, gmom, nd, PS0 + 1, m, perm, n);
    rt_stage<F, D, W>(f, vec, L.vstride, valid, gpol, (long long)states * nd, 0, n, perm, n);
    __syncthreads();

    // ---- a1: doubled prefix sums PS2_c = 2 (k_1 + .. + k_c)  (Eq.(7)), running sum by warp 0 ----
    if (warp == 0) {
        E run[DL];
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) run[mu] = f.ezero();
        st_vec<F, DL>(rec + PS0 * D, run);
#pragma unroll 1
        for (int c = 1; c <= m; ++c) {
            E k[DL];
            ld_vec<F, DL>(rec + (PS0 + c) * D, k);
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) run[mu] = f.add(run[mu], f.dbl(k[mu]));
            st_vec<F, DL>(rec + (PS0 + c) * D, run);
        }
    }
    __syncthreads();

    singles();                                                 // first state configuration

    // ---- a2 + a3: invariants 4 P_{i,j}^2 and -1/P^2 (the sign: bg_unit.cuh accumulates minus the bracket); the r
    //      proper ranges are dealt round-robin to the W*S (half-)warps, each batch-inverts its share (zero-safe).
    //      Momenta only: once per tile and ordering ----
    {
        constexpr int VW = W * S;
        const int vw = warp * S + t.half;
        E* Wt = sc + L.sc_w * TP;
        uint32_t status = 0;
#pragma unroll 1
        for (int r = vw; r < L.r; r += VW) {
            const uint32_t rg = P.tab.ranges[r];
            E lo[D], hi[D], x[D], nx[D];
            ld_vec<F, D>(recf + (PS0 + (rg & 255u)) * D, lo);
            ld_vec<F, D>(recf + (PS0 + (rg >> 8)) * D, hi);
#pragma unroll
            for (int mu = 0; mu < D; ++mu) x[mu] = f.sub(hi[mu], lo[mu]);
            lower_neg<F, MET, D>(f, 0, x, nx);
            Wt[r * TP] = f.canon(f.neg(f.reduce(dot_plain<F, D>(f, nx, x))));
        }
        if constexpr (F::kExact) {
            E* tmp = sc + L.sc_v * TP;                         // prefix products, in the V slots (dead until the sweep)
            E c = f.one();
#pragma unroll 1
            for (int r = vw; r < L.r; r += VW) {
                tmp[r * TP] = c;
                const E s = Wt[r * TP];
                const bool z = f.is_zero(s);
                if (z) status |= 1u;
                c = f.mul(c, z ? f.one() : s);
            }
            E u = f.neg(f.dbl(f.dbl(f.inv(c))));
            int rl = vw + ((L.r - 1 - vw) / VW) * VW;          // last r of this (half-)warp
            if (vw >= L.r) rl = -1;
#pragma unroll 1
            for (int r = rl; r >= 0; r -= VW) {
                const E s = Wt[r * TP];
                const bool z = f.is_zero(s);
                Wt[r * TP] = z ? f.ezero() : f.mul(u, tmp[r * TP]);
                u = f.mul(u, z ? f.one() : s);
            }
        } else {
#pragma unroll 1
            for (int r = vw; r < L.r; r += VW) {
                const E s = Wt[r * TP];
                if (f.is_zero(s)) status |= 1u;
                Wt[r * TP] = f.neg(f.dbl(f.dbl(f.inv(s))));
            }
        }
        if (gstat && status) atomicOr(&stat[point], status);
    }
    __syncthreads();
    if (gstat && warp == 0 && t.half == 0 && t.live) gstat[t.pt] = stat[point];   // (accumulates over the orderings)

    // ---- a4-a6: the level sweep (bg_unit.cuh), once per state configuration (Eq.(4)) ----
#pragma unroll 1
    for (int s = 0; s < states; ++s) {
        if (MULTI && s > 0) {
            __syncthreads();                                   // the previous sweep is done with eps_n
            rt_stage<F, D, W>(f, vec, L.vstride, valid, gpol + (long long)s * nd, (long long)states * nd, 0, n, perm, n);
            __syncthreads();
            singles();
            __syncthreads();
        }
        unit_sweep_body<F, MET, D, S>(f, lay, prog, t, warp, rec, sc, stat + TP + lane,
                                      ((uint32_t)o * (uint32_t)states + (uint32_t)s) * 16u, gout + s, prm.currents);
    }
    }
}

}  // namespace bg
