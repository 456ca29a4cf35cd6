// bg_common.cuh -- pieces shared by every Berends-Giele kernel: launch parameters, vector
// load/store, Minkowski products with a compile-time metric, lane-pair sums.
//
// Algebra used by all kernels ("factored form" of the i-free V3, V4 of Eq.(7), PAPER.md:99-101;
// DESIGN.md §6).  For the current (i..j) with own momentum X = P_{i,j} and a split
// A = J(i..k), B = J(k+1..j), with PS2_c = 2 (k_1+..+k_c) (Eq.(7)) and the
// per-current scalars U = 2 P.J + S, V = 2 P.J - S (P the current's own momentum,
// S(i..l) = sum_k J(i..k).J(k+1..l)):
//
//   bracket^mu = sum_k [ h_k PS2_k^mu + (2X.A - U_A) B^mu + (V_B - 2X.B) A^mu ]
//              - (sum_k h_k)/2 (PS2_{i-1} + PS2_j)^mu
//              + sum_{k<l} 2 (A_k . C_l) J(k+1..l)^mu ,        h_k = A.B
//
// Per 3-split 3 dot products + 3 axpys, per 4-split 1 dot + 1 axpy.  Exact over F_p, hence
// bit-identical to the literal evaluation; over complex128 a reordering within DESIGN.md R9/R10.
// The tiled kernel accumulates MINUS the bracket (with -g A as the left factor of the Minkowski products and
// -2 X, every coefficient but one comes out of its reduction with the right sign; the table holds -1/P^2).
#pragma once
#include "bg_field.cuh"

namespace bg {

// Shared-memory layout of a tile for a run-time n (bg_rt.cuh; the compile-time twin is TileCfg in bg_tile.cuh):
// vector record rows [0,n) eps, [n, n+r) multi-gluon currents, ps0 + c the doubled prefix sums; scalar tables
// [index][point]: U per row from 0, V per multi-gluon row from sc_v, 1/P^2 parked in the U slots (sc_w = n),
// scratch slots of d + 1 entries from sc_scr.  Counts in elements.
struct RtLayout {
    int n, m, r;
    int ps0, vstride;
    int sc_v, sc_w, sc_scr, nscal, nslots;
};

// Launch parameters of every recursion kernel.  blockIdx.y = index of the prime of a
// multi-prime call (0 otherwise): all arrays of prime q start q * (their size) elements in.
template <class F>
struct BgParams {
    typedef typename F::E E;
    const E* mom;         // [primes][batch][n][D]
    const E* pol;         // [primes][batch][states][n][D]
    E* out;               // [primes][batch][orderings][states]
    E* currents;          // NULL or [batch][m][m][D]   (states == 1, one prime)
    uint32_t* status;     // NULL or [primes][batch]
    long long batch;
    int states;           // S >= 1 polarisation configurations per momentum point (Eq.(4))
    int n_orderings;      // K >= 1 colour orderings per point (Eq.(5))
    const unsigned char* orderings;   // NULL (K == 1, the caller's order) or device [K][n]: leg at position i
    int n;                // general kernel only
    int stride;           // general kernel only: record stride in elements
    typename F::Params fld;
    RtLayout rt;          // bg_rt_kernel only (bg_rt.cuh): the tile layout of this n
};

// One op of the flat per-warp program of the tiled kernels (bg_unit.cuh: flat_build, unit_sweep_body).
struct FlatOp {
    uint32_t ab;       // row A | row B << 16      (byte offsets in the lane's vector record)
    uint32_t pso;      // row PS2_k | own row << 16
    uint32_t u, v;     // U_A, V_B                 (byte offsets from the lane's scalar base)
    uint32_t w;        // ci * m + j - 1 (position in the caller's `currents` array) | own row << 8 | level << 16
                       // | OP_PART: first parked flag of the slot (word index) << 20
    uint32_t lh;       // rows PS2_{i-1} | PS2_j << 16
    uint32_t qcf;      // first entry of the op's 4-gluon splits in quad[] | c4 << 16 | flags << 24
    uint32_t aux;      // OP_PART: scratch slot (byte offset from the first slot) ; OP_GATHER: mask of slots
};

// bg_rt_kernel: the schedule of a run-time n travels with the launch as a kernel PARAMETER (constant bank: the ops
// are read with uniform loads like the __constant__ tables of the compiled kernels; nothing is allocated or copied
// to the device).  sized for n = 16 with 8 warps; 29 KB of the 32 KB a kernel may take.
constexpr int kRtMaxOps = 680, kRtMaxQuad = 1820, kRtMaxRanges = 104;
struct RtTables {
    FlatOp ops[kRtMaxOps];
    uint32_t quad[kRtMaxQuad];    // row J(k+1..l) | row J(l+1..j) << 16 per 4-gluon split
    uint16_t beg[16];             // ops of warp w: [beg[w], beg[w+1])
    uint16_t ranges[kRtMaxRanges];   // lo | hi << 8 of the proper multi-gluon ranges
};
template <class F>
struct RtParams {
    BgParams<F> base;
    RtTables tab;
};
static_assert(sizeof(RtTables) + 512 <= 32764, "kernel parameters are limited to 32764 bytes");

template <class F, int D> struct VecWidth { static constexpr int value = 1; };
template <int D> struct VecWidth<Fp31, D> { static constexpr int value = (D % 4 == 0) ? 4 : (D % 2 == 0) ? 2 : 1; };
template <int D> struct VecWidth<FpMont, D> { static constexpr int value = VecWidth<Fp31, D>::value; };

// the memory type of one vector unit of U elements, and the input conversion applied to it
template <class F, int U> struct VecType { typedef typename F::E type; };
template <> struct VecType<Fp31, 2> { typedef uint2 type; };
template <> struct VecType<Fp31, 4> { typedef uint4 type; };
template <> struct VecType<FpMont, 2> { typedef uint2 type; };
template <> struct VecType<FpMont, 4> { typedef uint4 type; };
template <class F> __device__ __forceinline__ typename F::E load_unit(const F& f, typename F::E v) { return f.load_input(v); }
template <class F> __device__ __forceinline__ uint2 load_unit(const F& f, uint2 v)
{
    return make_uint2(f.load_input(v.x), f.load_input(v.y));
}
template <class F> __device__ __forceinline__ uint4 load_unit(const F& f, uint4 v)
{
    return make_uint4(f.load_input(v.x), f.load_input(v.y), f.load_input(v.z), f.load_input(v.w));
}

template <class F, int D>
__device__ __forceinline__ void ld_vec(const typename F::E* p, typename F::E (&v)[D])
{
    constexpr int W = VecWidth<F, D>::value;
    if constexpr (W == 4) {
#pragma unroll
        for (int q = 0; q < D / 4; ++q) {
            uint4 t = reinterpret_cast<const uint4*>(p)[q];
            v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
        }
    } else if constexpr (W == 2) {
#pragma unroll
        for (int q = 0; q < D / 2; ++q) {
            uint2 t = reinterpret_cast<const uint2*>(p)[q];
            v[2 * q] = t.x; v[2 * q + 1] = t.y;
        }
    } else {
#pragma unroll
        for (int q = 0; q < D; ++q) v[q] = p[q];
    }
}

template <class F, int D>
__device__ __forceinline__ void st_vec(typename F::E* p, const typename F::E (&v)[D])
{
    constexpr int W = VecWidth<F, D>::value;
    if constexpr (W == 4) {
#pragma unroll
        for (int q = 0; q < D / 4; ++q)
            reinterpret_cast<uint4*>(p)[q] = make_uint4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
    } else if constexpr (W == 2) {
#pragma unroll
        for (int q = 0; q < D / 2; ++q) reinterpret_cast<uint2*>(p)[q] = make_uint2(v[2 * q], v[2 * q + 1]);
    } else {
#pragma unroll
        for (int q = 0; q < D; ++q) p[q] = v[q];
    }
}

// sum_mu x_mu y_mu, plain (the metric is already inside one operand); headroom by relief (one
// operand of every product is a canonical residue <= p-1: stored vectors always are)
template <class F, int D>
__device__ __forceinline__ typename F::A dot_plain(const F& f, const typename F::E (&x)[D],
                                                    const typename F::E (&y)[D])
{
    typename F::A s = f.zero();
#pragma unroll
    for (int mu = 0; mu < D; ++mu) {
        if (mu >= F::kCap0 && ((mu - F::kCap0) % F::kCapR) == 0) s = f.relief(s);
        s = f.mad(x[mu], y[mu], s);
    }
    return s;
}

// init + sum_mu x_mu y_mu (init an element: one more product for the headroom rules unless F::kWidenFree)
template <class F, int D>
__device__ __forceinline__ typename F::A dot_plain_from(const F& f, typename F::E init, const typename F::E (&x)[D],
                                                         const typename F::E (&y)[D])
{
    constexpr int used = F::kWidenFree ? 0 : 1;
    typename F::A s = f.widen(init);
#pragma unroll
    for (int mu = 0; mu < D; ++mu) {
        if (mu + used >= F::kCap0 && ((mu + used - F::kCap0) % F::kCapR) == 0) s = f.relief(s);
        s = f.mad(x[mu], y[mu], s);
    }
    return s;
}

// x or -x (flag usually folds at compile time)
__device__ __forceinline__ uint32_t cneg(const Fp31&, uint32_t x, bool flag) { return x ^ (flag ? kP : 0u); }
__device__ __forceinline__ uint32_t cneg(const FpMont& f, uint32_t x, bool flag) { return flag ? f.p - x : x; }
__device__ __forceinline__ double2 cneg(const C128&, double2 x, bool flag)
{
    return flag ? make_double2(-x.x, -x.y) : x;
}

// nx_mu = -g_{mu mu} x_mu for the components mu0 .. mu0+DL-1 a lane owns, so that
// dot_plain(nx, y) = MINUS the Minkowski product x.y (restricted to those components)
template <class F, int MET, int DL>
__device__ __forceinline__ void lower_neg(const F& f, int mu0, const typename F::E (&x)[DL], typename F::E (&nx)[DL])
{
#pragma unroll
    for (int mu = 0; mu < DL; ++mu) nx[mu] = cneg(f, x[mu], !Metric<MET>::minus(mu0 + mu));
}

// x2_mu = g_{mu mu} (h - l)_mu : twice the covariant P_{i,j} from the doubled prefix sums
template <class F, int MET, int DL>
__device__ __forceinline__ void lower_diff(const F& f, int mu0, const typename F::E (&h)[DL],
                                           const typename F::E (&l)[DL], typename F::E (&x2)[DL])
{
#pragma unroll
    for (int mu = 0; mu < DL; ++mu) x2[mu] = cneg(f, f.sub(h[mu], l[mu]), Metric<MET>::minus(mu0 + mu));
}

// value summed over the S lanes that share a point (lanes l and l + TP of a warp when S == 2)
template <class F, int S, int TP>
__device__ __forceinline__ uint32_t lane_sum(const F& f, uint32_t x)
{
    if constexpr (S == 1) return x;
    else return f.add(x, __shfl_xor_sync(0xffffffffu, x, TP));
}
template <class F, int S, int TP>
__device__ __forceinline__ double2 lane_sum(const F&, double2 x)
{
    if constexpr (S == 1) return x;
    else return make_double2(x.x + __shfl_xor_sync(0xffffffffu, x.x, TP), x.y + __shfl_xor_sync(0xffffffffu, x.y, TP));
}

}  // namespace bg
