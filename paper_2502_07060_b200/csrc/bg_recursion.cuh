// bg_recursion.cuh -- the Berends-Giele level sweep as ONE sm_100a kernel.
//
// Mapping: one thread per phase-space point (points are independent).
// Each point owns a private RECORD in shared memory (array-of-structures, record
// stride padded so that the lanes of a warp hit distinct banks with 8/16-byte loads):
//
//   J table   slots [0, n + m(m-1)/2)  x D   currents J(i..j); singles first, so the
//                                             caller's [n][d] polarisations are copied in
//                                             verbatim (slot m holds eps_n)
//   P table   slots [0, slot(1,m))     x D   X(i..j) = 2 * covariant P_{i,j}: doubled and
//                                             index-lowered once, so that every
//                                             contraction below is a plain sum of products
//   S table   R scalars                      S(i..j) = sum_k J(i..k).J(k+1..j)
//   W table   R scalars                      1 / P_{i,j}^2  (batch-inverted)
//
// The recursion is Eq.(6) with V3, V4 of Eq.(7), i-free, in the
// algebraically identical "factored" form:
//
//   bracket(i..j)^mu = sum_k [ (A.B)(P-Q)^mu + (2 Q.A - S(i..k)) B^mu - (2 P.B + S(k+1..j)) A^mu ]
//                    + sum_{k<l} 2 (A_k . C_l) J(k+1..l)^mu
//   A = J(i..k), B = J(k+1..j), P = P_{i,k}, Q = P_{k+1,j}, C_l = J(l+1..j)
//
// i.e. the two single-dot terms of V4 are summed over the inner index first, which turns
// them into the by-product S of the 3-vertex loop (O(n^3) instead of O(n^4) work).  Over
// F_p this is exact, so the result is bit-identical to the literal form.
#pragma once
#include "bg_field.cuh"

namespace bg {

// slot of the range starting at i (1-based) with length L in the level-major tables
__host__ __device__ constexpr int slot_of(int n, int i, int L)
{
    return L == 1 ? i - 1 : n + (L - 2) * (n - 1) - (L - 1) * (L - 2) / 2 + (i - 1);
}

struct RecordLayout {
    int n, m, d;
    int j_slots, p_slots, r;      // table sizes (slots / scalars)
    int off_p, off_s, off_w;      // offsets in elements
    int size;                     // used elements
    int stride;                   // padded record stride in elements
};

__host__ __device__ constexpr RecordLayout make_layout(int n, int d, int vec)
{
    RecordLayout L{};
    L.n = n; L.m = n - 1; L.d = d;
    L.j_slots = n + (n - 1) * (n - 2) / 2;
    L.p_slots = slot_of(n, 1, n - 1);
    L.r = L.p_slots - n;
    L.off_p = L.j_slots * d;
    L.off_s = L.off_p + L.p_slots * d;
    L.off_w = L.off_s + L.r;
    L.size = L.off_w + L.r;
    int s = (L.size + vec - 1) / vec;     // in vector units
    if ((s & 1) == 0) ++s;                // odd number of vector units: conflict-free lanes
    L.stride = s * vec;
    return L;
}

template <class F, int D> struct VecWidth { static constexpr int value = 1; };
template <int D> struct VecWidth<Fp31, D> { static constexpr int value = (D % 4 == 0) ? 4 : (D % 2 == 0) ? 2 : 1; };

// the memory type of one vector unit of U elements, and the input reduction applied to it
template <class F, int U> struct VecType { typedef typename F::E type; };
template <> struct VecType<Fp31, 2> { typedef uint2 type; };
template <> struct VecType<Fp31, 4> { typedef uint4 type; };
template <class F> __device__ __forceinline__ typename F::E load_unit(typename F::E v) { return F::load_input(v); }
template <class F> __device__ __forceinline__ uint2 load_unit(uint2 v)
{
    return make_uint2(F::load_input(v.x), F::load_input(v.y));
}
template <class F> __device__ __forceinline__ uint4 load_unit(uint4 v)
{
    return make_uint4(F::load_input(v.x), F::load_input(v.y), F::load_input(v.z), F::load_input(v.w));
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

// sum_mu x_mu y_mu, plain (one operand already index-lowered); headroom by F::relief (one operand
// of every product is a canonical residue <= p-1: stored vectors always are)
template <class F, int D>
__device__ __forceinline__ typename F::A dot_plain(const typename F::E (&x)[D], const typename F::E (&y)[D])
{
    typename F::A s = F::zero();
#pragma unroll
    for (int mu = 0; mu < D; ++mu) {
        if (mu >= F::kCap0 && ((mu - F::kCap0) % F::kCapR) == 0) s = F::relief(s);
        s = F::mad(x[mu], y[mu], s);
    }
    return s;
}

// MINUS the Minkowski product of two contravariant vectors: sum_{mu>=1} x y + (-x0) y0
template <class F, int D>
__device__ __forceinline__ typename F::A dot_neg(typename F::E nx0, const typename F::E (&x)[D],
                                                  const typename F::E (&y)[D])
{
    typename F::A s = F::mad(nx0, y[0], F::zero());
#pragma unroll
    for (int mu = 1; mu < D; ++mu) {
        if (mu >= F::kCap0 && ((mu - F::kCap0) % F::kCapR) == 0) s = F::relief(s);
        s = F::mad(x[mu], y[mu], s);
    }
    return s;
}

template <class E>
struct KernelParams {
    const E* mom;         // [batch][n][D]
    const E* pol;         // [batch][n][D]
    E* out;               // [batch]
    E* currents;          // NULL or [batch][m][m][D]
    uint32_t* status;     // NULL or [batch]
    long long batch;
    int n;                // used when N == 0
    int stride;           // record stride in elements
};

template <class F, int N, int D>
__global__ void bg_recursion_kernel(const KernelParams<typename F::E> prm)
{
    typedef typename F::E E;
    typedef typename F::A A;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    E* smem = reinterpret_cast<E*>(smem_raw);

    const int n = N ? N : prm.n;
    const int m = n - 1;
    const int nd = n * D;
    const RecordLayout lay = make_layout(n, D, VecWidth<F, D>::value);
    const int stride = prm.stride;
    const int T = blockDim.x;
    const long long tile0 = (long long)blockIdx.x * T;
    const int valid = (int)min((long long)T, prm.batch - tile0);

    // ---- a0: stage the tile, coalesced, into the per-point records ------------------------
    {
        const E* gm = prm.mom + tile0 * nd;
        const E* gp = prm.pol + tile0 * nd;
        const int total = valid * nd;
        for (int g = threadIdx.x; g < total; g += T) {
            const int pt = g / nd, w = g - pt * nd;
            E* rec = smem + (size_t)pt * stride;
            rec[w] = F::load_input(gp[g]);
            rec[lay.off_p + w] = F::load_input(gm[g]);
        }
    }
    __syncthreads();
    if ((int)threadIdx.x >= valid) return;

    E* rec = smem + (size_t)threadIdx.x * stride;
    E* Jt = rec;
    E* Pt = rec + lay.off_p;
    E* St = rec + lay.off_s;
    E* Wt = rec + lay.off_w;
    uint32_t status = 0;

    // ---- a1: X(i..j) = 2 * covariant P_{i,j}  (Eq.(7); metric PAPER.md:140) ---
    for (int l = 0; l < m; ++l) {
        E k[D];
        ld_vec<F, D>(Pt + l * D, k);
        k[0] = F::dbl(k[0]);
#pragma unroll
        for (int mu = 1; mu < D; ++mu) k[mu] = F::canon(F::neg(F::dbl(k[mu])));
        st_vec<F, D>(Pt + l * D, k);
    }
    for (int L = 2; L < m; ++L)
        for (int i = 1; i + L - 1 <= m; ++i) {
            E a[D], b[D];
            ld_vec<F, D>(Pt + slot_of(n, i, L - 1) * D, a);
            ld_vec<F, D>(Pt + (i + L - 2) * D, b);
#pragma unroll
            for (int mu = 0; mu < D; ++mu) a[mu] = F::add(a[mu], b[mu]);
            st_vec<F, D>(Pt + slot_of(n, i, L) * D, a);
        }

    // ---- a2: invariants 4 P_{i,j}^2 for the R proper ranges --------------------------------
    const int R = lay.r;
    for (int r = 0; r < R; ++r) {
        E x[D];
        ld_vec<F, D>(Pt + (n + r) * D, x);
        A ns = dot_neg<F, D>(F::neg(x[0]), x, x);          // -(X.X) = -4 P^2
        E s4 = F::canon(F::neg(F::reduce(ns)));
        if (F::is_zero(s4)) status |= 1u;
        Wt[r] = s4;
    }

    // ---- a3: all propagators 1/P^2 = 4/(4P^2) at once ---------------------------------------
    if constexpr (F::kExact) {
        // Montgomery's trick, zero-safe: one field inversion per POINT.  inv(0) := 0.
        E c = F::one();
        for (int r = 0; r < R; ++r) {
            St[r] = c;
            E s = Wt[r];
            c = F::mul(c, F::is_zero(s) ? F::one() : s);
        }
        E u = F::inv(c);
        u = F::dbl(F::dbl(u));
        for (int r = R - 1; r >= 0; --r) {
            E s = Wt[r];
            const bool z = F::is_zero(s);
            Wt[r] = z ? F::ezero() : F::mul(u, St[r]);
            u = F::mul(u, z ? F::one() : s);
        }
    } else {
        for (int r = 0; r < R; ++r) Wt[r] = F::dbl(F::dbl(F::inv(Wt[r])));
    }

    // ---- a4: level sweep (Eq.(6)) ------------------------------------------------
    E top[D];
    for (int L = 2; L <= m; ++L) {
        for (int i = 1; i + L - 1 <= m; ++i) {
            const int j = i + L - 1;
            A acc[D];
#pragma unroll
            for (int mu = 0; mu < D; ++mu) acc[mu] = F::zero();
            E hsum = F::ezero();

            // 3-gluon vertex with the factored single-dot terms of the 4-gluon vertex
            for (int k = i; k < j; ++k) {
                const int la = k - i + 1, lb = j - k;
                const int sa = slot_of(n, i, la), sb = slot_of(n, k + 1, lb);
                E a[D], b[D], x[D], y[D];
                ld_vec<F, D>(Jt + sa * D, a);
                ld_vec<F, D>(Jt + sb * D, b);
                ld_vec<F, D>(Pt + sa * D, x);
                ld_vec<F, D>(Pt + sb * D, y);
                const A nab = dot_neg<F, D>(F::neg(a[0]), a, b);     // -(A.B)
                const A ya = dot_plain<F, D>(y, a);                  //  2 Q.A
                const A xb = dot_plain<F, D>(x, b);                  //  2 P.B
                const E h = F::reduce_half(nab);                     // -(A.B)/2
                const E nh = F::neg(h);
                E cb = F::reduce(ya);
                E ca = F::reduce(xb);
                if (la > 1) cb = F::sub(cb, St[sa - n]);
                if (lb > 1) ca = F::add(ca, St[sb - n]);
                ca = F::neg(ca);
                hsum = F::add(hsum, h);
                // (A.B)(P-Q)^mu = h g^{mu mu} (Y_mu - X_mu)
                acc[0] = F::fold(acc[0]);
                acc[0] = F::mad(h, y[0], acc[0]);
                acc[0] = F::mad(nh, x[0], acc[0]);
                acc[0] = F::mad(cb, b[0], acc[0]);
                acc[0] = F::mad(ca, a[0], acc[0]);
#pragma unroll
                for (int mu = 1; mu < D; ++mu) {
                    acc[mu] = F::fold(acc[mu]);
                    acc[mu] = F::mad(h, x[mu], acc[mu]);
                    acc[mu] = F::mad(nh, y[mu], acc[mu]);
                    acc[mu] = F::mad(cb, b[mu], acc[mu]);
                    acc[mu] = F::mad(ca, a[mu], acc[mu]);
                }
            }

            // remaining 4-gluon term: 2 (A_k . C_l) J(k+1..l)
            int room = 0;
            for (int k = i; k + 1 < j; ++k) {
                E a[D];
                ld_vec<F, D>(Jt + slot_of(n, i, k - i + 1) * D, a);
                const E na0 = F::neg(a[0]);
                for (int l = k + 1; l < j; ++l) {
                    E bm[D], c[D];
                    ld_vec<F, D>(Jt + slot_of(n, k + 1, l - k) * D, bm);
                    ld_vec<F, D>(Jt + slot_of(n, l + 1, j - l) * D, c);
                    const A nac = dot_neg<F, D>(na0, a, c);          // -(A.C)
                    const E cc = F::neg(F::reduce_double(nac));      // 2 (A.C)
                    if (room == 0) {
#pragma unroll
                        for (int mu = 0; mu < D; ++mu) acc[mu] = F::fold(acc[mu]);
                        room = F::kCap;
                    }
                    --room;
#pragma unroll
                    for (int mu = 0; mu < D; ++mu) acc[mu] = F::mad(cc, bm[mu], acc[mu]);
                }
            }

            // propagator (none on the top current) and store
            const int sj = slot_of(n, i, L);
            E v[D];
            if (L < m) {
                const E w = Wt[sj - n];
#pragma unroll
                for (int mu = 0; mu < D; ++mu) v[mu] = F::mul(F::reduce(acc[mu]), w);
                St[sj - n] = F::canon(F::neg(F::dbl(hsum)));         // S = -2 sum h
            } else {
#pragma unroll
                for (int mu = 0; mu < D; ++mu) v[mu] = F::reduce(acc[mu]);
#pragma unroll
                for (int mu = 0; mu < D; ++mu) top[mu] = v[mu];
            }
            st_vec<F, D>(Jt + sj * D, v);
        }
    }

    // ---- a5/a6: amplitude = eps_n . N(1..m) ------------------------------------------------------
    const long long pt = tile0 + threadIdx.x;
    {
        E e[D];
        ld_vec<F, D>(Jt + m * D, e);
        const A nout = dot_neg<F, D>(F::neg(e[0]), e, top);
        prm.out[pt] = F::canon(F::neg(F::reduce(nout)));
    }
    if (prm.status) prm.status[pt] = status;
    if (prm.currents) {
        E* cur = prm.currents + pt * (long long)m * m * D;
        for (int i = 1; i <= m; ++i)
            for (int jj = i; jj <= m; ++jj) {
                const E* src = Jt + slot_of(n, i, jj - i + 1) * D;
                E* dst = cur + ((long long)(i - 1) * m + (jj - 1)) * D;
#pragma unroll
                for (int mu = 0; mu < D; ++mu) dst[mu] = src[mu];
            }
    }
}

}  // namespace bg
