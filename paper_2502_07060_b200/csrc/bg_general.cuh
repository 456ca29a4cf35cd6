// bg_general.cuh -- the Berends-Giele recursion for ANY 4 <= n <= 16 at compile-time d: one thread
// per phase-space point, run-time loops over levels, currents and splittings (SURVEY.md 8(a) rows
// a0-a6 in one launch).  The path for every shape without a compiled bg_unit_kernel instance.
//
// Each point owns a private RECORD in shared memory (array of structures, record stride an odd
// number of vector units so that the lanes of a warp hit distinct banks with 8/16-byte loads):
//
//   rows [0, n)          eps_1..eps_n of the current state configuration
//   rows [n, n+R)        multi-gluon currents J(i..j), level-major, top excluded
//   rows PS0 + c         doubled prefix sums PS2_c = 2 (k_1+..+k_c), c = 0..m  (Eq.(7))
//   scalars              U, V per row; 1/P^2 per proper multi-gluon range
//
// Same algebra as the tiled kernel (bg_common.cuh), same states loop (bg_tile.cuh header).
#pragma once
#include "bg_common.cuh"
#include "bg_schedule.cuh"

namespace bg {

struct GeneralLayout {
    int n, m, r;                  // gluons, n-1, proper multi-gluon ranges
    int j_rows, ps0;              // rows of the vector part
    int off_u, off_v, off_w;      // scalar tables, offsets in elements
    int size, stride;             // used / padded record size in elements
};

__host__ __device__ constexpr GeneralLayout make_general_layout(int n, int d, int vec)
{
    GeneralLayout L{};
    L.n = n; L.m = n - 1;
    L.r = L.m * (L.m - 1) / 2 - 1;
    L.j_rows = n + L.r;
    L.ps0 = L.j_rows;
    L.off_u = (L.j_rows + L.m + 1) * d;
    L.off_v = L.off_u + L.j_rows;
    L.off_w = L.off_v + L.j_rows;
    L.size = L.off_w + L.r;
    int s = (L.size + vec - 1) / vec;     // in vector units
    if ((s & 1) == 0) ++s;                // odd number of vector units: conflict-free lanes
    L.stride = s * vec;
    return L;
}

template <class F, int MET, int D>
__global__ void bg_general_kernel(const BgParams<F> prm)
{
    typedef typename F::E E;
    typedef typename F::A A;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    E* smem = reinterpret_cast<E*>(smem_raw);
    const F f(prm.fld, blockIdx.y);

    const int n = prm.n, m = n - 1, nd = n * D;
    const GeneralLayout lay = make_general_layout(n, D, VecWidth<F, D>::value);
    const int stride = prm.stride, states = prm.states;
    const int T = blockDim.x;
    const long long tile0 = (long long)blockIdx.x * T;
    const int valid = (int)min((long long)T, prm.batch - tile0);
    const long long pbase = (long long)blockIdx.y * prm.batch;
    const bool live = (int)threadIdx.x < valid;
    const long long pt = tile0 + threadIdx.x;

    E* rec = smem + (size_t)threadIdx.x * stride;
    E* PS = rec + lay.ps0 * D;
    E* Ut = rec + lay.off_u;
    E* Vt = rec + lay.off_v;
    E* Wt = rec + lay.off_w;
    const int R = lay.r;

    uint32_t status = 0;
    const int n_ord = prm.n_orderings;
    for (int o = 0; o < n_ord; ++o) {
    // colour ordering o (Eq.(5)): the inputs are staged in that order, the rest is unchanged
    const unsigned char* perm = prm.orderings ? prm.orderings + o * n : nullptr;
    if (o > 0) __syncthreads();
    // ---- a0: stage the momenta k_1..k_m into the PS rows 1..m, coalesced ---------------------------
    {
        const E* gm = prm.mom + (pbase + tile0) * nd;
        const int per = m * D, total = valid * per;
        for (int g = threadIdx.x; g < total; g += T) {
            const int p = g / per, w = g - p * per;
            const int row = w / D, c = w - row * D;
            const int srow = perm ? min((int)perm[row], n - 1) : row;
            smem[(size_t)p * stride + (lay.ps0 + 1) * D + w] = f.load_input(gm[(long long)p * nd + srow * D + c]);
        }
    }
    __syncthreads();

    if (live) {
        // ---- a1: doubled prefix sums (Eq.(7)) ----------------------------------------
        E run[D];
#pragma unroll
        for (int mu = 0; mu < D; ++mu) run[mu] = f.ezero();
        st_vec<F, D>(PS, run);
        for (int c = 1; c <= m; ++c) {
            E k[D];
            ld_vec<F, D>(PS + c * D, k);
#pragma unroll
            for (int mu = 0; mu < D; ++mu) run[mu] = f.add(run[mu], f.dbl(k[mu]));
            st_vec<F, D>(PS + c * D, run);
        }
        // ---- a2: invariants 4 P_{i,j}^2 for the R proper ranges, level-major -------------------------
        {
            int r = 0;
            for (int L = 2; L <= m - 1; ++L)
                for (int i = 0; i + L <= m; ++i, ++r) {
                    E lo[D], hi[D], x[D], nx[D];
                    ld_vec<F, D>(PS + i * D, lo);
                    ld_vec<F, D>(PS + (i + L) * D, hi);
#pragma unroll
                    for (int mu = 0; mu < D; ++mu) x[mu] = f.sub(hi[mu], lo[mu]);
                    lower_neg<F, MET, D>(f, 0, x, nx);
                    const E s4 = f.canon(f.neg(f.reduce(dot_plain<F, D>(f, nx, x))));
                    if (f.is_zero(s4)) status |= 1u;
                    Wt[r] = s4;
                }
        }
        // ---- a3: all propagators 1/P^2 = 4/(4P^2) at once ----------------------------------------------
        if constexpr (F::kExact) {
            // Montgomery's trick, zero-safe: one field inversion per POINT.  inv(0) := 0.
            // Prefix products parked in the not-yet-used U slots of the multi-gluon currents.
            E* tmp = Ut + n;
            E c = f.one();
            for (int r = 0; r < R; ++r) {
                tmp[r] = c;
                const E s = Wt[r];
                c = f.mul(c, f.is_zero(s) ? f.one() : s);
            }
            E u = f.inv(c);
            u = f.dbl(f.dbl(u));
            for (int r = R - 1; r >= 0; --r) {
                const E s = Wt[r];
                const bool z = f.is_zero(s);
                Wt[r] = z ? f.ezero() : f.mul(u, tmp[r]);
                u = f.mul(u, z ? f.one() : s);
            }
        } else {
            for (int r = 0; r < R; ++r) Wt[r] = f.dbl(f.dbl(f.inv(Wt[r])));
        }
        if (prm.status) prm.status[pbase + pt] = status;
    }

    for (int s = 0; s < states; ++s) {
        // ---- a0 (states): eps_1..eps_n of configuration s, coalesced --------------------------------
        __syncthreads();
        {
            const E* gp = prm.pol + ((pbase + tile0) * states + s) * nd;
            const int total = valid * nd;
            for (int g = threadIdx.x; g < total; g += T) {
                const int p = g / nd, w = g - p * nd;
                const int row = w / D, c = w - row * D;
                const int srow = perm ? min((int)perm[row], n - 1) : row;
                smem[(size_t)p * stride + w] = f.load_input(gp[(long long)p * states * nd + srow * D + c]);
            }
        }
        __syncthreads();
        if (!live) continue;

        // single-gluon U = V = 2 k_c . eps_c
        for (int c = 1; c <= m; ++c) {
            E lo[D], hi[D], k2[D], e[D];
            ld_vec<F, D>(PS + (c - 1) * D, lo);
            ld_vec<F, D>(PS + c * D, hi);
            ld_vec<F, D>(rec + (c - 1) * D, e);
            lower_diff<F, MET, D>(f, 0, hi, lo, k2);
            const E u = f.reduce(dot_plain<F, D>(f, k2, e));
            Ut[c - 1] = u;
            Vt[c - 1] = u;
        }

        // ---- a4: level sweep (Eq.(6)) --------------------------------------------------
        for (int L = 2; L <= m; ++L) {
            for (int i = 1; i + L - 1 <= m; ++i) {
                E l[D], h[D], x2[D];
                ld_vec<F, D>(PS + (i - 1) * D, l);
                ld_vec<F, D>(PS + (i - 1 + L) * D, h);
                lower_diff<F, MET, D>(f, 0, h, l, x2);                    // 2 * covariant P_{i,j}
                A acc[D];
#pragma unroll
                for (int mu = 0; mu < D; ++mu) acc[mu] = f.zero();
                E hsum = f.ezero();
                int room = F::kCap0;
                auto need = [&](int k) {
                    if (room < k) {
#pragma unroll
                        for (int mu = 0; mu < D; ++mu) acc[mu] = f.relief(acc[mu]);
                        room = F::kCapR;
                    }
                    room -= k;
                };
                for (int la = 1; la <= L - 1; ++la) {
                    const int ra = tt_row(n, i, la), rb = tt_row(n, i + la, L - la);
                    E a[D], b[D], ps[D], na[D];
                    ld_vec<F, D>(rec + ra * D, a);
                    ld_vec<F, D>(rec + rb * D, b);
                    ld_vec<F, D>(PS + (i - 1 + la) * D, ps);
                    lower_neg<F, MET, D>(f, 0, a, na);
                    const E hk = f.neg(f.reduce(dot_plain<F, D>(f, na, b)));      // A.B
                    const E xa = f.reduce(dot_plain<F, D>(f, x2, a));             // 2 X.A
                    const E xb = f.reduce(dot_plain<F, D>(f, x2, b));             // 2 X.B
                    const E cb = f.sub(xa, Ut[ra]);
                    const E ca = f.sub(Vt[rb], xb);
                    hsum = f.add(hsum, hk);
                    need(2);
#pragma unroll
                    for (int mu = 0; mu < D; ++mu) {
                        acc[mu] = f.mad(hk, ps[mu], acc[mu]);
                        acc[mu] = f.mad(cb, b[mu], acc[mu]);
                    }
                    need(1);
#pragma unroll
                    for (int mu = 0; mu < D; ++mu) acc[mu] = f.mad(ca, a[mu], acc[mu]);
                    for (int lb = 1; lb <= L - la - 1; ++lb) {
                        // (i..k | k+1..l | l+1..j): 2 (A.C) J(k+1..l)
                        E bm[D], c[D];
                        ld_vec<F, D>(rec + tt_row(n, i + la, lb) * D, bm);
                        ld_vec<F, D>(rec + tt_row(n, i + la + lb, L - la - lb) * D, c);
                        const E cc = f.neg(f.dbl(f.reduce(dot_plain<F, D>(f, na, c))));
                        need(1);
#pragma unroll
                        for (int mu = 0; mu < D; ++mu) acc[mu] = f.mad(cc, bm[mu], acc[mu]);
                    }
                }
                // finish: boundary term of the (P-Q) sum, propagator (none on the top current)
                const E nhh = f.neg(f.mul(hsum, f.half()));
                need(2);
#pragma unroll
                for (int mu = 0; mu < D; ++mu) {
                    acc[mu] = f.mad(nhh, l[mu], acc[mu]);
                    acc[mu] = f.mad(nhh, h[mu], acc[mu]);
                }
                E v[D];
                if (L < m) {
                    const int own = tt_row(n, i, L);
                    const E w = Wt[own - n];
#pragma unroll
                    for (int mu = 0; mu < D; ++mu) v[mu] = f.mul(f.reduce(acc[mu]), w);
                    st_vec<F, D>(rec + own * D, v);
                    const E c2 = f.reduce(dot_plain<F, D>(f, x2, v));             // 2 P_{i,j} . J(i..j)
                    Ut[own] = f.add(c2, hsum);
                    Vt[own] = f.sub(c2, hsum);
                } else {
#pragma unroll
                    for (int mu = 0; mu < D; ++mu) v[mu] = f.reduce(acc[mu]);
                    E e[D], ne[D];
                    ld_vec<F, D>(rec + m * D, e);
                    lower_neg<F, MET, D>(f, 0, e, ne);
                    const E nout = f.reduce(dot_plain<F, D>(f, ne, v));
                    prm.out[((pbase + pt) * n_ord + o) * states + s] = f.to_output(f.neg(nout));
                }
                if (prm.currents) {
                    E* dst = prm.currents + (pt * m * m + (long long)(i - 1) * m + (i + L - 2)) * D;
#pragma unroll
                    for (int mu = 0; mu < D; ++mu) dst[mu] = f.to_output(v[mu]);
                }
            }
        }
        if (prm.currents)
            for (int c = 0; c < m; ++c) {
                E* dst = prm.currents + (pt * m * m + (long long)c * m + c) * D;
                for (int mu = 0; mu < D; ++mu) dst[mu] = f.to_output(rec[c * D + mu]);
            }
    }
    }
}

}  // namespace bg
