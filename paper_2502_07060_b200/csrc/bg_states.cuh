// bg_states.cuh -- device construction of the d-dimensional, square-root-free polarisation states
// of PAPER.md §2.3 (Eqs.(8)-(18)) from a massless d-vector k and a massless
// 4-vector chi: SURVEY.md 8(f) row f1.  The paper prepares these on the host with lips/syngular
// (PAPER.md:168); here one thread builds the D-2 states eps_x and their duals eps~_x of one vector.
//
//   k_4d = (k^0..k^3),  mu^2 = (k_4d, k_4d),  kb = k_4d - mu^2/(2 (chi, k_4d)) chi          Eqs.(9),(10)
//   eps_1 = <kb|gamma^mu|chi] / (2 [kb chi]),  eps_2 = [kb|gamma^mu|chi> / <kb chi>         Eq.(18)
//   eps~_1 = eps_2, eps~_2 = eps_1
//   eps_3 = kb - mu^2/(2 (chi, k_4d)) chi,  eps~_3 = eps_3 / mu^2
//   eps_4 = (0,0,0,0, k_5, -k_4, 0..),  eps~_4 = eps_4 / mu_6^2
//   eps_x = (0,0,0,0, k_4 k_q, .., k_{q-1} k_q, -mu_q^2, 0..),  q = x + 1 >= 6               Eq.(16)
//   eps~_x = eps_x / (mu_q^2 mu_{q+1}^2),  mu_q^2 = k_4^2 + .. + k_{q-1}^2                    Eq.(17)
//
// Readings R13-R15 of DESIGN.md (bracket normalisation, the index shift of Eq.(16), the signs
// s_y = -g_yy of the alternating metric).  Spinors are kept UNNORMALISED to save inversions:
// with M = [[M00, M01], [M10, M11]] the matrix of a massless 4-vector, lam = (M00, M10) and
// lamt' = (M00, M01) (= M00 lamt), so that
//   eps_1 = vec(lam_kb lamt'_chi^T) M00(kb) / [kb chi]',  eps_2 = 2 vec(lam_chi lamt'_kb^T) / (M00(kb) <kb chi>).
// All denominators of a vector are inverted with Montgomery's trick in two rounds (the second
// needs kb): two field inversions per vector over F_p.
#pragma once
#include "bg_field.cuh"

namespace bg {

constexpr int kMaxD = 16;

// metric at run time (this is not the hot path)
__device__ __forceinline__ bool metric_minus(int metric, int mu) { return metric == 0 ? mu >= 1 : (mu & 1) == 1; }

template <class F>
struct SpinorConsts {
    typename F::E jm;     // M01 = p1 - jm p2, M10 = p1 + jm p2: sqrt(-1) (mostly minus) or -1 (alternating)
    typename F::E jv;     // vec component 2 = jv (N01 - N10)/2:  sqrt(-1) (mostly minus) or +1 (alternating)
};

template <class F>
__device__ __forceinline__ typename F::E mdot4(const F& f, int metric, const typename F::E* x, const typename F::E* y)
{
    typename F::A s = f.zero();
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        const typename F::E xm = metric_minus(metric, mu) ? f.neg(x[mu]) : x[mu];
        s = f.mad(xm, f.canon(y[mu]), s);
    }
    return f.reduce(s);
}

// the 4-vector of the bispinor a b^T, times `scale`
template <class F>
__device__ __forceinline__ void bispinor_vec(const F& f, const SpinorConsts<F>& sc, const typename F::E (&a)[2],
                                             const typename F::E (&b)[2], typename F::E scale, typename F::E* out)
{
    typedef typename F::E E;
    const E N00 = f.mul(a[0], b[0]), N01 = f.mul(a[0], b[1]), N10 = f.mul(a[1], b[0]), N11 = f.mul(a[1], b[1]);
    const E hs = f.mul(f.half(), scale);
    out[0] = f.mul(hs, f.add(N00, N11));
    out[1] = f.mul(hs, f.add(N01, N10));
    out[2] = f.mul(f.mul(hs, sc.jv), f.sub(N01, N10));
    out[3] = f.mul(hs, f.sub(N00, N11));
}

template <class F>
__device__ __forceinline__ void spinors_unnormalised(const F& f, const SpinorConsts<F>& sc, const typename F::E* p,
                                                     typename F::E (&lam)[2], typename F::E (&lamt)[2])
{
    const typename F::E jp2 = f.mul(sc.jm, p[2]);
    lam[0] = lamt[0] = f.add(p[0], p[3]);            // M00
    lam[1] = f.add(p[1], jp2);                       // M10
    lamt[1] = f.sub(p[1], jp2);                      // M01
}

// inverses of cnt values in place (cnt <= kMaxD); returns false if one of them is zero (inv(0) := 0)
template <class F>
__device__ __forceinline__ bool batch_inverse(const F& f, typename F::E* v, int cnt)
{
    typedef typename F::E E;
    bool ok = true;
    if constexpr (F::kExact) {
        E pre[kMaxD];
        E c = f.one();
        for (int i = 0; i < cnt; ++i) {
            pre[i] = c;
            const bool z = f.is_zero(f.canon(v[i]));
            ok = ok && !z;
            c = f.mul(c, z ? f.one() : v[i]);
        }
        E u = f.inv(c);
        for (int i = cnt - 1; i >= 0; --i) {
            const bool z = f.is_zero(f.canon(v[i]));
            const E x = v[i];
            v[i] = z ? f.ezero() : f.mul(u, pre[i]);
            u = f.mul(u, z ? f.one() : x);
        }
    } else {
        for (int i = 0; i < cnt; ++i) {
            ok = ok && !f.is_zero(v[i]);
            v[i] = f.inv(v[i]);
        }
    }
    return ok;
}

// The D-2 states of one vector.  k: d elements (internal form), chi: 4 elements; eps, til: [d-2][d]
// written through `store(row, mu, value)` callbacks so that callers choose the destination.  Returns
// false when a denominator of Eqs.(10),(16)-(18) vanishes (the states are then undefined; zeros and
// inv(0) = 0 propagate).
template <class F, class StoreEps, class StoreTil>
__device__ bool build_states(const F& f, const SpinorConsts<F>& sc, int metric, int d, const typename F::E* k,
                             const typename F::E* chi, StoreEps store_eps, StoreTil store_til)
{
    typedef typename F::E E;
    const E zero = f.ezero();
    // s_y = -g_yy and mu_q^2 = sum_{4 <= y < q} s_y k_y^2 (Eq.(17), reading R15)
    E musq[kMaxD + 1];
    musq[4] = zero;
    for (int q = 5; q <= d; ++q) {
        const E t = f.mul(k[q - 1], k[q - 1]);
        musq[q] = metric_minus(metric, q - 1) ? f.add(musq[q - 1], t) : f.sub(musq[q - 1], t);
    }
    const E mu2 = mdot4<F>(f, metric, k, k);                        // = musq[d] for a massless k
    // round 1 of inversions: 2 (chi, k_4d), mu^2, and the normalisations of eps_4 .. eps_{d-2}
    E inv1[kMaxD];
    int cnt = 0;
    inv1[cnt++] = f.dbl(mdot4<F>(f, metric, chi, k));
    if (d >= 5) inv1[cnt++] = mu2;
    for (int q = 5; q < d; ++q) {
        const bool sq = !metric_minus(metric, q);                   // s_q < 0
        E den;
        if (q == 5) {
            const bool s45 = metric_minus(metric, 4) == metric_minus(metric, 5);     // s_4 s_5 > 0
            den = s45 ? musq[6] : f.neg(musq[6]);
        } else {
            den = f.mul(musq[q], musq[q + 1]);
            if (sq) den = f.neg(den);
        }
        inv1[cnt++] = den;
    }
    bool ok = batch_inverse<F>(f, inv1, cnt);
    const E c = f.mul(mu2, inv1[0]);                                // mu^2 / (2 (chi, k_4d))
    E kb[4];
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) kb[mu] = f.sub(k[mu], f.mul(c, chi[mu]));           // Eq.(10)
    E lk[2], ltk[2], lc[2], ltc[2];
    spinors_unnormalised<F>(f, sc, kb, lk, ltk);
    spinors_unnormalised<F>(f, sc, chi, lc, ltc);
    // round 2: [kb chi]' and M00(kb) <kb chi>; the oracle also divides by M00(kb), M00(chi)
    E inv2[2];
    inv2[0] = f.sub(f.mul(ltk[0], ltc[1]), f.mul(ltk[1], ltc[0]));
    inv2[1] = f.mul(lk[0], f.sub(f.mul(lk[0], lc[1]), f.mul(lk[1], lc[0])));
    ok = ok && !f.is_zero(f.canon(lk[0])) && !f.is_zero(f.canon(lc[0]));
    ok = batch_inverse<F>(f, inv2, 2) && ok;
    E e1[4], e2[4];
    bispinor_vec<F>(f, sc, lk, ltc, f.mul(lk[0], inv2[0]), e1);
    bispinor_vec<F>(f, sc, lc, ltk, f.dbl(inv2[1]), e2);
    for (int mu = 0; mu < d; ++mu) {
        const E a = mu < 4 ? e1[mu] : zero, b = mu < 4 ? e2[mu] : zero;
        store_eps(0, mu, a); store_til(1, mu, a);
        store_eps(1, mu, b); store_til(0, mu, b);
    }
    if (d >= 5) {
        for (int mu = 0; mu < d; ++mu) {
            const E e3 = mu < 4 ? f.sub(kb[mu], f.mul(c, chi[mu])) : zero;
            store_eps(2, mu, e3);
            store_til(2, mu, f.mul(e3, inv1[1]));
        }
    }
    for (int q = 5; q < d; ++q) {                                   // state x = q - 1
        const E iden = inv1[2 + (q - 5)];
        for (int mu = 0; mu < d; ++mu) {
            E e = zero;
            if (q == 5) {
                const bool s45 = metric_minus(metric, 4) == metric_minus(metric, 5);
                if (mu == 4) e = k[5];
                if (mu == 5) e = s45 ? f.neg(k[4]) : k[4];
            } else {
                if (mu >= 4 && mu < q) e = f.mul(k[mu], k[q]);
                if (mu == q) e = metric_minus(metric, q) ? f.neg(musq[q]) : musq[q];
            }
            store_eps(q - 2, mu, e);
            store_til(q - 2, mu, f.mul(e, iden));
        }
    }
    return ok;
}

}  // namespace bg
