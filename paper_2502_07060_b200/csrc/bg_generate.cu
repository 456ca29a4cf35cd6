// bg_generate.cu -- bg_generate(): the seeded phase-space generator ON THE DEVICE (SURVEY.md 8(f)
// row f1; the paper prepares momenta and states on the host, and names offloading
// that stage as possible future work).  One thread per phase-space point; the recipe is exactly
// BASELINE.json:configs' generator as restated in DESIGN.md §4 (the host version is
// paper_2502_07060_b200/inputs.py, which is this kernel's reference in the tests):
//
//   * counter-based RNG: draw c of point b, attempt a = SplitMix64 finaliser of key(seed,b,a) + c GOLDEN;
//   * massless vectors from light-cone data: p- = -(sum_{mu>=2} g_mu p_mu^2)/(2 p+), p0 = p+ + p-/2,
//     p1 = p+ - p-/2 (metric: PAPER.md:140, or the alternating one of PAPER.md:188);
//   * p_1..p_{n-2} free, K = -sum p_i, q massless, p_{n-1} = alpha q with alpha = K^2/(2 K.q),
//     p_n = K - p_{n-1};  eps_i = v_i - (v_i.p_i)/(r_i.p_i) r_i, or (d = 4) the spinor-helicity states
//     eps_-(k;r) = vec(lam_k lamt_r^T)/[r k], eps_+(k;r) = 2 vec(lam_r lamt_k^T)/<r k> (Eq.(11));
//   * F_p: points with K.q = 0, r_i.p_i = 0, a vanishing proper P_{i,j}^2 (or, with helicity states, a
//     vanishing M00 of k_i or r_i) are redrawn with attempt + 1.
//
// Over F_p the output is bit-identical to inputs.py (exact arithmetic); over complex128 it agrees to
// rounding (numpy sums and divides in its own order).  The 2n-1 light-cone 1/(2p+) go through Montgomery's
// trick; alpha and the polarisation coefficient of every leg cost one field inversion each.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/bg.h"
#include "bg_host_util.h"
#include "bg_states.cuh"

namespace {

using bg::C128;
using bg::Fp31;
using bg::FpMont;

constexpr uint64_t GOLDEN = 0x9E3779B97F4A7C15ull, M1 = 0xBF58476D1CE4E5B9ull, M2 = 0x94D049BB133111EBull;
constexpr int kMaxAttempts = 64;

__host__ __device__ inline uint64_t mix64(uint64_t z)
{
    z = (z ^ (z >> 30)) * M1;
    z = (z ^ (z >> 27)) * M2;
    return z ^ (z >> 31);
}

template <class F>
struct GenParams {
    typedef typename F::E E;
    E* mom;                   // [batch][n][d]
    E* pol;                   // [batch][n][d]
    E* ref;                   // NULL or [batch][n][d]: the reference vectors r_i
    unsigned long long* redraws;   // NULL or one device counter (incremented)
    long long batch, start;
    uint64_t seed;
    int n, d, metric;
    int use_hel;
    signed char hel[16];
    uint32_t p;               // F_p: the prime
    uint64_t rec_p, rec_pm1;  // floor((2^64-1)/p), floor((2^64-1)/(p-1))
    bg::SpinorConsts<F> sc;
    typename F::Params fld;
};

__device__ __forceinline__ uint32_t mod_u64(uint64_t u, uint32_t m, uint64_t rec)
{   // u mod m with the precomputed reciprocal rec = floor((2^64-1)/m): the quotient estimate is at most 2 low
    uint64_t r = u - __umul64hi(u, rec) * m;
    while (r >= m) r -= m;
    return (uint32_t)r;
}

// element e (0-based) of the point's stream: F_p uniform in [1,p) or in [0,p); complex (re, im) from two draws
template <class F>
struct Draws {
    uint64_t key;
    const GenParams<F>& prm;
    const F& f;
    __device__ __forceinline__ uint64_t draw(long long c) const { return mix64(key + (uint64_t)c * GOLDEN); }
    __device__ __forceinline__ typename F::E nonzero(int e) const
    {
        if constexpr (F::kExact) return f.load_input(1u + mod_u64(draw(e + 1), prm.p - 1u, prm.rec_pm1));
        else return any(e);
    }
    __device__ __forceinline__ typename F::E any(int e) const
    {
        if constexpr (F::kExact) {
            return f.load_input(mod_u64(draw(e + 1), prm.p, prm.rec_p));
        } else {
            const double re = (double)(draw(2 * e + 1) >> 11) * 0x1p-52 - 1.0;
            const double im = (double)(draw(2 * e + 2) >> 11) * 0x1p-52 - 1.0;
            return make_double2(re, im);
        }
    }
};

// (not inlined: four call sites of a 38-multiplication chain took the kernel to 59 KB of code, past the instruction
// cache: `no_instruction` 23 % of the stall samples)
template <class F>
__device__ __noinline__ typename F::E inv_call(const F& f, typename F::E a) { return f.inv(a); }

template <class F>
__device__ __forceinline__ typename F::E mdot(const F& f, int metric, int d, const typename F::E* x,
                                              const typename F::E* y)
{
    typename F::A s = f.zero();
    for (int mu = 0; mu < d; ++mu) {
        const typename F::E xm = bg::metric_minus(metric, mu) ? f.neg(x[mu]) : x[mu];
        s = f.relief(s);
        s = f.mad(xm, f.canon(y[mu]), s);
    }
    return f.reduce(s);
}

// light-cone -> Cartesian: out[0..d) from p+ = stream element e0, p_perp = elements e0+1 .. e0+d-2,
// inv2plus = 1/(2 p+)
template <class F>
__device__ __forceinline__ void massless(const F& f, const Draws<F>& dr, int metric, int d, int e0,
                                         typename F::E inv2plus, typename F::E* out)
{
    typedef typename F::E E;
    const E plus = dr.nonzero(e0);
    E perp2 = f.ezero();
    for (int mu = 2; mu < d; ++mu) {
        const E x = dr.nonzero(e0 + mu - 1);
        out[mu] = x;
        const E sq = f.mul(x, x);
        perp2 = bg::metric_minus(metric, mu) ? f.add(perp2, sq) : f.sub(perp2, sq);     // -(g_mu x^2)
    }
    const E half = f.mul(f.mul(perp2, inv2plus), f.half());      // p-/2
    out[0] = f.add(plus, half);
    out[1] = f.sub(plus, half);
}

// The point's vectors live in thread-local arrays (local memory is interleaved by thread, so the same element of
// neighbouring points is contiguous: conflict-free, cached in L1/L2) -- shared-memory tiles limited the kernel to
// 256 resident threads per SM, and its long dependent chains (three field inversions per point) need many more.
template <class F, int MAXND>
__global__ void __launch_bounds__(128) generate_kernel(const GenParams<F> prm)
{
    typedef typename F::E E;
    const F f(prm.fld, 0);
    const int n = prm.n, d = prm.d, nd = n * d, metric = prm.metric;
    const long long pt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = pt < prm.batch;

    if (live) {
        E km[MAXND], scr[4 * 16];                              // momenta; the light-cone inverses and 2 p+
        const uint64_t index = (uint64_t)(prm.start + pt);
        const int eq = (n - 2) * (d - 1);                      // first stream element of q
        const int ev = (n - 1) * (d - 1);                      // first stream element of the (v_i, r_i) block
        int attempt = 0;
        for (;; ++attempt) {
            uint64_t key = mix64(prm.seed + GOLDEN);
            key = mix64(key ^ (index * M1 + GOLDEN));
            key = mix64(key ^ ((uint64_t)attempt * M2 + GOLDEN));
            const Draws<F> dr{key, prm, f};
            bool ok = true;
            // ---- round A: 1/(2 p+) of every light-cone vector (free legs, q, r_1..r_n); p+ != 0 --------
            E* invA = scr;                                     // [2n-1]
            auto plus_elem = [&](int j) {
                return j < n - 2 ? j * (d - 1) : j == n - 2 ? eq : ev + (j - (n - 1)) * (2 * d - 1) + d;
            };
            if constexpr (F::kExact) {
                E* xp = scr + 32;                              // 2 p+ of every light-cone vector: drawn once
                E c = f.one();
                for (int j = 0; j < 2 * n - 1; ++j) {
                    invA[j] = c;
                    xp[j] = f.dbl(dr.nonzero(plus_elem(j)));
                    c = f.mul(c, xp[j]);
                }
                E u = inv_call<F>(f, c);
                for (int j = 2 * n - 2; j >= 0; --j) {
                    invA[j] = f.mul(u, invA[j]);
                    u = f.mul(u, xp[j]);
                }
            } else {
                for (int j = 0; j < 2 * n - 1; ++j) invA[j] = inv_call<F>(f, f.dbl(dr.nonzero(plus_elem(j))));
            }
            // ---- momenta ---------------------------------------------------------------------------------
            E ksum[bg::kMaxD], q[bg::kMaxD];
            for (int mu = 0; mu < d; ++mu) ksum[mu] = f.ezero();
            for (int i = 0; i < n - 2; ++i) {
                massless<F>(f, dr, metric, d, i * (d - 1), invA[i], km + i * d);
                for (int mu = 0; mu < d; ++mu) ksum[mu] = f.add(ksum[mu], km[i * d + mu]);
            }
            massless<F>(f, dr, metric, d, eq, invA[n - 2], q);
            for (int mu = 0; mu < d; ++mu) ksum[mu] = f.canon(f.neg(ksum[mu]));           // K
            const E K2 = mdot<F>(f, metric, d, ksum, ksum), Kq = mdot<F>(f, metric, d, ksum, q);
            if (F::kExact && f.is_zero(f.canon(Kq))) ok = false;
            const E alpha = f.mul(K2, inv_call<F>(f, f.dbl(Kq)));                                   // round B
            for (int mu = 0; mu < d; ++mu) {
                const E a = f.mul(alpha, q[mu]);
                km[(n - 2) * d + mu] = a;
                km[(n - 1) * d + mu] = f.sub(ksum[mu], a);
            }
            // ---- polarisations, leg by leg: v_i, r_i, eps_i = v_i - (v_i.p_i)/(r_i.p_i) r_i (or the helicity state on
            //      (k_i, r_i)), stored at once (a redraw overwrites them).  One field inversion per leg instead of
            //      Montgomery's trick over the legs: that needed every v_i and r_i kept until the common inverse was
            //      known -- 2 n d more words of thread-local memory, which spilled through L2 into HBM (3.2 GB of DRAM
            //      traffic per 2^20 cfg2 points against 0.8 GB of output, `long_scoreboard` 73 % of the stall samples).
            E* gp = prm.pol + pt * nd;
            E* gr = prm.ref ? prm.ref + pt * nd : nullptr;
            for (int i = 0; i < n; ++i) {
                const int e0 = ev + i * (2 * d - 1);
                E v[bg::kMaxD], r[bg::kMaxD];
                for (int mu = 0; mu < d; ++mu) v[mu] = dr.any(e0 + mu);
                massless<F>(f, dr, metric, d, e0 + d, invA[n - 1 + i], r);
                const E* k = km + i * d;
                if (!prm.use_hel) {
                    const E rp = mdot<F>(f, metric, d, r, k);
                    if (F::kExact && f.is_zero(f.canon(rp))) ok = false;
                    const E coef = f.mul(mdot<F>(f, metric, d, v, k), inv_call<F>(f, f.canon(rp)));      // inv(0) = 0
                    for (int mu = 0; mu < d; ++mu) v[mu] = f.sub(v[mu], f.mul(coef, r[mu]));
                } else {
                    // spinor-helicity states on (k_i, r_i), unnormalised spinors (bg_states.cuh):
                    //   eps_- = vec(lam_k lamt'_r^T) M00(k) / [r k]',  eps_+ = 2 vec(lam_r lamt'_k^T) / (M00(k) <r k>)
                    E lk[2], ltk[2], lr[2], ltr[2], v4[4];
                    bg::spinors_unnormalised<F>(f, prm.sc, k, lk, ltk);
                    bg::spinors_unnormalised<F>(f, prm.sc, r, lr, ltr);
                    if (F::kExact && (f.is_zero(f.canon(lk[0])) || f.is_zero(f.canon(lr[0])))) ok = false;
                    const E den = prm.hel[i] < 0 ? f.sub(f.mul(ltr[0], ltk[1]), f.mul(ltr[1], ltk[0]))
                                                 : f.mul(lk[0], f.sub(f.mul(lr[0], lk[1]), f.mul(lr[1], lk[0])));
                    if (F::kExact && f.is_zero(f.canon(den))) ok = false;
                    const E dinv = inv_call<F>(f, f.canon(den));
                    if (prm.hel[i] < 0) bg::bispinor_vec<F>(f, prm.sc, lk, ltr, f.mul(lk[0], dinv), v4);
                    else bg::bispinor_vec<F>(f, prm.sc, lr, ltk, f.dbl(dinv), v4);
                    for (int mu = 0; mu < 4; ++mu) v[mu] = v4[mu];
                }
                for (int mu = 0; mu < d; ++mu) {
                    gp[i * d + mu] = f.to_output(v[mu]);
                    if (gr) gr[i * d + mu] = f.to_output(r[mu]);
                }
            }
            // ---- F_p: reject points with a vanishing proper invariant P_{i,j}^2 ------------------------------
            if constexpr (F::kExact) {
                const int m = n - 1;
                for (int i = 0; i < m && ok; ++i) {
                    E run[bg::kMaxD];
                    for (int mu = 0; mu < d; ++mu) run[mu] = km[i * d + mu];
                    for (int j = i + 1; j < m; ++j) {
                        for (int mu = 0; mu < d; ++mu) run[mu] = f.canon(f.add(run[mu], km[j * d + mu]));
                        if (i == 0 && j == m - 1) continue;
                        if (f.is_zero(f.canon(mdot<F>(f, metric, d, run, run)))) ok = false;
                    }
                }
            }
            if (ok || !F::kExact || attempt + 1 >= kMaxAttempts) break;
        }
        if (attempt && prm.redraws) atomicAdd(prm.redraws, (unsigned long long)attempt);
        // every thread stores its own point (n d contiguous elements per array; L2 merges the sectors)
        E* gm = prm.mom + pt * nd;
        for (int w = 0; w < nd; ++w) gm[w] = f.to_output(km[w]);
    }
}

template <class F>
int launch(const typename F::Params& fld, const bg::SpinorConsts<F>& sc, uint32_t p, int metric, int n, int d,
           int64_t batch, uint64_t seed, int64_t start, const signed char* hel, void* mom, void* pol, void* ref,
           unsigned long long* redraws, cudaStream_t stream)
{
    typedef typename F::E E;
    GenParams<F> prm;
    prm.mom = static_cast<E*>(mom);
    prm.pol = static_cast<E*>(pol);
    prm.ref = static_cast<E*>(ref);
    prm.redraws = redraws;
    prm.batch = batch;
    prm.start = start;
    prm.seed = seed;
    prm.n = n; prm.d = d; prm.metric = metric;
    prm.use_hel = hel != nullptr;
    for (int i = 0; i < 16; ++i) prm.hel[i] = hel && i < n ? hel[i] : 0;
    prm.p = p;
    prm.rec_p = p ? ~0ull / p : 0;
    prm.rec_pm1 = p ? ~0ull / (p - 1u) : 0;
    prm.sc = sc;
    prm.fld = fld;
    const int64_t blocks = (batch + 127) / 128;
    if (blocks > 0x7fffffffLL) return BG_ERR_ARG;
    const int nd = n * d;
    if (nd <= 64) generate_kernel<F, 64><<<(unsigned)blocks, 128, 0, stream>>>(prm);
    else if (nd <= 128) generate_kernel<F, 128><<<(unsigned)blocks, 128, 0, stream>>>(prm);
    else generate_kernel<F, 256><<<(unsigned)blocks, 128, 0, stream>>>(prm);
    return cudaGetLastError() == cudaSuccess ? BG_OK : BG_ERR_CUDA;
}

}  // namespace

extern "C" int bg_generate(int field, uint32_t prime, int metric, int n, int d, int64_t batch, uint64_t seed,
                           int64_t start, const signed char* helicities, void* momenta, void* polarisations,
                           void* references, unsigned long long* redraws, cudaStream_t stream)
{
    if (n < 4 || n > 16 || d < 4 || d > 16 || batch < 0 || start < 0) return BG_ERR_ARG;
    if (metric != BG_METRIC_MOSTLY_MINUS && metric != BG_METRIC_ALTERNATING) return BG_ERR_ARG;
    if (helicities && d != 4) return BG_ERR_ARG;
    if (batch == 0) return BG_OK;
    if (!momenta || !polarisations || momenta == polarisations) return BG_ERR_ARG;
    switch (field) {
        case BG_FIELD_FP31: {
            bg::SpinorConsts<Fp31> sc{0u, 0u};
            if (helicities && !bg_spinor_consts_fp(bg::kP, metric, nullptr, &sc.jm, &sc.jv)) return BG_ERR_UNSUPPORTED;
            return launch<Fp31>(Fp31::Params{}, sc, bg::kP, metric, n, d, batch, seed, start, helicities, momenta,
                                polarisations, references, redraws, stream);
        }
        case BG_FIELD_FPMONT: {
            FpMont::Params q{};
            if (!bg_mont_constants(prime, 0, &q)) return BG_ERR_ARG;
            bg::SpinorConsts<FpMont> sc{0u, 0u};
            if (helicities && !bg_spinor_consts_fp(prime, metric, &q, &sc.jm, &sc.jv)) return BG_ERR_UNSUPPORTED;
            return launch<FpMont>(q, sc, prime, metric, n, d, batch, seed, start, helicities, momenta, polarisations,
                                  references, redraws, stream);
        }
        case BG_FIELD_C128: {
            bg::SpinorConsts<C128> sc;
            sc.jm = metric == BG_METRIC_MOSTLY_MINUS ? make_double2(0.0, 1.0) : make_double2(-1.0, 0.0);
            sc.jv = metric == BG_METRIC_MOSTLY_MINUS ? make_double2(0.0, 1.0) : make_double2(1.0, 0.0);
            return launch<C128>(C128::Params{}, sc, 0u, metric, n, d, batch, seed, start, helicities, momenta,
                                polarisations, references, redraws, stream);
        }
    }
    return BG_ERR_ARG;
}
