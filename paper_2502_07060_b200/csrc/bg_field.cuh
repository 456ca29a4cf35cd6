// bg_field.cuh -- device number types and metrics for the Berends-Giele kernels (sm_100a).
//
// Three field policies with one interface, so every kernel is written once.  A policy is an
// OBJECT (empty for the two fields without run-time constants), constructed in the kernel from
// the launch parameters:
//
//   Fp31    F_p, p = 2^31-1 (Mersenne).  Elements are canonical uint32 residues.
//   FpMont  F_p for ANY odd prime 2^30 < p < 2^31 given at run time; elements are kept in
//           Montgomery form x 2^32 mod p, so the reduction of a 64-bit accumulator is one REDC
//           (IMAD + IMAD.WIDE + conditional subtraction).  Inputs are converted on load, results
//           on store (the paper matches Caravel's F_p values).
//   C128    complex128 on the FP64 pipe; a multiply-add is 4 DFMA.
//
// Over both prime fields sums of products are accumulated LAZILY in a uint64: `acc = a*b + acc`
// is exactly one IMAD.WIDE.U32 with a 64-bit addend.  Headroom (any odd p < 2^31, one operand of
// every product <= p, the other <= p-1): a product raises the upper accumulator word by less
// than p^2/2^32 + 1 <= p/2, so from zero an accumulator takes kCap0 = 4 products (upper word
// < 2p); relief() subtracts p 2^32 (= 0 mod p) when the upper word allows it -- hi <- min(hi,
// hi - p), ONE VIADDMNMX.U32 -- which brings hi < p and buys kCapR = 2 more products (hi < 2p
// again).  reduce() gives the canonical residue when a value is needed as a multiplicand or
// stored.  All of it is exact field arithmetic: results are bit-identical to any other correct
// evaluation order.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace bg {

constexpr uint32_t kP = 0x7fffffffu;
constexpr int kMaxPrimes = 8;          // primes per call (bg_amplitudes_primes)

// 2^32 mod (2^31-1), read from constant memory so that it stays opaque to ptxas: with a literal 2
// the fold `hi * 2 + lo` is strength-reduced into five shift/add instructions instead of the
// single IMAD.WIDE.U32 it is meant to be.
__constant__ uint32_t c_two32 = 2u;

// ---- metric (PAPER.md:140 mostly minus; PAPER.md:188 Caravel's alternating diag(1,-1,1,-1,..)) ----
template <int MET>
struct Metric {
    static_assert(MET == 0 || MET == 1, "0: diag(+,-,-,..,-), 1: diag(+,-,+,-,..)");
    // g_{mu mu} = -1 ?
    __host__ __device__ static constexpr bool minus(int mu) { return MET == 0 ? mu >= 1 : (mu & 1) == 1; }
};

struct Fp31 {
    typedef uint32_t E;   // element
    typedef uint64_t A;   // lazy accumulator
    struct Params {};
    static constexpr int kCap0 = 4;           // products an accumulator takes starting from zero
    static constexpr int kCapR = 2;           // products an accumulator takes after relief()
    static constexpr bool kExact = true;
    static constexpr int kFieldId = 0;
    // an accumulator that starts from widen(a) instead of zero still takes kCap0 products: a < 2^31 and
    // 4 p (p-1) + 2^31 = 2^64 - 2^33 - 2^31 + 8, upper word < 2p
    static constexpr bool kWidenFree = true;

    __device__ __forceinline__ Fp31(const Params&, int) {}

    __device__ __forceinline__ E load_input(uint32_t raw) const
    {   // values >= p are reduced on load (bg.h); raw < 2^32 = 2p + 2
        uint32_t r = min(raw, raw - kP);                          // two conditional subtractions
        return min(r, r - kP);
    }
    __device__ __forceinline__ E to_output(E a) const { return canon(a); }
    __device__ __forceinline__ A zero() const { return 0ull; }
    __device__ __forceinline__ E ezero() const { return 0u; }
    __device__ __forceinline__ E one() const { return 1u; }
    __device__ __forceinline__ E half() const { return 0x40000000u; }          // 2^-1 = 2^30
    __device__ __forceinline__ bool is_zero(E a) const { return a == 0u; }
    // a*b + c: written as mul.wide + 64-bit add, which ptxas fuses into ONE IMAD.WIDE.U32 with a
    // 64-bit addend and keeps as a serial chain.  (An inline-PTX mad.wide.u32 is instead split
    // into IMAD.WIDE(..,RZ) + IADD3 + IADD3.X and re-associated: 1.9x the instructions.)
    __device__ __forceinline__ A mad(E a, E b, A c) const { return (uint64_t)a * b + c; }
    // accumulator holding the element a (counts as one product for the headroom rules)
    __device__ __forceinline__ A widen(E a) const { return (uint64_t)a; }
    // accumulator + element (counts as one product)
    __device__ __forceinline__ A addw(A x, E a) const { return x + (uint64_t)a; }
    // Headroom without touching the multiplier pipe (header comment): ONE ALU instruction.
    __device__ __forceinline__ A relief(A x) const
    {
        uint32_t lo, hi;
        asm("mov.b64 {%0, %1}, %2;" : "=r"(lo), "=r"(hi) : "l"(x));
        hi = min(hi, hi - kP);
        A r;
        asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(lo), "r"(hi));
        return r;
    }
    // canonical residue of an accumulator whose upper word is < 2p (what the headroom rules guarantee):
    // x = hi 2^32 + lo = 2 hi + (lo >> 31) + (lo & p) (mod p).  Five ALU instructions and one add, NO
    // multiplier: the FMA-heavy pipe is the binding one (71 % busy at cfg2), and the fold by 2^32 = 2 as an
    // IMAD.WIDE (rounds 1-2) spent 4 of its cycles per reduction, with both additions issued as IMAD.IADD
    // on the same pipe on top.
    __device__ __forceinline__ E reduce(A x) const
    {
        uint32_t lo, hi;
        asm("mov.b64 {%0, %1}, %2;" : "=r"(lo), "=r"(hi) : "l"(x));
        hi = min(hi, hi - kP);                                    // < p
        uint32_t s = __funnelshift_l(lo, hi, 1);                  // 2 hi + (lo >> 31) <= 2p - 1
        s = min(s, s - kP);                                       // < p
        const uint32_t r = (lo & kP) + s;                         // < 2p
        return min(r, r - kP);
    }
    __device__ __forceinline__ E neg(E a) const { return a ^ kP; }       // p - a, in [0,p]; 0 -> p
    __device__ __forceinline__ E canon(E a) const { return a == kP ? 0u : a; }
    __device__ __forceinline__ E add(E a, E b) const
    {
        uint32_t r = a + b;
        return min(r, r - kP);
    }
    __device__ __forceinline__ E sub(E a, E b) const
    {
        uint32_t r = a - b;
        return min(r, r + kP);
    }
    __device__ __forceinline__ E dbl(E a) const { return add(a, a); }
    __device__ __forceinline__ E mul(E a, E b) const
    {
        uint64_t x = (uint64_t)a * b;                              // < 2^62
        uint32_t r = (uint32_t)(x & kP) + (uint32_t)(x >> 31);
        return min(r, r - kP);
    }
    // a^(p-2) by the addition chain for 2^31-3: 30 squarings + 8 multiplications; inv(0)=0
    __device__ E inv(E a) const
    {
        auto sqn = [this](E x, int k) {
            for (int i = 0; i < k; ++i) x = mul(x, x);
            return x;
        };
        E x2 = mul(sqn(a, 1), a);        // a^(2^2-1)
        E x4 = mul(sqn(x2, 2), x2);      // 2^4-1
        E x8 = mul(sqn(x4, 4), x4);      // 2^8-1
        E x16 = mul(sqn(x8, 8), x8);     // 2^16-1
        E x24 = mul(sqn(x16, 8), x8);    // 2^24-1
        E x28 = mul(sqn(x24, 4), x4);    // 2^28-1
        E x29 = mul(sqn(x28, 1), a);     // 2^29-1
        return mul(sqn(x29, 2), a);      // 4(2^29-1)+1 = 2^31-3
    }
};

// Generic 31-bit prime, Montgomery form with R = 2^32.
struct FpMont {
    typedef uint32_t E;   // x R mod p, canonical (< p)
    typedef uint64_t A;
    struct Params {       // per prime of the call, filled by the host (bg_api.cu: mont_params)
        uint32_t p[kMaxPrimes];
        uint32_t pinv[kMaxPrimes];    // -p^-1 mod 2^32
        uint32_t r2[kMaxPrimes];      // R^2 mod p
        uint32_t one[kMaxPrimes];     // R mod p
        uint32_t half[kMaxPrimes];    // 2^-1 R mod p
    };
    static constexpr int kCap0 = 4;
    static constexpr int kCapR = 2;
    static constexpr bool kExact = true;
    static constexpr int kFieldId = 2;
    static constexpr bool kWidenFree = false;  // widen(a) = a R is a product like any other
    uint32_t p, pinv, r2, one_, half_;

    __device__ __forceinline__ FpMont(const Params& q, int i)
        : p(q.p[i]), pinv(q.pinv[i]), r2(q.r2[i]), one_(q.one[i]), half_(q.half[i]) {}

    // REDC: t 2^-32 mod p for t < p 2^32; canonical result
    __device__ __forceinline__ E redc(A t) const
    {
        const uint32_t m = (uint32_t)t * pinv;
        const A s = (uint64_t)m * p + t;                          // < 2 p 2^32 < 2^64, low word 0
        const uint32_t r = (uint32_t)(s >> 32);                   // < 2p
        return min(r, r - p);
    }
    __device__ __forceinline__ E load_input(uint32_t raw) const
    {   // raw < 2^32 < 4p: reduce, then to Montgomery form
        uint32_t r = min(raw, raw - 2u * p);
        r = min(r, r - p);
        return redc((uint64_t)r * r2);
    }
    __device__ __forceinline__ E to_output(E a) const { return redc((uint64_t)canon(a)); }   // out of Montgomery form
    __device__ __forceinline__ A zero() const { return 0ull; }
    __device__ __forceinline__ E ezero() const { return 0u; }
    __device__ __forceinline__ E one() const { return one_; }
    __device__ __forceinline__ E half() const { return half_; }
    __device__ __forceinline__ bool is_zero(E a) const { return a == 0u; }
    __device__ __forceinline__ A mad(E a, E b, A c) const { return (uint64_t)a * b + c; }
    // accumulators hold products of two Montgomery forms (scale R^2): an element enters as a * R
    __device__ __forceinline__ A widen(E a) const { return (uint64_t)a * one_; }
    __device__ __forceinline__ A addw(A x, E a) const { return (uint64_t)a * one_ + x; }
    __device__ __forceinline__ A relief(A x) const
    {
        uint32_t lo, hi;
        asm("mov.b64 {%0, %1}, %2;" : "=r"(lo), "=r"(hi) : "l"(x));
        hi = min(hi, hi - p);
        A r;
        asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(lo), "r"(hi));
        return r;
    }
    // canonical Montgomery form of (sum of products of Montgomery forms) : upper word < 2p on entry
    __device__ __forceinline__ E reduce(A x) const { return redc(relief(x)); }
    __device__ __forceinline__ E neg(E a) const { return p - a; }         // in [0,p]; 0 -> p
    __device__ __forceinline__ E canon(E a) const { return a == p ? 0u : a; }
    __device__ __forceinline__ E add(E a, E b) const
    {
        uint32_t r = a + b;
        return min(r, r - p);
    }
    __device__ __forceinline__ E sub(E a, E b) const
    {
        uint32_t r = a - b;
        return min(r, r + p);
    }
    __device__ __forceinline__ E dbl(E a) const { return add(a, a); }
    __device__ __forceinline__ E mul(E a, E b) const { return redc((uint64_t)a * b); }
    // a^(p-2), square and multiply over the bits of the exponent; inv(0) = 0
    __device__ E inv(E a) const
    {
        E r = one_, b = a;
        for (uint32_t e = p - 2u; e; e >>= 1) {
            if (e & 1u) r = mul(r, b);
            b = mul(b, b);
        }
        return a == 0u ? 0u : r;
    }
};

struct C128 {
    typedef double2 E;
    typedef double2 A;
    struct Params {};
    static constexpr int kCap0 = 1 << 30;     // never needs relief
    static constexpr int kCapR = 1 << 30;
    static constexpr bool kExact = false;
    static constexpr int kFieldId = 1;
    static constexpr bool kWidenFree = true;

    __device__ __forceinline__ C128(const Params&, int) {}

    __device__ __forceinline__ E load_input(double2 raw) const { return raw; }
    __device__ __forceinline__ E to_output(E a) const { return a; }
    __device__ __forceinline__ A zero() const { return make_double2(0.0, 0.0); }
    __device__ __forceinline__ E ezero() const { return make_double2(0.0, 0.0); }
    __device__ __forceinline__ E one() const { return make_double2(1.0, 0.0); }
    __device__ __forceinline__ E half() const { return make_double2(0.5, 0.0); }
    __device__ __forceinline__ bool is_zero(E a) const { return a.x == 0.0 && a.y == 0.0; }
    __device__ __forceinline__ A mad(E a, E b, A c) const
    {
        double re = fma(a.x, b.x, c.x);
        re = fma(-a.y, b.y, re);
        double im = fma(a.x, b.y, c.y);
        im = fma(a.y, b.x, im);
        return make_double2(re, im);
    }
    __device__ __forceinline__ A widen(E a) const { return a; }
    __device__ __forceinline__ A addw(A x, E a) const { return make_double2(x.x + a.x, x.y + a.y); }
    __device__ __forceinline__ A relief(A x) const { return x; }
    __device__ __forceinline__ E reduce(A x) const { return x; }
    __device__ __forceinline__ E neg(E a) const { return make_double2(-a.x, -a.y); }
    __device__ __forceinline__ E canon(E a) const { return a; }
    __device__ __forceinline__ E add(E a, E b) const { return make_double2(a.x + b.x, a.y + b.y); }
    __device__ __forceinline__ E sub(E a, E b) const { return make_double2(a.x - b.x, a.y - b.y); }
    __device__ __forceinline__ E dbl(E a) const { return make_double2(2.0 * a.x, 2.0 * a.y); }
    __device__ __forceinline__ E mul(E a, E b) const
    {
        return make_double2(fma(a.x, b.x, -(a.y * b.y)), fma(a.x, b.y, a.y * b.x));
    }
    __device__ __forceinline__ E inv(E a) const
    {   // 1/z = conj(z)/|z|^2 ; inv(0) := 0 (bg.h)
        double n2 = fma(a.x, a.x, a.y * a.y);
        if (n2 == 0.0) return make_double2(0.0, 0.0);
        double r = 1.0 / n2;
        return make_double2(a.x * r, -a.y * r);
    }
};

}  // namespace bg
