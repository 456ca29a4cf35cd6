// bg_field.cuh -- device number types for the Berends-Giele kernels (sm_100a).
//
// Two policies with one interface, so the recursion kernel is written once:
//
//   Fp31  F_p, p = 2^31-1 (Mersenne).  Elements are canonical uint32 residues.  Sums of
//         products are accumulated LAZILY in a uint64: `acc = a*b + acc` is exactly one
//         IMAD.WIDE.U32, so a modular multiply-add costs one FMA-pipe issue slot and no
//         ALU work; an accumulator is folded (2^32 = 2 mod p, one more IMAD.WIDE) before it
//         can overflow and reduced to a canonical residue only when the value is needed as
//         a multiplicand or stored.  Subtraction is addition of p - x = x XOR p (one LOP3).
//         All of it is exact field arithmetic: results are bit-identical to any other
//         correct evaluation order.
//   C128  complex128 on the FP64 pipe; accumulators are plain complex numbers, a
//         multiply-add is 4 DFMA.
//
// Headroom rules for Fp31 (p^2 < 2^62):
//   fold(x) <= 2*(2^32-1) + (2^32-1) < 3*2^32, and 3*2^32 + 4*p^2 < 2^64, so after a fold
//   (or from zero) an accumulator takes FOUR more products of operands <= p.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace bg {

constexpr uint32_t kP = 0x7fffffffu;

// 2^32 mod p, read from constant memory so that it stays opaque to ptxas: with a literal 2
// the fold `hi * 2 + lo` is strength-reduced into five shift/add instructions instead of the
// single IMAD.WIDE.U32 it is meant to be.
__constant__ uint32_t c_two32 = 2u;

struct Fp31 {
    typedef uint32_t E;   // element
    typedef uint64_t A;   // lazy accumulator
    static constexpr int kCap = 4;            // products an accumulator takes between folds
    static constexpr int kCap0 = 4;           // products an accumulator takes starting from zero
    static constexpr int kCapR = 2;           // products an accumulator takes after relief()
    static constexpr bool kExact = true;

    __device__ __forceinline__ static E load_input(uint32_t raw)
    {   // values >= p are reduced on load (bg.h); raw < 2^32 = 2p + 2
        uint32_t r = min(raw, raw - kP);                          // two conditional subtractions
        return min(r, r - kP);
    }
    __device__ __forceinline__ static A zero() { return 0ull; }
    __device__ __forceinline__ static E ezero() { return 0u; }
    __device__ __forceinline__ static E one() { return 1u; }
    __device__ __forceinline__ static bool is_zero(E a) { return a == 0u; }
    // a*b + c: written as mul.wide + 64-bit add, which ptxas fuses into ONE IMAD.WIDE.U32 with a
    // 64-bit addend and keeps as a serial chain.  (An inline-PTX mad.wide.u32 is instead split
    // into IMAD.WIDE(..,RZ) + IADD3 + IADD3.X and re-associated: 1.9x the instructions,
    // profiles/r01a_cfg2_sweep_w4_opmix.txt.)
    __device__ __forceinline__ static A mad(E a, E b, A c) { return (uint64_t)a * b + c; }
    __device__ __forceinline__ static A widen(E a) { return (uint64_t)a; }
    __device__ __forceinline__ static A accumulate(A c, E a) { return c + (uint64_t)a; }
    __device__ __forceinline__ static E half() { return 0x40000000u; }          // 2^-1 = 2^30
    // x = hi 2^32 + lo = 2 hi + lo (mod p), result < 3*2^32.  Written in place -- add 2 hi to
    // the whole accumulator (one IMAD.WIDE.U32), then take hi off the upper word (one IADD) --
    // so that no register pair has to be rebuilt around the low word.
    __device__ __forceinline__ static A fold(A x)
    {
        // the word split / join is opaque inline PTX (register renaming only) so that the
        // compiler cannot rewrite this back into "rebuild (lo, 0), then multiply-add"
        uint32_t lo, hi, tl, th;
        asm("mov.b64 {%0, %1}, %2;" : "=r"(lo), "=r"(hi) : "l"(x));
        const A t = mad(hi, c_two32, x);
        asm("mov.b64 {%0, %1}, %2;" : "=r"(tl), "=r"(th) : "l"(t));
        th -= hi;
        A r;
        asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(tl), "r"(th));
        return r;
    }
    // Headroom without touching the multiplier pipe: subtract p 2^32 (= 0 mod p) when the upper
    // word allows it, hi <- min(hi, hi - p) (unsigned): ONE ALU instruction (VIADDMNMX.U32).
    // A product of an operand <= p with one <= p-1 raises the upper word by at most 2^30 - 1
    // (carry included), so from zero an accumulator takes kCap0 = 4 products (hi <= 2^32 - 4),
    // relief() brings hi <= 2^31 - 2, and every relief() buys kCapR = 2 more products.
    // (IMAD.WIDE.U32 issues at a quarter of the ALU rate on sm_100 -- profiles/r01b -- so the
    // fold above, one more IMAD.WIDE, is kept for the final reduce only.)
    __device__ __forceinline__ static A relief(A x)
    {
        uint32_t lo, hi;
        asm("mov.b64 {%0, %1}, %2;" : "=r"(lo), "=r"(hi) : "l"(x));
        hi = min(hi, hi - kP);
        A r;
        asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(lo), "r"(hi));
        return r;
    }
    // canonical residue of y < 2^62 + 2^33 (so that (y>>31) + (y&p) < 2^32)
    __device__ __forceinline__ static E reduce62(A y)
    {
        uint32_t r = (uint32_t)(y & kP) + (uint32_t)(y >> 31);   // < 2^32
        r = (r & kP) + (r >> 31);                                 // <= p + 1
        return min(r, r - kP);
    }
    // canonical residue of any 64-bit accumulator
    __device__ __forceinline__ static E reduce(A x)
    {
        A t = fold(x);                                            // < 3*2^32
        uint32_t r = (uint32_t)(t & kP) + (uint32_t)(t >> 31);    // < 2^31 + 6
        return min(r, r - kP);
    }
    // canonical residue of x/2:  2^-1 = 2^30, so x/2 = hi 2^31 + lo 2^30 = hi + lo 2^30
    __device__ __forceinline__ static E reduce_half(A x)
    {
        A t = (uint64_t)(uint32_t)x * 0x40000000u + (uint32_t)(x >> 32);   // < 2^62 + 2^32
        // three 31-bit limbs (the top one is 0 or 1): the sum cannot overflow 32 bits
        uint32_t r = (uint32_t)(t & kP) + ((uint32_t)(t >> 31) & kP) + (uint32_t)(t >> 62);
        r = (r & kP) + (r >> 31);                                           // <= p + 1
        return min(r, r - kP);
    }
    // canonical residue of 2x
    __device__ __forceinline__ static E reduce_double(A x) { return dbl(reduce(x)); }
    __device__ __forceinline__ static E neg(E a) { return a ^ kP; }       // p - a, in [0,p]; 0 -> p
    __device__ __forceinline__ static E canon(E a) { return a == kP ? 0u : a; }
    __device__ __forceinline__ static E add(E a, E b)
    {
        uint32_t r = a + b;
        return min(r, r - kP);
    }
    __device__ __forceinline__ static E sub(E a, E b)
    {
        uint32_t r = a - b;
        return min(r, r + kP);
    }
    __device__ __forceinline__ static E dbl(E a) { return add(a, a); }
    __device__ __forceinline__ static E mul(E a, E b)
    {
        uint64_t x = (uint64_t)a * b;                              // < 2^62
        uint32_t r = (uint32_t)(x & kP) + (uint32_t)(x >> 31);
        return min(r, r - kP);
    }
    // a^(p-2) by the addition chain for 2^31-3: 30 squarings + 8 multiplications; inv(0)=0
    __device__ static E inv(E a)
    {
        auto sqn = [](E x, int k) {
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

struct C128 {
    typedef double2 E;
    typedef double2 A;
    static constexpr int kCap = 1 << 30;      // never needs folding
    static constexpr int kCap0 = 1 << 30;
    static constexpr int kCapR = 1 << 30;
    static constexpr bool kExact = false;

    __device__ __forceinline__ static E load_input(double2 raw) { return raw; }
    __device__ __forceinline__ static A zero() { return make_double2(0.0, 0.0); }
    __device__ __forceinline__ static E ezero() { return make_double2(0.0, 0.0); }
    __device__ __forceinline__ static E one() { return make_double2(1.0, 0.0); }
    __device__ __forceinline__ static bool is_zero(E a) { return a.x == 0.0 && a.y == 0.0; }
    __device__ __forceinline__ static A mad(E a, E b, A c)
    {
        double re = fma(a.x, b.x, c.x);
        re = fma(-a.y, b.y, re);
        double im = fma(a.x, b.y, c.y);
        im = fma(a.y, b.x, im);
        return make_double2(re, im);
    }
    __device__ __forceinline__ static A widen(E a) { return a; }
    __device__ __forceinline__ static A accumulate(A c, E a) { return make_double2(c.x + a.x, c.y + a.y); }
    __device__ __forceinline__ static E half() { return make_double2(0.5, 0.0); }
    __device__ __forceinline__ static A fold(A x) { return x; }
    __device__ __forceinline__ static A relief(A x) { return x; }
    __device__ __forceinline__ static E reduce(A x) { return x; }
    __device__ __forceinline__ static E reduce_half(A x) { return make_double2(0.5 * x.x, 0.5 * x.y); }
    __device__ __forceinline__ static E reduce_double(A x) { return make_double2(2.0 * x.x, 2.0 * x.y); }
    __device__ __forceinline__ static E neg(E a) { return make_double2(-a.x, -a.y); }
    __device__ __forceinline__ static E canon(E a) { return a; }
    __device__ __forceinline__ static E add(E a, E b) { return make_double2(a.x + b.x, a.y + b.y); }
    __device__ __forceinline__ static E sub(E a, E b) { return make_double2(a.x - b.x, a.y - b.y); }
    __device__ __forceinline__ static E dbl(E a) { return make_double2(2.0 * a.x, 2.0 * a.y); }
    __device__ __forceinline__ static E mul(E a, E b)
    {
        return make_double2(fma(a.x, b.x, -(a.y * b.y)), fma(a.x, b.y, a.y * b.x));
    }
    __device__ __forceinline__ static E inv(E a)
    {   // 1/z = conj(z)/|z|^2 ; inv(0) := 0 (bg.h)
        double n2 = fma(a.x, a.x, a.y * a.y);
        if (n2 == 0.0) return make_double2(0.0, 0.0);
        double r = 1.0 / n2;
        return make_double2(a.x * r, -a.y * r);
    }
};

}  // namespace bg
