/* oracle/bg_oracle.c -- CPU oracle for colour-ordered n-gluon tree amplitudes by
 * Berends-Giele recursion (arXiv:2502.07060, §2.2, Eqs.(6),(7)).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  It is a plain, slow, literal
 * implementation used only by tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py.  It shares no code, header,
 * table or helper with the CUDA path under paper_2502_07060_b200/csrc/, and
 * neither side includes or imports the other.
 *
 * What it computes (per phase-space point, points independent):
 *   out = eps_n . N(1..n-1),  N = the bracket of Eq.(6) for the (n-1)-gluon current,
 * with every lower current J(i..j) = bracket / P_{i,j}^2; see bg_recursion.inc,
 * which follows Eq.(6)/(7) term by term in the paper's order and notation.
 *
 * Metric: g = diag(+,-,...,-) or, on request, Caravel's alternating
 * diag(+,-,+,-,...) ("a modification of the metric in our code").
 *
 * Number types:
 *   field 0  F_p, p = 2^31-1 or any other prime below 2^31 given by the caller (the paper never
 *            names its prime): uint32 residues, every operation is uint64 `% p`,
 *            one Fermat inverse a^(p-2) by square-and-multiply PER propagator
 *            (no batching trick here on purpose).  Inputs >= p are reduced on load.
 *   field 1  complex128: C99 `double _Complex`, compiled with -ffp-contract=off,
 *            reciprocal as 1.0/z.
 *   field 2  the same recursion in `long double _Complex` (x87 80-bit, 64-bit
 *            mantissa) on the SAME double inputs; output as long double pairs.
 *            Used only as "truth" for the complex128 tolerance rule (R9).
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): Parke-Taylor Eq.(19)
 * (PAPER.md:186), brute-force Feynman-diagram sums n<=6 with the full symmetric
 * 3-vertex, Ward identity, cyclicity, reflection, U(1) decoupling,
 * current conservation, exact-rational cross-field homomorphism, survey worked
 * examples (tests/golden/).  Not pinned by any closed form for d>4: "d>4
 * closed-form parity unpinned" -- d>4 rests on diagrams, identities, conservation
 * and the cross-field check.
 */
#include <complex.h>
#include <stdint.h>
#include <stddef.h>

#define BG_P31 2147483647ULL

/* the prime and the metric of the evaluation in progress (set per call, per thread) */
static _Thread_local uint64_t bg_p = BG_P31;
static _Thread_local int bg_alternating = 0;
/* g_{mu mu} = -1 ?   mostly minus: every mu >= 1; alternating: odd mu */
static int metric_minus(int mu) { return bg_alternating ? (mu & 1) : (mu >= 1); }

/* ---------------------------------------------------------------- F_p ---- */
static uint32_t fp_add(uint32_t a, uint32_t b) { return (uint32_t)(((uint64_t)a + b) % bg_p); }
static uint32_t fp_sub(uint32_t a, uint32_t b) { return (uint32_t)(((uint64_t)a + bg_p - b) % bg_p); }
static uint32_t fp_mul(uint32_t a, uint32_t b) { return (uint32_t)(((uint64_t)a * b) % bg_p); }
static uint32_t fp_inv(uint32_t a)
{   /* Fermat: a^(p-2); gives 0 for a = 0 */
    uint64_t r = 1, base = a, e = bg_p - 2;
    while (e) {
        if (e & 1) r = (r * base) % bg_p;
        base = (base * base) % bg_p;
        e >>= 1;
    }
    return (uint32_t)r;
}
static uint32_t fp_load(const void* p, long idx) { return (uint32_t)(((const uint32_t*)p)[idx] % bg_p); }

#define SCALAR uint32_t
#define S_ZERO 0u
#define S_TWO 2u
#define S_ADD(a, b) fp_add(a, b)
#define S_SUB(a, b) fp_sub(a, b)
#define S_MUL(a, b) fp_mul(a, b)
#define S_INV(a) fp_inv(a)
#define S_ISZERO(a) ((a) == 0u)
#define S_LOAD(p, idx) fp_load(p, idx)
#define FN(name) fp31_##name
#include "bg_recursion.inc"
#undef SCALAR
#undef S_ZERO
#undef S_TWO
#undef S_ADD
#undef S_SUB
#undef S_MUL
#undef S_INV
#undef S_ISZERO
#undef S_LOAD
#undef FN

/* --------------------------------------------------------- complex128 ---- */
typedef double _Complex c128;
static c128 c128_inv(c128 z) { return (creal(z) == 0.0 && cimag(z) == 0.0) ? 0.0 : 1.0 / z; }
static c128 c128_load(const void* p, long idx)
{
    const double* q = (const double*)p;
    return CMPLX(q[2 * idx], q[2 * idx + 1]);
}
#define SCALAR c128
#define S_ZERO ((c128)0.0)
#define S_TWO ((c128)2.0)
#define S_ADD(a, b) ((a) + (b))
#define S_SUB(a, b) ((a) - (b))
#define S_MUL(a, b) ((a) * (b))
#define S_INV(a) c128_inv(a)
#define S_ISZERO(a) (creal(a) == 0.0 && cimag(a) == 0.0)
#define S_LOAD(p, idx) c128_load(p, idx)
#define FN(name) c128_##name
#include "bg_recursion.inc"
#undef SCALAR
#undef S_ZERO
#undef S_TWO
#undef S_ADD
#undef S_SUB
#undef S_MUL
#undef S_INV
#undef S_ISZERO
#undef S_LOAD
#undef FN

/* ------------------------------------- extended precision (truth only) ---- */
typedef long double _Complex c80;
static c80 c80_inv(c80 z) { return (creall(z) == 0.0L && cimagl(z) == 0.0L) ? 0.0L : 1.0L / z; }
static c80 c80_load(const void* p, long idx)
{
    const double* q = (const double*)p;
    return CMPLXL((long double)q[2 * idx], (long double)q[2 * idx + 1]);
}
#define SCALAR c80
#define S_ZERO ((c80)0.0L)
#define S_TWO ((c80)2.0L)
#define S_ADD(a, b) ((a) + (b))
#define S_SUB(a, b) ((a) - (b))
#define S_MUL(a, b) ((a) * (b))
#define S_INV(a) c80_inv(a)
#define S_ISZERO(a) (creall(a) == 0.0L && cimagl(a) == 0.0L)
#define S_LOAD(p, idx) c80_load(p, idx)
#define FN(name) c80_##name
#include "bg_recursion.inc"

/* ----------------------------------------------------------- exports ---- */
enum { ORACLE_FP31 = 0, ORACLE_C128 = 1, ORACLE_C80 = 2 };

static int check_args(int field, int n, int d, int64_t batch)
{
    if (field < 0 || field > 2) return -1;
    if (n < 4 || n > 16 || d < 4 || d > 16 || batch < 0) return -1;
    return 0;
}

/* All pointers are HOST pointers; caller owns every buffer.
 *   metric:   0 mostly minus, 1 alternating
 *   prime:    field 0 only: 0 = 2^31-1, else a prime 2 < prime < 2^31 (primality is the caller's job)
 *   states:   S >= 1 polarisation configurations per momentum point (the state sum of Eq.(4),
 *             PAPER.md:79-81): the literal recursion is simply run S times, nothing is shared
 *   momenta:  [batch][n][d] scalars (uint32 | double[2] | double[2]);
 *   polarisations: [batch][S][n][d]
 *   out:      [batch][S] scalars (uint32 | double[2] | long double[2])
 *   currents: NULL or [batch][S][m][m][d] scalars of the output type, m = n-1
 *             (entry (i-1,j-1) = J(i..j) for i<=j; the top one without propagator)
 *   status:   NULL or [batch] uint32, bit0 = some proper P_{i,j}^2 == 0
 * Returns 0, or -1 on bad arguments.  Single-threaded: callers that want more
 * cores call it on disjoint batch slices from several threads. */
int oracle_bg_evaluate(int field, int metric, uint32_t prime, int n, int d, int64_t batch, int states,
                       const void* momenta, const void* polarisations, void* out, void* currents,
                       uint32_t* status)
{
    if (check_args(field, n, d, batch) || (batch > 0 && (!momenta || !polarisations || !out))) return -1;
    if ((metric != 0 && metric != 1) || states < 1 || (field == ORACLE_FP31 && prime == 1)) return -1;
    if (field == ORACLE_FP31 && prime >= 0x80000000u) return -1;
    bg_p = (field == ORACLE_FP31 && prime) ? prime : BG_P31;
    bg_alternating = metric;
    const int m = n - 1;
    const long nd = (long)n * d, cur = (long)m * m * d;
    for (int64_t b = 0; b < batch; ++b) {
        unsigned st = 0;
        for (int s = 0; s < states; ++s) {
            const int64_t o = b * states + s;
            if (field == ORACLE_FP31) {
                uint32_t* J = currents ? (uint32_t*)currents + o * cur : NULL;
                ((uint32_t*)out)[o] = fp31_point(n, d, momenta, polarisations, b * nd, o * nd, J, &st);
            } else if (field == ORACLE_C128) {
                c128* J = currents ? (c128*)currents + o * cur : NULL;
                ((c128*)out)[o] = c128_point(n, d, momenta, polarisations, b * nd, o * nd, J, &st);
            } else {
                c80* J = currents ? (c80*)currents + o * cur : NULL;
                ((c80*)out)[o] = c80_point(n, d, momenta, polarisations, b * nd, o * nd, J, &st);
            }
        }
        if (status) status[b] = st;
    }
    bg_p = BG_P31;
    bg_alternating = 0;
    return 0;
}

/* mostly-minus metric, p = 2^31-1, one state configuration */
int oracle_bg_currents(int field, int n, int d, int64_t batch, const void* momenta,
                       const void* polarisations, void* out, void* currents, uint32_t* status)
{
    return oracle_bg_evaluate(field, 0, 0, n, d, batch, 1, momenta, polarisations, out, currents, status);
}

int oracle_bg_amplitudes(int field, int n, int d, int64_t batch, const void* momenta,
                         const void* polarisations, void* out, uint32_t* status)
{
    return oracle_bg_currents(field, n, d, batch, momenta, polarisations, out, NULL, status);
}

uint32_t oracle_bg_modulus(void) { return (uint32_t)BG_P31; }
