/* bg.h -- C ABI of libbg_b200: batched colour-ordered n-gluon tree amplitudes by
 * Berends-Giele recursion in d space-time dimensions, over F_p (p = 2^31-1) and
 * complex128, on one NVIDIA B200 (sm_100a).
 *
 * Reference: arXiv:2502.07060 ("Accelerating Berends-Giele recursion for gluons in
 * arbitrary dimensions over finite fields"); citations are PAPER.md:<line>.
 *
 * What one call computes, per phase-space point b (points are independent; the paper
 * parallelises "strictly along the event dimension"):
 *
 *     P_{i,j} = sum_{l=i..j} k_l                                   Eq.(7)
 *     J(i..i) = eps_i
 *     J(i..j) = 1/P_{i,j}^2 [ sum_k V3(P_{i,k},P_{k+1,j}) J(i..k) J(k+1..j)
 *                           + sum_{k<l} V4 J(i..k) J(k+1..l) J(l+1..j) ]   Eq.(6)
 *     out[b]  = eps_n . N(1..n-1)     N = the bracket above for the (n-1)-gluon current,
 *                                     no propagator on it
 *
 * with V3, V4 of Eq.(7), metric g = diag(+,-,...,-) and
 * the factors of i cancelled: (-i) of Eq.(6) times i of Eq.(7) = 1, so everything stays in
 * F_p; the physical colour-ordered amplitude is i * out (readings R1-R5).
 * The momenta and polarisation states are prepared by the caller on the host, exactly as
 * in the paper.  Every step above runs inside hand-written sm_100a kernels;
 * there is no CPU fallback and no other backend.
 *
 * Conventions common to all entry points
 *   scalars   BG_FIELD_FP31: uint32_t residues mod p = 2^31-1; values >= p are reduced mod p on load;
 *             results are canonical, in [0,p).
 *             BG_FIELD_C128: double[2] = (re, im), interleaved.
 *             BG_FIELD_FPMONT: uint32_t residues mod a prime 2^30 < p < 2^31 given per call
 *             (plain residues at the boundary; Montgomery form is internal to the kernels).
 *   metric    BG_METRIC_MOSTLY_MINUS g = diag(+,-,..,-) unless an entry point takes a
 *             metric argument; BG_METRIC_ALTERNATING g = diag(+,-,+,-,..) is the switch the paper
 *             added to match Caravel.
 *   layout    momenta, polarisations: [batch][n][d] scalars, point-major, contravariant
 *             components, all momenta outgoing (sum_l k_l = 0 is the caller's job; the
 *             library evaluates the map above for whatever it is given, reading R4).
 *             out: [batch] scalars.
 *   limits    4 <= n <= 16, 4 <= d <= 16 (the paper validates d = 4..10).
 *   memory    the caller owns every buffer; DEVICE pointers unless the name says host.
 *             Device pointers must be 16-byte aligned; out must not alias the inputs.
 *             The library allocates no device memory and keeps no per-call state; on the host a call
 *             allocates nothing either (a shape's launch plan is built on its first use and cached; shapes
 *             without a compiled instance stage their 29 KB schedule in a per-thread block).
 *   stream    launches are asynchronous on `stream`; nothing synchronises.
 *   errors    return value: BG_OK or a negative bg_status_t; nothing is thrown, nothing
 *             aborts.  Arguments are checked on the host before any launch.  batch == 0 is
 *             a no-op returning BG_OK.
 *   tuning    bg_set_kernel_override() restricts the kernel selection for A/B measurements (it never
 *             changes results); the environment variables BG_KERNEL = unit1 | unit2 | reg | rt | general and
 *             BG_KERNEL_W = <warps per tile> give its initial value, read ONCE when the library is loaded.
 *             Without either (the normal case) the default instance of the shape is launched.
 *   1/0       inv(0) := 0 in both fields (what Fermat's a^(p-2) gives); a point where some
 *             proper P_{i,j}^2 vanishes gets status bit0 set (reading R6).
 */
#ifndef BG_B200_H
#define BG_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* cudaStream_t without dragging cuda_runtime.h into C callers */
#ifndef __DRIVER_TYPES_H__
typedef struct CUstream_st* cudaStream_t;
#endif

typedef enum { BG_FIELD_FP31 = 0, BG_FIELD_C128 = 1, BG_FIELD_FPMONT = 2 } bg_field_t;
typedef enum { BG_METRIC_MOSTLY_MINUS = 0, BG_METRIC_ALTERNATING = 1 } bg_metric_t;
#define BG_MAX_PRIMES 8
#define BG_MAX_TREES 8

typedef enum {
    BG_OK = 0,
    BG_ERR_ARG = -1,          /* bad n, d, batch, field, metric, prime, null or misaligned pointer */
    BG_ERR_UNSUPPORTED = -2,  /* (field, n, d) needs more shared memory per point than an SM has */
    BG_ERR_CUDA = -3,         /* a CUDA runtime call or launch failed */
    BG_ERR_TOO_LARGE = -4     /* bg_amplitudes_host_noalloc: batch > bg_noalloc_max_batch(field, n, d) */
} bg_status_t;

/* ---- the hot path (SURVEY.md §8(a) rows a0-a6 in ONE kernel launch) ------------------- */

/* Amplitudes for `batch` points.  Device pointers.  Eq.(6)/(7). */
int bg_amplitudes(int field, int n, int d, int64_t batch,
                  const void* momenta, const void* polarisations, void* out,
                  cudaStream_t stream);

/* Same, plus a per-point status word: status[b] bit0 = some proper P_{i,j}^2 == 0
 * (its propagator was taken as 0).  status: device, [batch] uint32, or NULL. */
int bg_amplitudes_status(int field, int n, int d, int64_t batch,
                         const void* momenta, const void* polarisations, void* out,
                         uint32_t* status, cudaStream_t stream);

/* Same map, but also returns every off-shell current (Eq.(6) by-products):
 * currents: device, [batch][m][m][d] scalars, m = n-1; entry (i-1, j-1), i <= j, holds
 * J(i..j) (the top one, J(1..m), WITHOUT propagator); entries with i > j are not written.
 * currents may be NULL. */
int bg_currents(int field, int n, int d, int64_t batch,
                const void* momenta, const void* polarisations, void* out,
                void* currents, uint32_t* status, cudaStream_t stream);

/* ---- the same path, generalised --------------------------------- */

/* What to evaluate.  states = S >= 1 polarisation configurations per momentum point: the partial
 * momenta, invariants and propagators (rows a1-a3) depend on the momenta only and are formed once
 * per point, the level sweep runs per configuration -- the workload of the cut equation Eq.(4),
 * PAPER.md:79-81, whose state sum "runs over all D_s-dimensional particle states".
 * BG_FIELD_FPMONT: n_primes = 1..BG_MAX_PRIMES primes, each odd and 2^30 < p < 2^31 (primality is the
 * caller's job: the inverse is a^(p-2)); every array then has a leading [n_primes] axis and prime q
 * works on slice q (ONE launch, grid.y = n_primes).  Other fields: n_primes = 0. */
typedef struct {
    int field;               /* bg_field_t */
    int metric;              /* bg_metric_t */
    int n, d;
    int states;              /* S */
    int n_primes;
    uint32_t primes[BG_MAX_PRIMES];
    int n_orderings;         /* K colour orderings per point (Eq.(5)); 0 or 1: the caller's order.
                                K <= 2^24 and max(K,1) * S < 2^27 (BG_ERR_ARG otherwise) */
    const unsigned char* orderings;   /* NULL, or DEVICE [K][n]: row o lists, for positions 1..n, which of the
                                caller's legs (0-based) stands there; every row must be a permutation of
                                0..n-1 (not checked: entries >= n are clamped to n-1) */
} bg_problem_t;

/* momenta [P][batch][n][d], polarisations [P][batch][S][n][d], out [P][batch][K][S], status NULL or
 * [P][batch] (P = max(1, n_primes), K = max(1, n_orderings)); currents NULL, or [batch][m][m][d] when
 * S == 1, P == 1 and K == 1.  Device pointers, asynchronous on `stream`. */
int bg_evaluate(const bg_problem_t* problem, int64_t batch, const void* momenta, const void* polarisations,
                void* out, void* currents, uint32_t* status, cudaStream_t stream);

/* S state configurations per momentum point, mostly-minus metric (Eq.(4)):
 * polarisations [batch][S][n][d], out [batch][S]. */
int bg_amplitudes_states(int field, int n, int d, int64_t batch, int states, const void* momenta,
                         const void* polarisations, void* out, uint32_t* status, cudaStream_t stream);

/* K colour orderings of every point in one launch: the colour-ordered amplitudes C(sigma_o(1), .., sigma_o(n))
 * that the colour decomposition Eq.(5), sums over the permutations P(1..n-1) with the
 * traces Tr(T^a_sigma(1) .. T^a_n).  The inputs of a point are read from HBM once; every ordering re-stages
 * them in its order (rows a1-a6 per ordering).  orderings: DEVICE [K][n] as in bg_problem_t; out [batch][K];
 * status bit0 = some proper P^2 vanished in SOME ordering.  Mostly-minus metric. */
int bg_amplitudes_orderings(int field, int n, int d, int64_t batch, int n_orderings, const unsigned char* orderings,
                            const void* momenta, const void* polarisations, void* out, uint32_t* status,
                            cudaStream_t stream);

/* Several generic 31-bit primes in one launch (Q-reconstruction from the F_p values);
 * momenta, polarisations [n_primes][batch][n][d] residues mod primes[q], out [n_primes][batch]. */
int bg_amplitudes_primes(int metric, int n, int d, int64_t batch, int n_primes, const uint32_t* primes,
                         const void* momenta, const void* polarisations, void* out, uint32_t* status,
                         cudaStream_t stream);

/* The left-hand side of the cut equation Eq.(4), PAPER.md:79-81 -- "sum over states" of the product of
 * the tree amplitudes of a cut:  out[b] = sum_{s<S} prod_{t<trees} amps[t][b][s].
 * amps: HOST array of `trees` (1..BG_MAX_TREES) DEVICE pointers, each [batch][S] scalars as written by
 * bg_amplitudes_states / bg_evaluate; out: device [batch], must not alias an input.  prime: the
 * modulus for BG_FIELD_FPMONT (plain residues in and out), ignored otherwise. */
int bg_state_sum(int field, uint32_t prime, int64_t batch, int states, int trees,
                 const void* const* amps, void* out, cudaStream_t stream);

/* ---- the stage in front of the path, on the device ---------------------------- */

/* The D-2 square-root-free polarisation states eps_x and their duals eps~_x (Eqs.(8)-(18))
 * of `count` massless d-vectors: momenta [count][d], chi [count][4] (the massless 4-dimensional reference
 * vector of Eq.(8)), eps and eps_tilde [count][d-2][d] (row x-1 = eps_x; eps~_1 = eps_2, eps~_2 = eps_1),
 * status NULL or [count] (bit0: a denominator of Eqs.(10),(16)-(18) vanished, the states are undefined).
 * 4 <= d <= 16.  prime: BG_FIELD_FPMONT only.  The mostly-minus spinors contain sqrt(-1): over F_p they
 * exist only for p = 1 mod 4 (BG_ERR_UNSUPPORTED otherwise, in particular for BG_FIELD_FP31; also for a
 * composite p with no quadratic non-residue below 256 -- primality stays the caller's job, the search is bounded); with
 * BG_METRIC_ALTERNATING they are rational.  Readings R13-R15 of DESIGN.md. */
int bg_states(int field, uint32_t prime, int metric, int d, int64_t count, const void* momenta, const void* chi,
              void* eps, void* eps_tilde, uint32_t* status, cudaStream_t stream);

/* The seeded synthetic phase-space generator of DESIGN.md §4 (the recipe of BASELINE.json:configs; the
 * paper draws its points on the host with lips) for points [start, start + batch) of the
 * workload `seed`: momenta, polarisations (and references, NULL or the massless reference vectors r_i)
 * [batch][n][d].  helicities: NULL for the generic transverse polarisations, else n signs (d = 4) for the
 * spinor-helicity states on (k_i, r_i); redraws: NULL or one device counter, incremented by the number
 * of rejected attempts (F_p).  Over F_p the result is bit-identical to the host generator
 * (paper_2502_07060_b200/inputs.py), over complex128 it agrees to rounding. */
int bg_generate(int field, uint32_t prime, int metric, int n, int d, int64_t batch, uint64_t seed, int64_t start,
                const signed char* helicities, void* momenta, void* polarisations, void* references,
                unsigned long long* redraws, cudaStream_t stream);

/* End-to-end variant with HOST buffers (pinned memory recommended): copies the inputs to
 * the device in chunks, runs the kernel and copies the results back, overlapping the three
 * on internal streams; returns after everything has completed.  `workspace` is DEVICE
 * scratch owned by the caller, `workspace_bytes` >= bg_host_workspace_bytes(...) for at
 * least one chunk of 1024 points; more workspace = larger chunks. */
int bg_amplitudes_host(int field, int n, int d, int64_t batch,
                       const void* host_momenta, const void* host_polarisations,
                       void* host_out, uint32_t* host_status,
                       void* workspace, size_t workspace_bytes);
size_t bg_host_workspace_bytes(int field, int n, int d, int64_t chunk_points);

/* The same call for a caller that CANNOT ALLOCATE device memory -- a plug-in beside a framework whose
 * caching allocator already holds nearly all of HBM (its own cudaMalloc fails), a caller that must not pay
 * cudaMalloc / cudaFree's device-wide synchronisation, or a plain C / Fortran program that owns host arrays
 * only.  Such a caller has no `workspace` to pass to bg_amplitudes_host.  Here the device staging area is a
 * fixed array of BG_NOALLOC_SCRATCH_BYTES inside the library image (a file-scope __device__ array): the CUDA
 * runtime reserves it on every GPU that loads libbg_b200.so and keeps it until the process exits, whether
 * or not this entry point is ever called.  The call allocates nothing (no cudaMalloc / cudaFree /
 * cudaMallocAsync, no stream or event creation): H2D copies, ONE launch of the kernel bg_amplitudes_status
 * would launch, D2H copies, all on `stream`, then it waits for `stream` and returns.
 *   arguments  as bg_amplitudes_host: HOST arrays momenta, polarisations [batch][n][d], out [batch],
 *              status NULL or [batch]; field BG_FIELD_FP31 or BG_FIELD_C128; mostly-minus metric.
 *              Pageable host memory works, pinned memory is faster.
 *   limit      one call takes at most bg_noalloc_max_batch(field, n, d) points (21 398 for n = 8, d = 6 over
 *              F_p); a larger batch returns BG_ERR_TOO_LARGE before anything is copied or launched -- call
 *              again with the next slice.  Nothing is chunked internally.
 *   first call the first call on each device (with that device current) looks up the device address of the
 *              array (cudaGetSymbolAddress); make that call before any stream capture begins.
 *   sharing    every call on a device uses the same array.  Calls whose GPU work can overlap (two host threads,
 *              two streams) race on it and return garbage: serialise them.  The array keeps the previous
 *              call's bytes; a call reads back only what it has written itself, so nothing is cleared. */
#define BG_NOALLOC_SCRATCH_BYTES (8u << 20)
int bg_amplitudes_host_noalloc(int field, int n, int d, int64_t batch,
                               const void* host_momenta, const void* host_polarisations,
                               void* host_out, uint32_t* host_status, cudaStream_t stream);
int64_t bg_noalloc_max_batch(int field, int n, int d);   /* 0 for an invalid (field, n, d) */
size_t bg_noalloc_scratch_bytes(void);                   /* BG_NOALLOC_SCRATCH_BYTES of the loaded library */

/* ---- introspection --------------------------------------------------------------------- */

uint32_t bg_modulus(void);             /* 2147483647 */
const char* bg_status_string(int status);
const char* bg_version(void);

/* Algorithmic operation counts per amplitude for the literal Eq.(6) evaluation (M_ref of
 * SURVEY.md §8(d)), by formula; and the counts the shipped kernel executes. */
typedef struct {
    int64_t currents;        /* n(n-1)/2 */
    int64_t propagators;     /* R = (n-1)(n-2)/2 - 1 */
    int64_t splits3;         /* C(n,3) */
    int64_t splits4;         /* C(n,4) */
    int64_t mul_v3;          /* 6 d C(n,3) */
    int64_t mul_v4;          /* 6 d C(n,4) */
    int64_t mul_other;       /* d R + 3(R-1) + d R + d */
    int64_t mul_ref;         /* M_ref = the three above */
    int64_t mul_factored;    /* field multiplications the kernels' factored form executes (bg_common.cuh):
                                6d per 3-split, 2d per 4-split, per current d (boundary term) + d (propagator)
                                + d (2P.J) + 1, per single gluon d, d R invariants, 3(R-1) + ~45 batch inverse */
    int64_t bytes_in;        /* 2 n d w */
    int64_t bytes_out;       /* w */
} bg_opcount_t;
int bg_op_count(int field, int n, int d, bg_opcount_t* out);

/* Launch configuration the library would use for (field, n, d). */
typedef struct {
    int specialised;         /* (n, d) compiled in: 1 bg_unit_kernel with one lane per point, 2 bg_unit_kernel with
                                two lanes per point, 3 bg_reg_kernel (currents in registers); any other shape:
                                4 bg_rt_kernel (the tiled kernel with a run-time n and a host-built schedule; one
                                state configuration, one ordering), 0 bg_general_kernel (one thread per point:
                                several state configurations / orderings on an uncompiled shape, and records too
                                large for a 16-point tile) -- the one a call would launch */
    int threads_per_block;
    int points_per_block;
    int smem_bytes_per_block;
    int smem_bytes_per_point;
    int blocks_per_sm;       /* limited by shared memory */
    int regs_per_thread;
} bg_kernel_info_t;
int bg_kernel_info(int field, int n, int d, bg_kernel_info_t* out);             /* mostly-minus metric, S = 1 */
int bg_kernel_info_problem(const bg_problem_t* problem, bg_kernel_info_t* out);

/* Restrict the kernel selection of all later calls (process-wide; for A/B measurements, not meant to
 * be changed while other threads are inside the library).  kind: -1 default, 1 / 2 / 3 / 4 as in
 * bg_kernel_info_t.specialised (4 also on compiled shapes), 0 the general kernel; warps: warps per tile, 0 = the first instance
 * of that kind.  A shape with no matching instance falls back to its default.  Returns BG_OK. */
int bg_set_kernel_override(int kind, int warps);

/* Host-side self-check of the compile-time work schedules of the tiled kernels (every splitting
 * of Eq.(6), executed exactly once; a current shared between warps finished by the owner
 * of its first units as that warp's last task, every other part parked once in a scratch slot of its
 * own as its warp's first task and added exactly once), and of the schedules the host builds at run time
 * for shapes without a compiled instance (equal to the compiled ones on compiled shapes).  Needs no GPU.
 * Returns 0, or a negative code naming the first violated rule. */
int bg_selftest_schedules(void);

/* ---- measurement support ---------------------------------------------------------------- */

/* Register-resident issue-rate microbenchmarks (csrc/bg_peaks.cu): launches one kernel of
 * `blocks` x `threads` threads, each executing *ops_per_thread operations of the given
 * kind.  The caller times the launch with CUDA events.  sink: device scratch of at least
 * blocks*threads uint32 (never actually written). */
typedef enum {
    BG_PEAK_IMAD_WIDE = 0,   /* IMAD.WIDE.U32 (32x32+64 -> 64) */
    BG_PEAK_IMAD = 1,        /* IMAD (32x32+32 -> 32) */
    BG_PEAK_ALU = 2,         /* LOP3 / IADD3 */
    BG_PEAK_MIX = 3,         /* IMAD.WIDE and ALU alternating (counts both) */
    BG_PEAK_MODMUL = 4,      /* canonical Mersenne-31 modular multiplication: R_mm */
    BG_PEAK_DFMA = 5,        /* FP64 fused multiply-add: R_dfma */
    BG_PEAK_LDS32 = 6,       /* shared-memory loads, 4/8/16 bytes per lane */
    BG_PEAK_LDS64 = 7,
    BG_PEAK_LDS128 = 8,
    BG_PEAK_MIX2 = 9,        /* one IMAD.WIDE + two ALU ops per step (counts all three) */
    BG_PEAK_MIX3 = 10,       /* one IMAD.WIDE + three ALU ops per step (counts all four) */
    BG_PEAK_IMAD_WIDE_RZ = 11 /* IMAD.WIDE.U32 without addend (32x32 -> 64): the bare multiplier rate */
} bg_peak_kind_t;
int bg_peak_probe(int kind, int iters, int blocks, int threads, uint32_t* sink,
                  int64_t* ops_per_thread, cudaStream_t stream);

#ifdef __cplusplus
}
#endif
#endif /* BG_B200_H */
