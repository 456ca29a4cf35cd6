// bg_peaks.cu -- register-resident issue-rate microbenchmarks for sm_100a.
//
// MEASURED_PEAKS.json only carries HBM and bf16-GEMM peaks; the Berends-Giele path is
// bound by the plain integer / FP64 pipes, so the roofline denominators of SURVEY.md
// §8(d) (R_mm = canonical Mersenne-31 modmuls/s, IMAD.WIDE/s, ALU ops/s, DFMA/s, and
// the shared-memory load rates the kernel design depends on) are measured on the box by
// these kernels, at whatever clock the box sustains, and timed by bench.py with CUDA
// events.  Each thread runs `iters` iterations of an unrolled body of CHAINS independent
// dependency chains x UNROLL steps; nothing touches memory until the final store.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/bg.h"

namespace {

constexpr uint32_t kP = 0x7fffffffu;
constexpr int CHAINS = 8;
constexpr int UNROLL = 8;

__device__ __forceinline__ uint32_t mad_lo(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;
    asm volatile("mad.lo.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
__device__ __forceinline__ uint32_t lop_xor_and(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;   // (a ^ b) & c : one LOP3
    asm volatile("lop3.b32 %0, %1, %2, %3, 0x60;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
__device__ __forceinline__ uint32_t add3(uint32_t a, uint32_t b)
{
    uint32_t d;
    asm volatile("add.u32 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
    return d;
}
__device__ __forceinline__ double dfma(double a, double b, double c)
{
    double d;
    asm volatile("fma.rn.f64 %0, %1, %2, %3;" : "=d"(d) : "d"(a), "d"(b), "d"(c));
    return d;
}
// canonical Mersenne-31 modular multiplication: the unit R_mm counts (SURVEY.md §8(d) iii)
__device__ __forceinline__ uint32_t modmul(uint32_t a, uint32_t b)
{
    uint64_t x = (uint64_t)a * b;
    uint32_t r = (uint32_t)(x & kP) + (uint32_t)(x >> 31);
    return min(r, r - kP);
}

template <int KIND>
__global__ void __launch_bounds__(256) peak_kernel(int iters, uint32_t seed, uint32_t* sink)
{
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    if constexpr (KIND == BG_PEAK_IMAD_WIDE) {
        // acc_c = lo(acc_{c+1}) * b + acc_c: the multiplicand comes from another chain, so the
        // product can neither be hoisted nor strength-reduced; SASS is IMAD.WIDE.U32 R, R, R, R
        // with a 64-bit addend (checked with cuobjdump; an inline-PTX mad.wide.u32 with a
        // loop-invariant product is turned into plain adds and measures nothing).
        uint64_t acc[CHAINS];
        const uint32_t b = (seed ^ 0x9e3779b9u) | 1u;
#pragma unroll
        for (int c = 0; c < CHAINS; ++c) acc[c] = ((const uint64_t*)sink)[(t * CHAINS + c) & 1023];
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int u = 0; u < UNROLL; ++u)
#pragma unroll
                for (int c = 0; c < CHAINS; ++c)
                    acc[c] = (uint64_t)(uint32_t)acc[(c + 1) % CHAINS] * b + acc[c];
        }
        uint64_t s = 0;
#pragma unroll
        for (int c = 0; c < CHAINS; ++c) s ^= acc[c];
        if (s == 0x123456789abcdefull) sink[t] = (uint32_t)s;
    } else if constexpr (KIND == BG_PEAK_IMAD_WIDE_RZ) {
        // acc = hi(acc) * lo(acc): IMAD.WIDE.U32 R, R, R, RZ -- the bare 32x32 -> 64 multiplier rate
        uint64_t acc[CHAINS];
#pragma unroll
        for (int c = 0; c < CHAINS; ++c) acc[c] = ((const uint64_t*)sink)[(t * CHAINS + c) & 1023] | 0x300000005ull;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int u = 0; u < UNROLL; ++u)
#pragma unroll
                for (int c = 0; c < CHAINS; ++c) acc[c] = (uint64_t)(uint32_t)(acc[c] >> 32) * (uint32_t)acc[c];
        }
        uint64_t s = 0;
#pragma unroll
        for (int c = 0; c < CHAINS; ++c) s ^= acc[c];
        if (s == 0x123456789abcdefull) sink[t] = (uint32_t)s;
    } else if constexpr (KIND == BG_PEAK_IMAD) {
        uint32_t acc[CHAINS];
        uint32_t a = seed + t, b = (seed ^ 0x9e3779b9u) | 1u;
#pragma unroll
        for (int c = 0; c < CHAINS; ++c) acc[c] = t + c;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int u = 0; u < UNROLL; ++u)
#pragma unroll
                for (int c = 0; c < CHAINS; ++c) acc[c] = mad_lo(a, b, acc[c]);
        }
        uint32_t s = 0;
#pragma unroll
        for (int c = 0; c < CHAINS; ++c) s ^= acc[c];
        if (s == 0x12345678u) sink[t] = s;
    } else if constexpr (KIND == BG_PEAK_ALU) {
        uint32_t acc[CHAINS];
        uint32_t a = seed + t;
#pragma unroll
        for (int c = 0; c < CHAINS; ++c) acc[c] = t + c;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int u = 0; u < UNROLL; ++u)
#pragma unroll
                for (int c = 0; c < CHAINS; ++c)
                    acc[c] = (u & 1) ? add3(acc[c], a) : lop_xor_and(acc[c], a, 0x7fffffffu);
        }
        uint32_t s = 0;
#pragma unroll
        for (int c = 0; c < CHAINS; ++c) s ^= acc[c];
        if (s == 0x12345678u) sink[t] = s;
    } else if constexpr (KIND == BG_PEAK_MIX || KIND == BG_PEAK_MIX2 || KIND == BG_PEAK_MIX3) {
        // one IMAD.WIDE (64-bit addend) + NALU ALU ops per step on independent chains: do the pipes
        // co-issue?  (Measured: no -- the cost is additive, about 3.2 + 2 NALU cycles per warp and
        // step, where independent pipes would give max(4, 2 NALU).)
        constexpr int NALU = KIND == BG_PEAK_MIX ? 1 : KIND == BG_PEAK_MIX2 ? 2 : 3;
        uint64_t acc[CHAINS / 2];
        uint32_t alu[CHAINS / 2];
        const uint32_t a = seed + t, b = (seed ^ 0x9e3779b9u) | 1u;
#pragma unroll
        for (int c = 0; c < CHAINS / 2; ++c) {
            acc[c] = ((const uint64_t*)sink)[(t * CHAINS + c) & 1023];
            alu[c] = t ^ c;
        }
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int u = 0; u < UNROLL; ++u)
#pragma unroll
                for (int c = 0; c < CHAINS / 2; ++c) {
                    acc[c] = (uint64_t)(uint32_t)acc[(c + 1) % (CHAINS / 2)] * b + acc[c];
#pragma unroll
                    for (int j = 0; j < NALU; ++j) alu[c] = lop_xor_and(alu[c], a + j, 0x7fffffffu);
                }
        }
        uint64_t s = 0;
#pragma unroll
        for (int c = 0; c < CHAINS / 2; ++c) s ^= acc[c] ^ alu[c];
        if (s == 0x123456789abcdefull) sink[t] = (uint32_t)s;
    } else if constexpr (KIND == BG_PEAK_MODMUL) {
        uint32_t x[CHAINS];
        uint32_t b = ((seed ^ 0x9e3779b9u) & kP) | 1u;
#pragma unroll
        for (int c = 0; c < CHAINS; ++c) x[c] = (t + c + 1) & kP;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int u = 0; u < UNROLL; ++u)
#pragma unroll
                for (int c = 0; c < CHAINS; ++c) x[c] = modmul(x[c], b);
        }
        uint32_t s = 0;
#pragma unroll
        for (int c = 0; c < CHAINS; ++c) s ^= x[c];
        if (s == 0xffffffffu) sink[t] = s;
    } else if constexpr (KIND == BG_PEAK_DFMA) {
        double acc[CHAINS];
        double a = 1.0 + 1e-9 * (double)(seed & 15), b = 1e-9 * (double)t;
#pragma unroll
        for (int c = 0; c < CHAINS; ++c) acc[c] = (double)c;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int u = 0; u < UNROLL; ++u)
#pragma unroll
                for (int c = 0; c < CHAINS; ++c) acc[c] = dfma(acc[c], a, b);
        }
        double s = 0;
#pragma unroll
        for (int c = 0; c < CHAINS; ++c) s += acc[c];
        if (s == 12345.678) sink[t] = 1;
    } else {   // shared-memory load rates: LDS.32 / LDS.64 / LDS.128, conflict-free
        constexpr int W = (KIND == BG_PEAK_LDS32) ? 1 : (KIND == BG_PEAK_LDS64) ? 2 : 4;
        __shared__ __align__(16) uint32_t tile[256 * 4 * 4];
        for (int i = threadIdx.x; i < 256 * 4 * 4; i += blockDim.x) tile[i] = seed + i;
        __syncthreads();
        uint32_t s = 0;
        uint32_t off = threadIdx.x * W;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int u = 0; u < UNROLL * CHAINS / 4; ++u) {
                const uint32_t idx = (off + u * 256 * W) & (256 * 4 * 4 - 1);
                const uint32_t addr = (uint32_t)__cvta_generic_to_shared(&tile[idx]);
                if constexpr (W == 1) {
                    uint32_t v;
                    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
                    s ^= v;
                } else if constexpr (W == 2) {
                    uint2 v;
                    asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
                    s ^= v.x ^ v.y;
                } else {
                    uint4 v;
                    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];"
                                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                                 : "r"(addr));
                    s ^= v.x ^ v.y ^ v.z ^ v.w;
                }
            }
            off = (off + s) & 0;   // keeps a (trivially zero) dependence on the loaded data
            off += threadIdx.x * W;
        }
        if (s == 0x12345678u) sink[t] = s;
    }
}

template <int KIND>
int launch(int iters, int blocks, int threads, uint32_t* sink, cudaStream_t stream)
{
    peak_kernel<KIND><<<blocks, threads, 0, stream>>>(iters, 12345u, sink);
    return cudaGetLastError() == cudaSuccess ? BG_OK : BG_ERR_CUDA;
}

}  // namespace

extern "C" int bg_peak_probe(int kind, int iters, int blocks, int threads, uint32_t* sink,
                             int64_t* ops_per_thread, cudaStream_t stream)
{
    if (iters < 0 || blocks <= 0 || threads <= 0 || threads > 256 || !sink) return BG_ERR_ARG;
    int64_t per_iter = (int64_t)CHAINS * UNROLL;
    int rc;
    switch (kind) {
        case BG_PEAK_IMAD_WIDE: rc = launch<BG_PEAK_IMAD_WIDE>(iters, blocks, threads, sink, stream); break;
        case BG_PEAK_IMAD_WIDE_RZ: rc = launch<BG_PEAK_IMAD_WIDE_RZ>(iters, blocks, threads, sink, stream); break;
        case BG_PEAK_IMAD: rc = launch<BG_PEAK_IMAD>(iters, blocks, threads, sink, stream); break;
        case BG_PEAK_ALU: rc = launch<BG_PEAK_ALU>(iters, blocks, threads, sink, stream); break;
        case BG_PEAK_MIX: rc = launch<BG_PEAK_MIX>(iters, blocks, threads, sink, stream); break;
        case BG_PEAK_MIX2: rc = launch<BG_PEAK_MIX2>(iters, blocks, threads, sink, stream); per_iter = per_iter * 3 / 2; break;
        case BG_PEAK_MIX3: rc = launch<BG_PEAK_MIX3>(iters, blocks, threads, sink, stream); per_iter *= 2; break;
        case BG_PEAK_MODMUL: rc = launch<BG_PEAK_MODMUL>(iters, blocks, threads, sink, stream); break;
        case BG_PEAK_DFMA: rc = launch<BG_PEAK_DFMA>(iters, blocks, threads, sink, stream); break;
        case BG_PEAK_LDS32: rc = launch<BG_PEAK_LDS32>(iters, blocks, threads, sink, stream); per_iter /= 4; break;
        case BG_PEAK_LDS64: rc = launch<BG_PEAK_LDS64>(iters, blocks, threads, sink, stream); per_iter /= 4; break;
        case BG_PEAK_LDS128: rc = launch<BG_PEAK_LDS128>(iters, blocks, threads, sink, stream); per_iter /= 4; break;
        default: return BG_ERR_ARG;
    }
    if (ops_per_thread) *ops_per_thread = per_iter * iters;
    return rc;
}
