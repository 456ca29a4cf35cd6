// bg_state_sum.cu -- the left-hand side of the cut equation Eq.(4), PAPER.md:79-81:
//     out[b] = sum_{s < S} prod_{t < T} amps_t[b][s]
// "sum over states" of the product of the tree amplitudes of a cut, for arrays of amplitudes
// produced by bg_amplitudes_states / bg_evaluate ([batch][S] each).  Bound by HBM traffic (T S + 1 scalars
// per point), not by arithmetic: the arrays are read as ONE coalesced stream (16 bytes per thread and tree), the
// products are formed element-wise and the S elements of a point are summed inside the thread and then across the
// S / VEC neighbouring lanes with shuffles.  (One thread per point -- the first version, still the fallback for an S
// that is not VEC times a power of two -- reads with a stride of S elements between lanes: 0.25 of the HBM peak.)
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/bg.h"
#include "bg_field.cuh"

namespace {

using bg::C128;
using bg::Fp31;
using bg::FpMont;

template <class F>
struct SumParams {
    const typename F::E* amps[BG_MAX_TREES];
    typename F::E* out;
    long long batch;
    int states, trees;
    typename F::Params fld;
};

template <class F>
__global__ void __launch_bounds__(256) state_sum_kernel(const SumParams<F> prm)
{
    typedef typename F::E E;
    const F f(prm.fld, 0);
    const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= prm.batch) return;
    E total = f.ezero();
    for (int s = 0; s < prm.states; ++s) {
        E prod = f.load_input(__ldg(prm.amps[0] + b * prm.states + s));
        for (int t = 1; t < prm.trees; ++t) prod = f.mul(prod, f.load_input(__ldg(prm.amps[t] + b * prm.states + s)));
        total = f.add(total, prod);
    }
    prm.out[b] = f.to_output(total);
}

template <class F> struct SumVec { static constexpr int value = 4; typedef uint4 type; };      // 4-byte residues
template <> struct SumVec<C128> { static constexpr int value = 1; typedef double2 type; };

template <class F>
__device__ __forceinline__ void sum_unpack(const uint4& v, typename F::E (&x)[4]) { x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w; }
template <class F>
__device__ __forceinline__ void sum_unpack(const double2& v, typename F::E (&x)[1]) { x[0] = v; }

__device__ __forceinline__ uint32_t sum_shfl(uint32_t x, int off) { return __shfl_xor_sync(0xffffffffu, x, off); }
__device__ __forceinline__ double2 sum_shfl(double2 x, int off)
{
    return make_double2(__shfl_xor_sync(0xffffffffu, x.x, off), __shfl_xor_sync(0xffffffffu, x.y, off));
}

// states = VEC * lanes_per_point, lanes_per_point a power of two <= 32; thread i owns the elements [VEC i, VEC (i + 1))
// of the flattened [batch][S] arrays
constexpr int kSumUnroll = 4;           // vectors per thread, all loads of a tree in flight together

template <class F, int VEC>
__global__ void __launch_bounds__(256) state_sum_stream_kernel(const SumParams<F> prm, int lanes_per_point)
{
    typedef typename F::E E;
    typedef typename SumVec<F>::type V;
    const F f(prm.fld, 0);
    const long long nvec = prm.batch * prm.states / VEC;
    const long long i0 = (long long)blockIdx.x * (256 * kSumUnroll) + threadIdx.x;
    V raw[kSumUnroll];
    E prod[kSumUnroll][VEC];
#pragma unroll
    for (int k = 0; k < kSumUnroll; ++k)
        if (i0 + 256 * k < nvec) raw[k] = __ldg(reinterpret_cast<const V*>(prm.amps[0]) + i0 + 256 * k);
#pragma unroll
    for (int k = 0; k < kSumUnroll; ++k) {
        sum_unpack<F>(raw[k], prod[k]);
#pragma unroll
        for (int j = 0; j < VEC; ++j) prod[k][j] = f.load_input(prod[k][j]);
    }
    for (int t = 1; t < prm.trees; ++t) {
#pragma unroll
        for (int k = 0; k < kSumUnroll; ++k)
            if (i0 + 256 * k < nvec) raw[k] = __ldg(reinterpret_cast<const V*>(prm.amps[t]) + i0 + 256 * k);
#pragma unroll
        for (int k = 0; k < kSumUnroll; ++k) {
            E x[VEC];
            sum_unpack<F>(raw[k], x);
#pragma unroll
            for (int j = 0; j < VEC; ++j) prod[k][j] = f.mul(prod[k][j], f.load_input(x[j]));
        }
    }
#pragma unroll
    for (int k = 0; k < kSumUnroll; ++k) {
        const long long i = i0 + 256 * k;
        E part = f.ezero();
#pragma unroll
        for (int j = 0; j < VEC; ++j) part = f.add(part, prod[k][j]);
        for (int off = lanes_per_point >> 1; off >= 1; off >>= 1) part = f.add(part, sum_shfl(part, off));
        if (i < nvec && (threadIdx.x & (lanes_per_point - 1)) == 0) prm.out[i / lanes_per_point] = f.to_output(part);
    }
}

template <class F>
int launch(const typename F::Params& fld, int64_t batch, int states, int trees, const void* const* amps, void* out,
           cudaStream_t stream)
{
    SumParams<F> prm;
    for (int t = 0; t < BG_MAX_TREES; ++t)
        prm.amps[t] = t < trees ? static_cast<const typename F::E*>(amps[t]) : nullptr;
    prm.out = static_cast<typename F::E*>(out);
    prm.batch = batch;
    prm.states = states;
    prm.trees = trees;
    prm.fld = fld;
    constexpr int VEC = SumVec<F>::value;
    const int lpp = states % VEC == 0 ? states / VEC : 0;
    bool aligned = true;
    for (int t = 0; t < trees; ++t) aligned = aligned && (reinterpret_cast<uintptr_t>(amps[t]) & 15u) == 0;
    if (aligned && lpp >= 1 && lpp <= 32 && (lpp & (lpp - 1)) == 0) {
        const int64_t nvec = batch * lpp, blocks = (nvec + 256 * kSumUnroll - 1) / (256 * kSumUnroll);
        if (blocks > 0x7fffffffLL) return BG_ERR_ARG;
        state_sum_stream_kernel<F, VEC><<<(unsigned)blocks, 256, 0, stream>>>(prm, lpp);
        return cudaGetLastError() == cudaSuccess ? BG_OK : BG_ERR_CUDA;
    }
    const int64_t blocks = (batch + 255) / 256;
    if (blocks > 0x7fffffffLL) return BG_ERR_ARG;
    state_sum_kernel<F><<<(unsigned)blocks, 256, 0, stream>>>(prm);
    if (cudaGetLastError() != cudaSuccess) return BG_ERR_CUDA;
    return BG_OK;
}

}  // namespace

#include "bg_host_util.h"

extern "C" int bg_state_sum(int field, uint32_t prime, int64_t batch, int states, int trees,
                            const void* const* amps, void* out, cudaStream_t stream)
{
    if (batch < 0 || states < 1 || trees < 1 || trees > BG_MAX_TREES || !amps) return BG_ERR_ARG;
    if (batch == 0) return BG_OK;
    if (!out) return BG_ERR_ARG;
    for (int t = 0; t < trees; ++t)
        if (!amps[t] || amps[t] == out) return BG_ERR_ARG;
    switch (field) {
        case BG_FIELD_FP31: return launch<Fp31>(Fp31::Params{}, batch, states, trees, amps, out, stream);
        case BG_FIELD_C128: return launch<C128>(C128::Params{}, batch, states, trees, amps, out, stream);
        case BG_FIELD_FPMONT: {
            FpMont::Params q{};
            if (!bg_mont_constants(prime, 0, &q)) return BG_ERR_ARG;
            return launch<FpMont>(q, batch, states, trees, amps, out, stream);
        }
    }
    return BG_ERR_ARG;
}
