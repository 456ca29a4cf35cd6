// bg_state_sum.cu -- the left-hand side of the cut equation Eq.(4), PAPER.md:79-81:
//     out[b] = sum_{s < S} prod_{t < T} amps_t[b][s]
// "sum over states" of the product of the tree amplitudes of a cut, for arrays of amplitudes
// produced by bg_amplitudes_states / bg_evaluate ([batch][S] each).  One thread per momentum
// point; the kernel is bound by HBM traffic (T S + 1 scalars per point), not by arithmetic.
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
