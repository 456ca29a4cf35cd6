// bg_states.cu -- bg_states(): the D-2 sqrt-free polarisation states of PAPER.md §2.3 for a batch of
// massless vectors, one thread per vector (device code: bg_states.cuh).
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/bg.h"
#include "bg_states.cuh"
#include "bg_host_util.h"

namespace {

using bg::C128;
using bg::Fp31;
using bg::FpMont;

template <class F>
struct StatesParams {
    const typename F::E* mom;     // [count][d]
    const typename F::E* chi;     // [count][4]
    typename F::E* eps;           // [count][d-2][d]
    typename F::E* til;           // [count][d-2][d]
    uint32_t* status;             // NULL or [count]
    long long count;
    int d, metric;
    bg::SpinorConsts<F> sc;
    typename F::Params fld;
};

// STAGED: the 2 (d-2) d outputs of a thread go to a shared-memory row first and the block copies them out as one
// contiguous, coalesced stream.  (Storing them element by element -- the fallback when a row does not fit -- puts
// the lanes of a warp 4 (d-2) d bytes apart: 48 scattered stores per thread at d = 6, `lg_throttle` + `mio_throttle`
// 58 % of the stall samples, 0.15 of the HBM peak.)
template <class F, bool STAGED>
__global__ void __launch_bounds__(128) states_kernel(const StatesParams<F> prm)
{
    typedef typename F::E E;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const F f(prm.fld, 0);
    const long long b0 = (long long)blockIdx.x * blockDim.x, b = b0 + threadIdx.x;
    const bool live = b < prm.count;
    const int d = prm.d, per = (d - 2) * d;                    // elements per vector and output array
    const int stride = 2 * per + 1;                            // odd: conflict-free rows
    E* row = reinterpret_cast<E*>(smem_raw) + (size_t)threadIdx.x * stride;
    if (live) {
        E k[bg::kMaxD], chi[4];
        for (int mu = 0; mu < d; ++mu) k[mu] = f.load_input(prm.mom[b * d + mu]);
        for (int mu = 0; mu < 4; ++mu) chi[mu] = f.load_input(prm.chi[b * 4 + mu]);
        E* eo = prm.eps + b * (long long)per;
        E* to = prm.til + b * (long long)per;
        const bool ok = bg::build_states<F>(
            f, prm.sc, prm.metric, d, k, chi,
            [&](int r, int mu, E v) {
                if (STAGED) row[r * d + mu] = f.to_output(v);
                else eo[r * d + mu] = f.to_output(v);
            },
            [&](int r, int mu, E v) {
                if (STAGED) row[per + r * d + mu] = f.to_output(v);
                else to[r * d + mu] = f.to_output(v);
            });
        if (prm.status) prm.status[b] = ok ? 0u : 1u;
    }
    if constexpr (STAGED) {
        __syncthreads();
        const int nlive = (int)min((long long)blockDim.x, prm.count - b0);
        const E* tile = reinterpret_cast<const E*>(smem_raw);
        E* ge = prm.eps + b0 * (long long)per;
        E* gt = prm.til + b0 * (long long)per;
        const int total = nlive * per;
        for (int i = threadIdx.x; i < total; i += blockDim.x) {
            const int t = i / per, w = i - t * per;
            ge[i] = tile[(size_t)t * stride + w];
            gt[i] = tile[(size_t)t * stride + per + w];
        }
    }
}

template <class F>
int launch(const typename F::Params& fld, const bg::SpinorConsts<F>& sc, int metric, int d, int64_t count,
           const void* mom, const void* chi, void* eps, void* til, uint32_t* status, cudaStream_t stream)
{
    StatesParams<F> prm;
    prm.mom = static_cast<const typename F::E*>(mom);
    prm.chi = static_cast<const typename F::E*>(chi);
    prm.eps = static_cast<typename F::E*>(eps);
    prm.til = static_cast<typename F::E*>(til);
    prm.status = status;
    prm.count = count;
    prm.d = d;
    prm.metric = metric;
    prm.sc = sc;
    prm.fld = fld;
    // staged through shared memory with as many threads per block (<= 128) as rows fit in 96 KB (two blocks per SM)
    const size_t row_bytes = (size_t)(2 * (d - 2) * d + 1) * sizeof(typename F::E);
    int threads = (int)((96 * 1024) / row_bytes) / 32 * 32;
    if (threads > 128) threads = 128;
    if (threads >= 32) {
        const size_t smem = row_bytes * threads;
        static bool attr_done[64] = {};
        int dev = 0;
        if (cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < 64 && !attr_done[dev]) {
            if (cudaFuncSetAttribute(states_kernel<F, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024) != cudaSuccess) {
                cudaGetLastError();
                return BG_ERR_CUDA;
            }
            attr_done[dev] = true;
        }
        const int64_t blocks = (count + threads - 1) / threads;
        if (blocks > 0x7fffffffLL) return BG_ERR_ARG;
        states_kernel<F, true><<<(unsigned)blocks, threads, smem, stream>>>(prm);
        return cudaGetLastError() == cudaSuccess ? BG_OK : BG_ERR_CUDA;
    }
    const int64_t blocks = (count + 127) / 128;
    if (blocks > 0x7fffffffLL) return BG_ERR_ARG;
    states_kernel<F, false><<<(unsigned)blocks, 128, 0, stream>>>(prm);
    return cudaGetLastError() == cudaSuccess ? BG_OK : BG_ERR_CUDA;
}

}  // namespace

extern "C" int bg_states(int field, uint32_t prime, int metric, int d, int64_t count, const void* momenta,
                         const void* chi, void* eps, void* eps_tilde, uint32_t* status, cudaStream_t stream)
{
    if (d < 4 || d > 16 || count < 0) return BG_ERR_ARG;
    if (metric != BG_METRIC_MOSTLY_MINUS && metric != BG_METRIC_ALTERNATING) return BG_ERR_ARG;
    if (count == 0) return BG_OK;
    if (!momenta || !chi || !eps || !eps_tilde || eps == eps_tilde) return BG_ERR_ARG;
    switch (field) {
        case BG_FIELD_FP31: {
            bg::SpinorConsts<Fp31> sc;
            if (!bg_spinor_consts_fp(bg::kP, metric, nullptr, &sc.jm, &sc.jv)) return BG_ERR_UNSUPPORTED;
            return launch<Fp31>(Fp31::Params{}, sc, metric, d, count, momenta, chi, eps, eps_tilde, status, stream);
        }
        case BG_FIELD_FPMONT: {
            FpMont::Params q{};
            if (!bg_mont_constants(prime, 0, &q)) return BG_ERR_ARG;
            bg::SpinorConsts<FpMont> sc;
            if (!bg_spinor_consts_fp(prime, metric, &q, &sc.jm, &sc.jv)) return BG_ERR_UNSUPPORTED;
            return launch<FpMont>(q, sc, metric, d, count, momenta, chi, eps, eps_tilde, status, stream);
        }
        case BG_FIELD_C128: {
            bg::SpinorConsts<C128> sc;
            sc.jm = metric == BG_METRIC_MOSTLY_MINUS ? make_double2(0.0, 1.0) : make_double2(-1.0, 0.0);
            sc.jv = metric == BG_METRIC_MOSTLY_MINUS ? make_double2(0.0, 1.0) : make_double2(1.0, 0.0);
            return launch<C128>(C128::Params{}, sc, metric, d, count, momenta, chi, eps, eps_tilde, status, stream);
        }
    }
    return BG_ERR_ARG;
}
