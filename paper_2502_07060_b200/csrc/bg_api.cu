// bg_api.cu -- host side of libbg_b200: argument checks, kernel selection, launches.
// The C ABI is declared and documented in include/bg.h.
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include "../../include/bg.h"
#include "bg_recursion.cuh"
#include "bg_tile.cuh"      // TileParams
#include "bg_entries.h"
#include <stdlib.h>

namespace {

using bg::C128;
using bg::Fp31;
using bg::KernelParams;

constexpr int kMaxSmemPerBlock = 232448;   // 227 KB opt-in limit per CTA on sm_100
constexpr int kSmemPerSm = 233472;         // 228 KB per SM
constexpr int kSmemReservedPerBlock = 1024;

struct LaunchPlan {
    const void* func;
    int specialised;
    int threads;
    int stride;            // record stride in elements
    int elem_bytes;
    int smem_bytes;
};

template <class F, int N, int D>
const void* kernel_ptr()
{
    return reinterpret_cast<const void*>(&bg::bg_recursion_kernel<F, N, D>);
}

template <class F, int D>
const void* pick_d(int n, int* specialised);

// the (n, d) pairs of BASELINE.json:configs get fully compile-time instances
template <>
const void* pick_d<Fp31, 4>(int n, int* s)
{
    if (n == 4) { *s = 1; return kernel_ptr<Fp31, 4, 4>(); }
    *s = 0; return kernel_ptr<Fp31, 0, 4>();
}
template <>
const void* pick_d<Fp31, 6>(int n, int* s)
{
    if (n == 8) { *s = 1; return kernel_ptr<Fp31, 8, 6>(); }
    if (n == 12) { *s = 1; return kernel_ptr<Fp31, 12, 6>(); }
    *s = 0; return kernel_ptr<Fp31, 0, 6>();
}
template <>
const void* pick_d<Fp31, 8>(int n, int* s)
{
    if (n == 10) { *s = 1; return kernel_ptr<Fp31, 10, 8>(); }
    *s = 0; return kernel_ptr<Fp31, 0, 8>();
}
template <>
const void* pick_d<C128, 4>(int n, int* s)
{
    if (n == 6) { *s = 1; return kernel_ptr<C128, 6, 4>(); }
    *s = 0; return kernel_ptr<C128, 0, 4>();
}
template <>
const void* pick_d<C128, 6>(int n, int* s)
{
    if (n == 12) { *s = 1; return kernel_ptr<C128, 12, 6>(); }
    *s = 0; return kernel_ptr<C128, 0, 6>();
}
template <class F, int D>
const void* pick_d(int, int* s)
{
    *s = 0;
    return kernel_ptr<F, 0, D>();
}

template <class F>
const void* pick(int n, int d, int* s)
{
    switch (d) {
        case 4: return pick_d<F, 4>(n, s);
        case 5: return pick_d<F, 5>(n, s);
        case 6: return pick_d<F, 6>(n, s);
        case 7: return pick_d<F, 7>(n, s);
        case 8: return pick_d<F, 8>(n, s);
        case 9: return pick_d<F, 9>(n, s);
        case 10: return pick_d<F, 10>(n, s);
        case 11: return pick_d<F, 11>(n, s);
        case 12: return pick_d<F, 12>(n, s);
        case 13: return pick_d<F, 13>(n, s);
        case 14: return pick_d<F, 14>(n, s);
        case 15: return pick_d<F, 15>(n, s);
        case 16: return pick_d<F, 16>(n, s);
    }
    return nullptr;
}

// ---- the compile-time (n, d) fast path -------------------------------------------------------------
// The instances live in several translation units (bg_inst_*.cu): the work lists of a kernel
// instance sit in constant memory, and one module has 64 KB of it.
const SweepEntry* find_sweep(int field, int n, int d)
{
    const char* env = getenv("BG_SWEEP_W");
    const int want = env ? atoi(env) : 0;
    if (env && want == 0) return nullptr;            // BG_SWEEP_W=0: force the runtime-n kernel
    const char* kenv = getenv("BG_KERNEL");          // restrict the kernel family (A/B runs)
    const int kind = !kenv ? -1 : strcmp(kenv, "tile") == 0 ? 0 : strcmp(kenv, "level") == 0 ? 1 :
                                  strcmp(kenv, "split") == 0 ? 2 : strcmp(kenv, "reg") == 0 ? 3 :
                                  strcmp(kenv, "unit") == 0 ? 4 : -1;
    typedef const SweepEntry* (*TableFn)(int*);
    static const TableFn tables[] = {bg_entries_default, bg_entries_paper, bg_entries_grid0, bg_entries_grid1, bg_entries_grid2,
                                     bg_entries_cgrid0, bg_entries_cgrid1,
                                     bg_entries_fp_alt, bg_entries_c128_alt};
    const SweepEntry* first = nullptr;
    for (TableFn fn : tables) {
        int count = 0;
        const SweepEntry* t = fn(&count);
        for (int i = 0; i < count; ++i) {
            if (t[i].field != field || t[i].n != n || t[i].d != d) continue;
            if (kind >= 0 && t[i].kind != kind) continue;
            if (t[i].smem > (size_t)kMaxSmemPerBlock) continue;
            if (!first) first = &t[i];
            if (t[i].w == want) return &t[i];
        }
    }
    return first;
}

int vec_width(int field, int d)
{
    if (field == BG_FIELD_C128) return 1;
    return (d % 4 == 0) ? 4 : (d % 2 == 0) ? 2 : 1;
}

int check_shape(int field, int n, int d)
{
    if (field != BG_FIELD_FP31 && field != BG_FIELD_C128) return BG_ERR_ARG;
    if (n < 4 || n > 16 || d < 4 || d > 16) return BG_ERR_ARG;
    return BG_OK;
}

int make_plan(int field, int n, int d, LaunchPlan* plan)
{
    int rc = check_shape(field, n, d);
    if (rc != BG_OK) return rc;
    const bg::RecordLayout lay = bg::make_layout(n, d, vec_width(field, d));
    plan->elem_bytes = field == BG_FIELD_FP31 ? 4 : 16;
    plan->stride = lay.stride;
    const int per_point = lay.stride * plan->elem_bytes;
    int t = kMaxSmemPerBlock / per_point;
    if (t < 1) return BG_ERR_UNSUPPORTED;
    if (t > 32) t = 32;
    plan->threads = t;
    plan->smem_bytes = t * per_point;
    plan->func = field == BG_FIELD_FP31 ? pick<Fp31>(n, d, &plan->specialised)
                                        : pick<C128>(n, d, &plan->specialised);
    return plan->func ? BG_OK : BG_ERR_UNSUPPORTED;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

template <class E>
int launch_typed(const LaunchPlan& plan, int n, int64_t batch, const void* mom, const void* pol,
                 void* out, void* cur, uint32_t* status, cudaStream_t stream)
{
    KernelParams<E> prm;
    prm.mom = static_cast<const E*>(mom);
    prm.pol = static_cast<const E*>(pol);
    prm.out = static_cast<E*>(out);
    prm.currents = static_cast<E*>(cur);
    prm.status = status;
    prm.batch = batch;
    prm.n = n;
    prm.stride = plan.stride;
    if (cudaFuncSetAttribute(plan.func, cudaFuncAttributeMaxDynamicSharedMemorySize, plan.smem_bytes) !=
        cudaSuccess) {
        cudaGetLastError();
        return BG_ERR_CUDA;
    }
    const int64_t blocks = (batch + plan.threads - 1) / plan.threads;
    if (blocks > 0x7fffffffLL) return BG_ERR_ARG;
    void* args[] = {&prm};
    if (cudaLaunchKernel(plan.func, dim3((unsigned)blocks), dim3(plan.threads), args, plan.smem_bytes,
                         stream) != cudaSuccess) {
        cudaGetLastError();
        return BG_ERR_CUDA;
    }
    return BG_OK;
}

template <class E>
int launch_sweep(const SweepEntry& e, int64_t batch, const void* mom, const void* pol, void* out, void* cur,
                 uint32_t* status, cudaStream_t stream)
{
    bg::TileParams<E> prm;
    prm.mom = static_cast<const E*>(mom);
    prm.pol = static_cast<const E*>(pol);
    prm.out = static_cast<E*>(out);
    prm.currents = static_cast<E*>(cur);
    prm.status = status;
    prm.batch = batch;
    if (cudaFuncSetAttribute(e.func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)e.smem) != cudaSuccess) {
        cudaGetLastError();
        return BG_ERR_CUDA;
    }
    const int64_t blocks = (batch + e.tp - 1) / e.tp;
    if (blocks > 0x7fffffffLL) return BG_ERR_ARG;
    void* args[] = {&prm};
    if (cudaLaunchKernel(e.func, dim3((unsigned)blocks), dim3(32 * e.w), args, e.smem, stream) != cudaSuccess) {
        cudaGetLastError();
        return BG_ERR_CUDA;
    }
    return BG_OK;
}

int run(int field, int n, int d, int64_t batch, const void* mom, const void* pol, void* out, void* cur,
        uint32_t* status, cudaStream_t stream)
{
    LaunchPlan plan;
    int rc = make_plan(field, n, d, &plan);
    if (rc != BG_OK) return rc;
    if (batch < 0) return BG_ERR_ARG;
    if (batch == 0) return BG_OK;
    if (!mom || !pol || !out) return BG_ERR_ARG;
    if (!aligned16(mom) || !aligned16(pol) || !aligned16(out) || !aligned16(cur) ||
        (reinterpret_cast<uintptr_t>(status) & 3u))
        return BG_ERR_ARG;
    if (out == mom || out == pol) return BG_ERR_ARG;
    if (const SweepEntry* e = find_sweep(field, n, d)) {
        if (field == BG_FIELD_FP31) return launch_sweep<uint32_t>(*e, batch, mom, pol, out, cur, status, stream);
        return launch_sweep<double2>(*e, batch, mom, pol, out, cur, status, stream);
    }
    if (field == BG_FIELD_FP31)
        return launch_typed<uint32_t>(plan, n, batch, mom, pol, out, cur, status, stream);
    return launch_typed<double2>(plan, n, batch, mom, pol, out, cur, status, stream);
}

int64_t binom(int n, int k)
{
    if (k < 0 || k > n) return 0;
    int64_t r = 1;
    for (int i = 1; i <= k; ++i) r = r * (n - k + i) / i;
    return r;
}

size_t round256(size_t x) { return (x + 255) & ~(size_t)255; }

}  // namespace

extern "C" {

int bg_amplitudes(int field, int n, int d, int64_t batch, const void* momenta, const void* polarisations,
                  void* out, cudaStream_t stream)
{
    return run(field, n, d, batch, momenta, polarisations, out, nullptr, nullptr, stream);
}

int bg_amplitudes_status(int field, int n, int d, int64_t batch, const void* momenta,
                         const void* polarisations, void* out, uint32_t* status, cudaStream_t stream)
{
    return run(field, n, d, batch, momenta, polarisations, out, nullptr, status, stream);
}

int bg_currents(int field, int n, int d, int64_t batch, const void* momenta, const void* polarisations,
                void* out, void* currents, uint32_t* status, cudaStream_t stream)
{
    return run(field, n, d, batch, momenta, polarisations, out, currents, status, stream);
}

size_t bg_host_workspace_bytes(int field, int n, int d, int64_t chunk_points)
{
    if (check_shape(field, n, d) != BG_OK || chunk_points <= 0) return 0;
    const size_t w = field == BG_FIELD_FP31 ? 4 : 16;
    const size_t in = round256((size_t)chunk_points * n * d * w);
    const size_t o = round256((size_t)chunk_points * w);
    const size_t st = round256((size_t)chunk_points * 4);
    return 2 * (2 * in + o + st);
}

int bg_amplitudes_host(int field, int n, int d, int64_t batch, const void* host_momenta,
                       const void* host_polarisations, void* host_out, uint32_t* host_status,
                       void* workspace, size_t workspace_bytes)
{
    LaunchPlan plan;
    int rc = make_plan(field, n, d, &plan);
    if (rc != BG_OK) return rc;
    if (batch < 0) return BG_ERR_ARG;
    if (batch == 0) return BG_OK;
    if (!host_momenta || !host_polarisations || !host_out || !workspace) return BG_ERR_ARG;
    if (reinterpret_cast<uintptr_t>(workspace) & 255u) return BG_ERR_ARG;
    // largest chunk (multiple of 1024 points) whose double-buffered slots fit the workspace
    int64_t chunk = 0;
    for (int64_t c = 1024; c <= (int64_t)1 << 22; c += (c < 65536 ? 1024 : 65536)) {
        if (bg_host_workspace_bytes(field, n, d, c) <= workspace_bytes) chunk = c; else break;
        if (c >= batch) break;
    }
    if (chunk == 0) return BG_ERR_ARG;
    const size_t w = field == BG_FIELD_FP31 ? 4 : 16;
    const size_t in_b = round256((size_t)chunk * n * d * w);
    const size_t out_b = round256((size_t)chunk * w);
    const size_t st_b = round256((size_t)chunk * 4);
    const size_t slot_b = 2 * in_b + out_b + st_b;

    cudaStream_t s[2] = {nullptr, nullptr};
    for (int i = 0; i < 2; ++i)
        if (cudaStreamCreateWithFlags(&s[i], cudaStreamNonBlocking) != cudaSuccess) {
            cudaGetLastError();
            if (s[0]) cudaStreamDestroy(s[0]);
            return BG_ERR_CUDA;
        }
    rc = BG_OK;
    int64_t done = 0;
    for (int c = 0; done < batch && rc == BG_OK; ++c, done += chunk) {
        const int64_t nb = batch - done < chunk ? batch - done : chunk;
        unsigned char* base = static_cast<unsigned char*>(workspace) + (size_t)(c & 1) * slot_b;
        void* dm = base;
        void* dp = base + in_b;
        void* dout = base + 2 * in_b;
        uint32_t* dst = reinterpret_cast<uint32_t*>(base + 2 * in_b + out_b);
        cudaStream_t st = s[c & 1];
        const size_t off_in = (size_t)done * n * d * w;
        const size_t nbytes = (size_t)nb * n * d * w;
        cudaError_t e = cudaMemcpyAsync(dm, static_cast<const unsigned char*>(host_momenta) + off_in,
                                        nbytes, cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(dp, static_cast<const unsigned char*>(host_polarisations) + off_in,
                                nbytes, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) { rc = BG_ERR_CUDA; break; }
        rc = run(field, n, d, nb, dm, dp, dout, nullptr, host_status ? dst : nullptr, st);
        if (rc != BG_OK) break;
        e = cudaMemcpyAsync(static_cast<unsigned char*>(host_out) + (size_t)done * w, dout, (size_t)nb * w,
                            cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && host_status)
            e = cudaMemcpyAsync(host_status + done, dst, (size_t)nb * 4, cudaMemcpyDeviceToHost, st);
        if (e != cudaSuccess) { rc = BG_ERR_CUDA; break; }
    }
    for (int i = 0; i < 2; ++i) {
        if (cudaStreamSynchronize(s[i]) != cudaSuccess) rc = BG_ERR_CUDA;
        cudaStreamDestroy(s[i]);
    }
    if (rc == BG_ERR_CUDA) cudaGetLastError();
    return rc;
}

uint32_t bg_modulus(void) { return bg::kP; }

const char* bg_status_string(int status)
{
    switch (status) {
        case BG_OK: return "ok";
        case BG_ERR_ARG: return "invalid argument";
        case BG_ERR_UNSUPPORTED: return "unsupported (field, n, d)";
        case BG_ERR_CUDA: return "CUDA error";
    }
    return "unknown status";
}

const char* bg_version(void) { return "bg_b200 0.1 (sm_100a)"; }

int bg_op_count(int field, int n, int d, bg_opcount_t* out)
{
    if (check_shape(field, n, d) != BG_OK || !out) return BG_ERR_ARG;
    const int m = n - 1;
    const int64_t R = (int64_t)m * (m - 1) / 2 - 1;
    const int64_t w = field == BG_FIELD_FP31 ? 4 : 16;
    out->currents = (int64_t)n * (n - 1) / 2;
    out->propagators = R;
    out->splits3 = binom(n, 3);
    out->splits4 = binom(n, 4);
    out->mul_v3 = 6 * d * out->splits3;
    out->mul_v4 = 6 * d * out->splits4;
    out->mul_other = d * R + 3 * (R - 1) + d * R + d;
    out->mul_ref = out->mul_v3 + out->mul_v4 + out->mul_other;
    // kernel: per 3-split 3 dots + 4 axpys, per 4-split 1 dot + 1 axpy, invariants, propagators,
    // Montgomery trick, final contraction
    out->mul_factored = 7 * d * out->splits3 + 2 * d * out->splits4 + d * R + 3 * (R - 1) + d * R + d;
    out->bytes_in = 2 * (int64_t)n * d * w;
    out->bytes_out = w;
    return BG_OK;
}

int bg_kernel_info(int field, int n, int d, bg_kernel_info_t* out)
{
    if (!out) return BG_ERR_ARG;
    LaunchPlan plan;
    int rc = make_plan(field, n, d, &plan);
    if (rc != BG_OK) return rc;
    const void* func = plan.func;
    if (const SweepEntry* e = find_sweep(field, n, d)) {
        // the compile-time (n, d) fast path: one tile of 32 points per block, e->w warps
        out->specialised = 1 + e->kind;          // 1: bg_tile_kernel, 2: bg_level_kernel, 3: bg_split_kernel
        out->threads_per_block = 32 * e->w;
        out->points_per_block = e->tp;
        out->smem_bytes_per_block = (int)e->smem;
        out->smem_bytes_per_point = (int)(e->smem / e->tp);
        func = e->func;
    } else {
        out->specialised = 0;
        out->threads_per_block = plan.threads;
        out->points_per_block = plan.threads;
        out->smem_bytes_per_block = plan.smem_bytes;
        out->smem_bytes_per_point = plan.stride * plan.elem_bytes;
    }
    int bps = kSmemPerSm / (out->smem_bytes_per_block + kSmemReservedPerBlock);
    out->blocks_per_sm = bps > 32 ? 32 : bps;
    cudaFuncAttributes attr;
    if (cudaFuncGetAttributes(&attr, func) == cudaSuccess) {
        out->regs_per_thread = attr.numRegs;
    } else {
        cudaGetLastError();
        out->regs_per_thread = -1;
    }
    return BG_OK;
}

}  // extern "C"
