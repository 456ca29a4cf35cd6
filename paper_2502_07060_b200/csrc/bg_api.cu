// bg_api.cu -- host side of libbg_b200: argument checks, kernel selection, launches.
// The C ABI is declared and documented in include/bg.h.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#include <atomic>
#include <mutex>

#include "../../include/bg.h"
#include "bg_common.cuh"
#include "bg_entries.h"
#include "bg_general.cuh"     // GeneralLayout (host side of the record layout)
#include "bg_host_util.h"
#include "bg_rt_host.h"

namespace {

using bg::BgParams;
using bg::C128;
using bg::Fp31;
using bg::FpMont;

constexpr int kMaxSmemPerBlock = 232448;   // 227 KB opt-in limit per CTA on sm_100
constexpr int kSmemPerSm = 233472;         // 228 KB per SM
constexpr int kSmemReservedPerBlock = 1024;
constexpr int kMaxDevices = 64;

// ---- kernel selection ------------------------------------------------------------------------------
// What a call launches, resolved ONCE per (field, metric, n, d, needs-states) and cached; the
// steady-state call path does no table scan, no getenv and no cudaFuncSetAttribute.
struct Launch {
    const void* func = nullptr;
    int kind = BG_KIND_GENERAL;        // BgKernelKind
    int threads = 0;
    int points_per_block = 0;
    int smem = 0;
    int stride = 0;                    // general kernel: record stride in elements
    std::atomic<uint64_t> attr_done{0};   // bit i: cudaFuncSetAttribute done on device i
    // bg_rt_kernel: layout and schedule built by the host (kept for the life of the process); every launch
    // carries them in its parameter block
    RtHost* rt = nullptr;
    uint64_t rt_id = 0;                // identifies the contents of *rt (the override path rebuilds it in place)
};

std::atomic<uint64_t> g_rt_ids{0};

std::atomic<int> g_override_kind{-1};   // bg_kernel_info_t.specialised numbering; -1 = default
std::atomic<int> g_override_w{0};

struct EnvInit {
    EnvInit()
    {   // initial value of the override, read once at load time (bg.h "tuning")
        const char* k = getenv("BG_KERNEL");
        const char* w = getenv("BG_KERNEL_W");
        if (k) {
            g_override_kind = strcmp(k, "general") == 0 ? 0 : strcmp(k, "unit1") == 0 ? 1 :
                              strcmp(k, "unit2") == 0 ? 2 : strcmp(k, "reg") == 0 ? 3 : strcmp(k, "rt") == 0 ? 4 : -1;
        }
        if (w) g_override_w = atoi(w);
    }
} g_env_init;

int elem_bytes(int field) { return field == BG_FIELD_C128 ? 16 : 4; }
int vec_width(int field, int d)
{
    if (field == BG_FIELD_C128) return 1;
    return (d % 4 == 0) ? 4 : (d % 2 == 0) ? 2 : 1;
}

const KernelEntry* find_entry(int field, int metric, int n, int d, bool multi_state, int want_kind, int want_w)
{
    typedef const KernelEntry* (*TableFn)(int*);
#define BG_TABLE_PTR(name) bg_entries_##name,
    static const TableFn tables[] = {BG_ENTRY_TABLES(BG_TABLE_PTR)};
#undef BG_TABLE_PTR
    const KernelEntry* first = nullptr;
    for (TableFn fn : tables) {
        int count = 0;
        const KernelEntry* t = fn(&count);
        for (int i = 0; i < count; ++i) {
            const KernelEntry& e = t[i];
            if (e.field != field || e.metric != metric || e.n != n || e.d != d) continue;
            if ((multi_state ? e.smem_multi : e.smem) > (size_t)kMaxSmemPerBlock) continue;
            if (multi_state && !e.func_multi) continue;                 // bg_reg_kernel: one configuration only
            if (want_kind >= 0 && e.kind != want_kind) continue;
            if (!first) first = &e;
            if (want_w == 0 || e.w == want_w) return &e;
        }
    }
    return first;
}

const void* general_ptr(int field, int metric, int d)
{
    switch (field) {
        case BG_FIELD_FP31: return bg_general_kernel_ptr_fp31(metric, d);
        case BG_FIELD_C128: return bg_general_kernel_ptr_c128(metric, d);
        case BG_FIELD_FPMONT: return bg_general_kernel_ptr_mont(metric, d);
    }
    return nullptr;
}

int fill_general(int field, int metric, int n, int d, Launch* L)
{
    const bg::GeneralLayout lay = bg::make_general_layout(n, d, vec_width(field, d));
    const int per_point = lay.stride * elem_bytes(field);
    int t = kMaxSmemPerBlock / per_point;
    if (t < 1) return BG_ERR_UNSUPPORTED;
    if (t > 32) t = 32;
    L->func = general_ptr(field, metric, d);
    if (!L->func) return BG_ERR_UNSUPPORTED;
    L->kind = BG_KIND_GENERAL;
    L->threads = t;
    L->points_per_block = t;
    L->smem = t * per_point;
    L->stride = lay.stride;
    return BG_OK;
}

const void* rt_ptr(int field, int metric, int d, int s, int w, bool multi)
{
    switch (field) {
        case BG_FIELD_FP31: return bg_rt_kernel_ptr_fp31(metric, d, s, w, multi);
        case BG_FIELD_C128: return bg_rt_kernel_ptr_c128(metric, d, s, w, multi);
        case BG_FIELD_FPMONT: return bg_rt_kernel_ptr_mont(metric, d, s, w, multi);
    }
    return nullptr;
}

// the tiled kernel for a run-time n: one lane per point if a 32-point tile fits shared memory (complex128: two
// lanes per point first, as in the compiled tables), else two lanes per point, else not available
int fill_rt(int field, int metric, int n, int d, bool multi, Launch* L)
{
    const int first = field == BG_FIELD_C128 && d % 2 == 0 ? 2 : 1;
    for (int pass = 0; pass < 2; ++pass) {
        const int s = pass == 0 ? first : 3 - first;
        if (d % s != 0) continue;
        const void* fn = rt_ptr(field, metric, d, s, bg_rt_warps(n), multi);
        if (!fn) continue;
        // a cached Launch is filled once and keeps its RtHost for the life of the process; the one Launch of
        // the override path is refilled when the override changes and reuses its RtHost
        RtHost* h = L->rt ? L->rt : new RtHost();
        memset(static_cast<void*>(h), 0, sizeof(RtHost));
        if (!bg_rt_make(elem_bytes(field), vec_width(field, d), n, d, s, multi, h) || h->smem > (size_t)kMaxSmemPerBlock) {
            if (!L->rt) delete h;
            continue;
        }
        L->func = fn;
        L->kind = BG_KIND_RT;
        L->threads = h->threads;
        L->points_per_block = h->points_per_block;
        L->smem = (int)h->smem;
        L->stride = 0;
        L->rt = h;
        L->rt_id = ++g_rt_ids;
        return BG_OK;
    }
    return BG_ERR_UNSUPPORTED;
}

// run-time-n shapes: the tiled kernel where it applies, else one thread per point
int fill_uncompiled(int field, int metric, int n, int d, bool multi_state, Launch* L)
{
    if (fill_rt(field, metric, n, d, multi_state, L) == BG_OK) return BG_OK;
    return fill_general(field, metric, n, d, L);
}

void fill_entry(const KernelEntry& e, bool multi, Launch* L)
{
    L->func = multi ? e.func_multi : e.func;
    L->kind = e.kind;
    L->threads = 32 * e.w;
    L->points_per_block = e.tp;
    L->smem = (int)(multi ? e.smem_multi : e.smem);
    L->stride = 0;
}

int check_shape(int field, int metric, int n, int d)
{
    if (field != BG_FIELD_FP31 && field != BG_FIELD_C128 && field != BG_FIELD_FPMONT) return BG_ERR_ARG;
    if (metric != BG_METRIC_MOSTLY_MINUS && metric != BG_METRIC_ALTERNATING) return BG_ERR_ARG;
    if (n < 4 || n > 16 || d < 4 || d > 16) return BG_ERR_ARG;
    return BG_OK;
}

// default selection, cached: [field][metric][multi_state][n][d]
Launch g_cache[3][2][2][17][17];
std::atomic<unsigned char> g_cache_state[3][2][2][17][17];      // 0 empty, 1 ready, 2 unsupported
std::mutex g_cache_mutex;
// selection under an override: rebuilt when the override changes (measurement path, not hot)
Launch g_over;
int g_over_key[7] = {-2, 0, 0, 0, 0, 0, 0};

int select(int field, int metric, int n, int d, bool multi_state, Launch** out)
{
    const int ok = g_override_kind.load(std::memory_order_relaxed), ow = g_override_w.load(std::memory_order_relaxed);
    if (ok >= 0) {
        std::lock_guard<std::mutex> lock(g_cache_mutex);
        const int key[7] = {ok, ow, field, metric, n, d, (int)multi_state};
        if (memcmp(key, g_over_key, sizeof(key)) != 0) {
            g_over.attr_done = 0;
            const KernelEntry* e = ok == 0 || ok == 4 ? nullptr
                                                      : find_entry(field, metric, n, d, multi_state, ok - 1, ow);
            int rc = BG_OK;
            if (e) fill_entry(*e, multi_state, &g_over);
            else if (ok == 0) rc = fill_general(field, metric, n, d, &g_over);
            else if (ok == 4) rc = fill_uncompiled(field, metric, n, d, multi_state, &g_over);
            else if (!(e = find_entry(field, metric, n, d, multi_state, -1, 0)))
                rc = fill_uncompiled(field, metric, n, d, multi_state, &g_over);
            else fill_entry(*e, multi_state, &g_over);
            if (rc != BG_OK) { g_over_key[0] = -2; return rc; }
            memcpy(g_over_key, key, sizeof(key));
        }
        *out = &g_over;
        return BG_OK;
    }
    Launch* L = &g_cache[field][metric][multi_state][n][d];
    std::atomic<unsigned char>& st = g_cache_state[field][metric][multi_state][n][d];
    unsigned char s = st.load(std::memory_order_acquire);
    if (s == 0) {
        std::lock_guard<std::mutex> lock(g_cache_mutex);
        s = st.load(std::memory_order_relaxed);
        if (s == 0) {
            int rc = BG_OK;
            if (const KernelEntry* e = find_entry(field, metric, n, d, multi_state, -1, 0)) fill_entry(*e, multi_state, L);
            else rc = fill_uncompiled(field, metric, n, d, multi_state, L);
            s = rc == BG_OK ? 1 : 2;
            st.store(s, std::memory_order_release);
        }
    }
    if (s != 1) return BG_ERR_UNSUPPORTED;
    *out = L;
    return BG_OK;
}

int ensure_attr(Launch* L)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) { cudaGetLastError(); return BG_ERR_CUDA; }
    const uint64_t bit = 1ull << dev;
    if (L->attr_done.load(std::memory_order_acquire) & bit) return BG_OK;
    if (cudaFuncSetAttribute(L->func, cudaFuncAttributeMaxDynamicSharedMemorySize, L->smem) != cudaSuccess) {
        cudaGetLastError();
        return BG_ERR_CUDA;
    }
    L->attr_done.fetch_or(bit, std::memory_order_release);
    return BG_OK;
}

}  // namespace

// ---- Montgomery constants of a prime (also used by bg_state_sum.cu) ----------------------------------
bool bg_mont_constants(uint32_t p, int i, bg::FpMont::Params* q)
{
    if (!(p & 1u) || p <= (1u << 30) || p >= (1u << 31)) return false;
    uint32_t inv = p;                                  // Newton: inv = p^-1 mod 2^32 (p odd; 3 bits correct at start)
    for (int k = 0; k < 5; ++k) inv *= 2u - p * inv;
    const uint64_t r = ((uint64_t)1 << 32) % p;
    q->p[i] = p;
    q->pinv[i] = 0u - inv;
    q->one[i] = (uint32_t)r;
    q->r2[i] = (uint32_t)(r * r % p);
    q->half[i] = (uint32_t)(r * ((p + 1u) / 2u) % p);
    return true;
}

namespace {

uint64_t powmod(uint64_t a, uint64_t e, uint64_t p)
{
    uint64_t r = 1;
    for (a %= p; e; e >>= 1) {
        if (e & 1) r = r * a % p;
        a = a * a % p;
    }
    return r;
}

}  // namespace

bool bg_spinor_consts_fp(uint32_t p, int metric, const bg::FpMont::Params* q, uint32_t* jm, uint32_t* jv)
{
    uint64_t m, v;
    if (metric == BG_METRIC_ALTERNATING) {
        m = p - 1u;
        v = 1u;
    } else {
        if (p % 4u != 1u) return false;
        // a quadratic non-residue: g^((p-1)/2) = -1.  For a prime the smallest one is tiny (half of all residues
        // qualify); primality is the caller's job, so the search is bounded: a composite p for which no small g
        // passes is refused instead of hanging the host
        uint64_t g = 2;
        while (g < 256 && powmod(g, (p - 1u) / 2u, p) != p - 1u) ++g;
        if (g == 256) return false;
        m = v = powmod(g, (p - 1u) / 4u, p);              // sqrt(-1)
    }
    if (q) {                                              // to Montgomery form: x R mod p
        m = m * q->one[0] % p;
        v = v * q->one[0] % p;
    }
    *jm = (uint32_t)m;
    *jv = (uint32_t)v;
    return true;
}

namespace {

int sm_count()
{
    static std::atomic<int> cached[kMaxDevices];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) { cudaGetLastError(); return 0; }
    int n = cached[dev].load(std::memory_order_relaxed);
    if (n == 0) {
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) { cudaGetLastError(); n = 0; }
        cached[dev].store(n, std::memory_order_relaxed);
    }
    return n;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

template <class F>
int launch_typed(Launch* L, const bg_problem_t& pb, const typename F::Params& fld, int64_t batch, const void* mom,
                 const void* pol, void* out, void* cur, uint32_t* status, cudaStream_t stream)
{
    typedef typename F::E E;
    BgParams<F> prm;
    prm.mom = static_cast<const E*>(mom);
    prm.pol = static_cast<const E*>(pol);
    prm.out = static_cast<E*>(out);
    prm.currents = static_cast<E*>(cur);
    prm.status = status;
    prm.batch = batch;
    prm.states = pb.states;
    prm.n_orderings = pb.n_orderings > 1 || pb.orderings ? (pb.n_orderings < 1 ? 1 : pb.n_orderings) : 1;
    prm.orderings = pb.orderings;
    prm.n = pb.n;
    prm.stride = L->stride;
    prm.fld = fld;
    int rc = ensure_attr(L);
    if (rc != BG_OK) return rc;
    if (L->kind == BG_KIND_RT) prm.rt = L->rt->lay;
    int64_t blocks = (batch + L->points_per_block - 1) / L->points_per_block;
    if (blocks > 0x7fffffffLL) return BG_ERR_ARG;
    if (L->kind == BG_KIND_REG) {                       // persistent warps: at most the resident blocks of the device
        const int64_t resident = (int64_t)sm_count() * (kSmemPerSm / (L->smem + kSmemReservedPerBlock));
        if (resident > 0 && blocks > resident) blocks = resident;
    }
    const unsigned gy = pb.field == BG_FIELD_FPMONT ? (unsigned)pb.n_primes : 1u;
    bg::RtParams<F>* rp = nullptr;
    if (L->kind == BG_KIND_RT) {
        // the schedule travels in the parameter block (29 KB).  It is staged in a per-thread block that keeps the
        // tables of the shape launched last: a repeated shape costs no allocation and no 29 KB copy, only `base`
        // is patched (cudaLaunchKernel copies the parameters before it returns)
        thread_local bg::RtParams<F> staged;
        thread_local uint64_t staged_id = 0;
        if (staged_id != L->rt_id) {
            staged.tab = L->rt->tab;
            staged_id = L->rt_id;
        }
        staged.base = prm;
        rp = &staged;
    }
    void* args[] = {rp ? static_cast<void*>(rp) : static_cast<void*>(&prm)};
    const cudaError_t err = cudaLaunchKernel(L->func, dim3((unsigned)blocks, gy), dim3(L->threads), args, L->smem, stream);
    if (err != cudaSuccess) {
        cudaGetLastError();
        return BG_ERR_CUDA;
    }
    return BG_OK;
}

int check_problem(const bg_problem_t* pb)
{
    if (!pb) return BG_ERR_ARG;
    int rc = check_shape(pb->field, pb->metric, pb->n, pb->d);
    if (rc != BG_OK) return rc;
    if (pb->states < 1 || pb->states > 65535) return BG_ERR_ARG;
    if (pb->n_orderings < 0 || pb->n_orderings > (1 << 24) || (pb->n_orderings > 1 && !pb->orderings)) return BG_ERR_ARG;
    // the sweeps of one tile are numbered o * states + s (times 16 levels) in 32-bit arithmetic inside the kernels
    if ((int64_t)(pb->n_orderings < 1 ? 1 : pb->n_orderings) * pb->states >= ((int64_t)1 << 27)) return BG_ERR_ARG;
    if (pb->field == BG_FIELD_FPMONT) {
        if (pb->n_primes < 1 || pb->n_primes > BG_MAX_PRIMES) return BG_ERR_ARG;
    } else if (pb->n_primes != 0) {
        return BG_ERR_ARG;
    }
    return BG_OK;
}

int run(const bg_problem_t& pb, int64_t batch, const void* mom, const void* pol, void* out, void* cur,
        uint32_t* status, cudaStream_t stream)
{
    int rc = check_problem(&pb);
    if (rc != BG_OK) return rc;
    FpMont::Params mont{};
    if (pb.field == BG_FIELD_FPMONT)
        for (int i = 0; i < pb.n_primes; ++i)
            if (!bg_mont_constants(pb.primes[i], i, &mont)) return BG_ERR_ARG;
    Launch* L = nullptr;
    rc = select(pb.field, pb.metric, pb.n, pb.d, pb.states > 1 || pb.orderings, &L);
    if (rc != BG_OK) return rc;
    if (batch < 0) return BG_ERR_ARG;
    if (batch == 0) return BG_OK;
    if (!mom || !pol || !out) return BG_ERR_ARG;
    if (!aligned16(mom) || !aligned16(pol) || !aligned16(out) || !aligned16(cur) ||
        (reinterpret_cast<uintptr_t>(status) & 3u))
        return BG_ERR_ARG;
    if (out == mom || out == pol) return BG_ERR_ARG;
    if (cur && (pb.states != 1 || pb.n_primes > 1 || pb.orderings)) return BG_ERR_ARG;
    switch (pb.field) {
        case BG_FIELD_FP31: return launch_typed<Fp31>(L, pb, Fp31::Params{}, batch, mom, pol, out, cur, status, stream);
        case BG_FIELD_C128: return launch_typed<C128>(L, pb, C128::Params{}, batch, mom, pol, out, cur, status, stream);
        default: return launch_typed<FpMont>(L, pb, mont, batch, mom, pol, out, cur, status, stream);
    }
}

bg_problem_t simple_problem(int field, int metric, int n, int d, int states)
{
    bg_problem_t pb;
    memset(&pb, 0, sizeof(pb));
    pb.field = field; pb.metric = metric; pb.n = n; pb.d = d; pb.states = states;
    return pb;
}

int64_t binom(int n, int k)
{
    if (k < 0 || k > n) return 0;
    int64_t r = 1;
    for (int i = 1; i <= k; ++i) r = r * (n - k + i) / i;
    return r;
}

size_t round256(size_t x) { return (x + 255) & ~(size_t)255; }

// two persistent streams per device for bg_amplitudes_host, created on first use and never destroyed
cudaStream_t g_host_streams[kMaxDevices][2];
std::atomic<bool> g_host_streams_ready[kMaxDevices];
std::mutex g_host_mutex;

int host_streams(cudaStream_t (&s)[2])
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) { cudaGetLastError(); return BG_ERR_CUDA; }
    if (!g_host_streams_ready[dev].load(std::memory_order_acquire)) {
        std::lock_guard<std::mutex> lock(g_host_mutex);
        if (!g_host_streams_ready[dev].load(std::memory_order_relaxed)) {
            for (int i = 0; i < 2; ++i)
                if (cudaStreamCreateWithFlags(&g_host_streams[dev][i], cudaStreamNonBlocking) != cudaSuccess) {
                    cudaGetLastError();
                    return BG_ERR_CUDA;
                }
            g_host_streams_ready[dev].store(true, std::memory_order_release);
        }
    }
    s[0] = g_host_streams[dev][0];
    s[1] = g_host_streams[dev][1];
    return BG_OK;
}

}  // namespace

extern "C" {

int bg_amplitudes(int field, int n, int d, int64_t batch, const void* momenta, const void* polarisations,
                  void* out, cudaStream_t stream)
{
    if (field == BG_FIELD_FPMONT) return BG_ERR_ARG;          // needs a prime: bg_amplitudes_primes / bg_evaluate
    return run(simple_problem(field, BG_METRIC_MOSTLY_MINUS, n, d, 1), batch, momenta, polarisations, out, nullptr,
               nullptr, stream);
}

int bg_amplitudes_status(int field, int n, int d, int64_t batch, const void* momenta,
                         const void* polarisations, void* out, uint32_t* status, cudaStream_t stream)
{
    if (field == BG_FIELD_FPMONT) return BG_ERR_ARG;
    return run(simple_problem(field, BG_METRIC_MOSTLY_MINUS, n, d, 1), batch, momenta, polarisations, out, nullptr,
               status, stream);
}

int bg_currents(int field, int n, int d, int64_t batch, const void* momenta, const void* polarisations,
                void* out, void* currents, uint32_t* status, cudaStream_t stream)
{
    if (field == BG_FIELD_FPMONT) return BG_ERR_ARG;
    return run(simple_problem(field, BG_METRIC_MOSTLY_MINUS, n, d, 1), batch, momenta, polarisations, out, currents,
               status, stream);
}

int bg_evaluate(const bg_problem_t* problem, int64_t batch, const void* momenta, const void* polarisations,
                void* out, void* currents, uint32_t* status, cudaStream_t stream)
{
    if (!problem) return BG_ERR_ARG;
    return run(*problem, batch, momenta, polarisations, out, currents, status, stream);
}

int bg_amplitudes_states(int field, int n, int d, int64_t batch, int states, const void* momenta,
                         const void* polarisations, void* out, uint32_t* status, cudaStream_t stream)
{
    if (field == BG_FIELD_FPMONT) return BG_ERR_ARG;
    return run(simple_problem(field, BG_METRIC_MOSTLY_MINUS, n, d, states), batch, momenta, polarisations, out,
               nullptr, status, stream);
}

int bg_amplitudes_orderings(int field, int n, int d, int64_t batch, int n_orderings, const unsigned char* orderings,
                            const void* momenta, const void* polarisations, void* out, uint32_t* status,
                            cudaStream_t stream)
{
    if (field == BG_FIELD_FPMONT || n_orderings < 1 || !orderings) return BG_ERR_ARG;
    bg_problem_t pb = simple_problem(field, BG_METRIC_MOSTLY_MINUS, n, d, 1);
    pb.n_orderings = n_orderings;
    pb.orderings = orderings;
    return run(pb, batch, momenta, polarisations, out, nullptr, status, stream);
}

int bg_amplitudes_primes(int metric, int n, int d, int64_t batch, int n_primes, const uint32_t* primes,
                         const void* momenta, const void* polarisations, void* out, uint32_t* status,
                         cudaStream_t stream)
{
    if (!primes || n_primes < 1 || n_primes > BG_MAX_PRIMES) return BG_ERR_ARG;
    bg_problem_t pb = simple_problem(BG_FIELD_FPMONT, metric, n, d, 1);
    pb.n_primes = n_primes;
    for (int i = 0; i < n_primes; ++i) pb.primes[i] = primes[i];
    return run(pb, batch, momenta, polarisations, out, nullptr, status, stream);
}

int bg_set_kernel_override(int kind, int warps)
{
    g_override_kind = kind < 0 || kind > 4 ? -1 : kind;
    g_override_w = warps < 0 ? 0 : warps;
    return BG_OK;
}

size_t bg_host_workspace_bytes(int field, int n, int d, int64_t chunk_points)
{
    if (check_shape(field, BG_METRIC_MOSTLY_MINUS, n, d) != BG_OK || field == BG_FIELD_FPMONT || chunk_points <= 0)
        return 0;
    const size_t w = elem_bytes(field);
    const size_t in = round256((size_t)chunk_points * n * d * w);
    const size_t o = round256((size_t)chunk_points * w);
    const size_t st = round256((size_t)chunk_points * 4);
    return 2 * (2 * in + o + st);
}

int bg_amplitudes_host(int field, int n, int d, int64_t batch, const void* host_momenta,
                       const void* host_polarisations, void* host_out, uint32_t* host_status,
                       void* workspace, size_t workspace_bytes)
{
    if (field == BG_FIELD_FPMONT) return BG_ERR_ARG;
    const bg_problem_t pb = simple_problem(field, BG_METRIC_MOSTLY_MINUS, n, d, 1);
    int rc = check_problem(&pb);
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
    const size_t w = elem_bytes(field);
    const size_t in_b = round256((size_t)chunk * n * d * w);
    const size_t out_b = round256((size_t)chunk * w);
    const size_t st_b = round256((size_t)chunk * 4);
    const size_t slot_b = 2 * in_b + out_b + st_b;

    cudaStream_t s[2];
    rc = host_streams(s);
    if (rc != BG_OK) return rc;
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
        rc = run(pb, nb, dm, dp, dout, nullptr, host_status ? dst : nullptr, st);
        if (rc != BG_OK) break;
        e = cudaMemcpyAsync(static_cast<unsigned char*>(host_out) + (size_t)done * w, dout, (size_t)nb * w,
                            cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && host_status)
            e = cudaMemcpyAsync(host_status + done, dst, (size_t)nb * 4, cudaMemcpyDeviceToHost, st);
        if (e != cudaSuccess) { rc = BG_ERR_CUDA; break; }
    }
    for (int i = 0; i < 2; ++i)
        if (cudaStreamSynchronize(s[i]) != cudaSuccess) rc = BG_ERR_CUDA;
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
        case BG_ERR_TOO_LARGE: return "batch exceeds bg_noalloc_max_batch (the fixed scratch array of the no-allocation entry point)";
    }
    return "unknown status";
}

const char* bg_version(void) { return "bg_b200 0.2 (sm_100a)"; }

int bg_op_count(int field, int n, int d, bg_opcount_t* out)
{
    if (check_shape(field, BG_METRIC_MOSTLY_MINUS, n, d) != BG_OK || !out) return BG_ERR_ARG;
    const int m = n - 1;
    const int64_t R = (int64_t)m * (m - 1) / 2 - 1;
    const int64_t w = elem_bytes(field);
    out->currents = (int64_t)n * (n - 1) / 2;
    out->propagators = R;
    out->splits3 = binom(n, 3);
    out->splits4 = binom(n, 4);
    out->mul_v3 = 6 * d * out->splits3;
    out->mul_v4 = 6 * d * out->splits4;
    out->mul_other = d * R + 3 * (R - 1) + d * R + d;
    out->mul_ref = out->mul_v3 + out->mul_v4 + out->mul_other;
    // what the kernels' factored form executes (bg.h): per 3-split 3 dots + 3 axpys, per 4-split 1 dot + 1
    // axpy; per multi-gluon current (R + 1 of them) the boundary term (d), sum_k h_k / 2 (1) and, unless
    // top, the propagator (d) and 2 P.J (d); the final contraction (d); single-gluon 2 k.eps (m d);
    // invariants (d R) and the batch inverse (3 (R-1) + 38 for the inversion chain)
    out->mul_factored = 6 * d * out->splits3 + 2 * d * out->splits4 + (R + 1) * (d + 1) + 2 * d * R + d +
                        (int64_t)m * d + d * R + 3 * (R - 1) + 38;
    out->bytes_in = 2 * (int64_t)n * d * w;
    out->bytes_out = w;
    return BG_OK;
}

int bg_kernel_info_problem(const bg_problem_t* problem, bg_kernel_info_t* out)
{
    if (!out) return BG_ERR_ARG;
    int rc = check_problem(problem);
    if (rc != BG_OK) return rc;
    Launch* L = nullptr;
    rc = select(problem->field, problem->metric, problem->n, problem->d, problem->states > 1 || problem->orderings, &L);
    if (rc != BG_OK) return rc;
    out->specialised = L->kind == BG_KIND_GENERAL ? 0 : L->kind == BG_KIND_RT ? 4 : 1 + L->kind;
    out->threads_per_block = L->threads;
    out->points_per_block = L->points_per_block;
    out->smem_bytes_per_block = L->smem;
    out->smem_bytes_per_point = L->smem / L->points_per_block;
    int bps = kSmemPerSm / (out->smem_bytes_per_block + kSmemReservedPerBlock);
    out->blocks_per_sm = bps > 32 ? 32 : bps;
    cudaFuncAttributes attr;
    if (cudaFuncGetAttributes(&attr, L->func) == cudaSuccess) {
        out->regs_per_thread = attr.numRegs;
    } else {
        cudaGetLastError();
        out->regs_per_thread = -1;
    }
    return BG_OK;
}

int bg_kernel_info(int field, int n, int d, bg_kernel_info_t* out)
{
    bg_problem_t pb = simple_problem(field, BG_METRIC_MOSTLY_MINUS, n, d, 1);
    if (field == BG_FIELD_FPMONT) { pb.n_primes = 1; pb.primes[0] = 2147483629u; }
    return bg_kernel_info_problem(&pb, out);
}

}  // extern "C"
