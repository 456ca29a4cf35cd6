// bg_noalloc.cu -- bg_amplitudes_host_noalloc: the host-buffer entry point for callers that cannot
// allocate device memory.  Declared and documented in include/bg.h.
//
// Who this is for.  bg_amplitudes_host needs device scratch (the staging area its H2D copies land in and
// its D2H copies leave from) and asks the caller for it.  Some callers have no way to provide any:
//   * a plug-in that runs beside a framework whose caching allocator has already taken (nearly) all of
//     HBM -- a cudaMalloc of its own fails there although the framework's pool is mostly idle;
//   * a caller on a latency-critical path: cudaMalloc / cudaFree synchronise the whole device, which stalls
//     every other stream of the process for as long as the longest running kernel;
//   * a plain C or Fortran host program that owns host arrays only and links no allocator at all.
// For them the staging area lives in the library image itself: a file-scope __device__ array, reserved by
// the CUDA runtime when the module is loaded on a device and held until the process exits.  Nothing is
// allocated at call time (no cudaMalloc / cudaFree / cudaMallocAsync, no stream or event creation, no
// library routine that allocates): the call is two H2D copies, one kernel launch through bg_amplitudes_status,
// one or two D2H copies, all on the caller's stream, then a wait for that stream.
//
// The price: BG_NOALLOC_SCRATCH_BYTES of HBM are held on every GPU that loads libbg_b200.so, used or not,
// and one call is limited to what fits (bg_noalloc_max_batch); no chunking is attempted -- a caller with
// more points calls again.  All calls share the one array: two calls whose GPU work overlaps (different
// streams, different host threads) race on it.  Calls are otherwise independent: the array keeps the
// previous call's bytes, but every byte a call reads back it has written first (inputs by the copies,
// out[b] and status[b] by the kernel for every b < batch), so nothing needs clearing.
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <mutex>

#include "../../include/bg.h"

namespace {

// the staging area.  In HOST code this name is only a handle for the runtime's symbol table -- it is not
// a device address and must never be passed to a kernel or a copy; scratch_base() asks the runtime for the
// address the symbol has on the current device.
static __device__ __align__(256) unsigned char g_noalloc_scratch[BG_NOALLOC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
void* g_base[kMaxDevices];                      // device address of g_noalloc_scratch, per device
std::atomic<bool> g_base_ready[kMaxDevices];
std::mutex g_base_mutex;

// Set-up, once per device, with that device current: resolve the symbol to its device address.
int scratch_base(unsigned char** base)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) { cudaGetLastError(); return BG_ERR_CUDA; }
    if (!g_base_ready[dev].load(std::memory_order_acquire)) {
        std::lock_guard<std::mutex> lock(g_base_mutex);
        if (!g_base_ready[dev].load(std::memory_order_relaxed)) {
            void* p = nullptr;
            if (cudaGetSymbolAddress(&p, g_noalloc_scratch) != cudaSuccess || !p) { cudaGetLastError(); return BG_ERR_CUDA; }
            if (reinterpret_cast<uintptr_t>(p) & 255u) return BG_ERR_CUDA;       // __align__(256) not honoured
            g_base[dev] = p;
            g_base_ready[dev].store(true, std::memory_order_release);
        }
    }
    *base = static_cast<unsigned char*>(g_base[dev]);
    return BG_OK;
}

bool shape_ok(int field, int n, int d)
{
    return (field == BG_FIELD_FP31 || field == BG_FIELD_C128) && n >= 4 && n <= 16 && d >= 4 && d <= 16;
}

size_t elem_bytes(int field) { return field == BG_FIELD_C128 ? 16 : 4; }
size_t round256(size_t x) { return (x + 255) & ~(size_t)255; }

// bytes of the staging area a call with `batch` points uses: momenta | polarisations | out | status
size_t need_bytes(int field, int n, int d, int64_t batch)
{
    const size_t w = elem_bytes(field);
    return 2 * round256((size_t)batch * n * d * w) + round256((size_t)batch * w) + round256((size_t)batch * 4);
}

}  // namespace

extern "C" {

size_t bg_noalloc_scratch_bytes(void) { return BG_NOALLOC_SCRATCH_BYTES; }

int64_t bg_noalloc_max_batch(int field, int n, int d)
{
    if (!shape_ok(field, n, d)) return 0;
    const size_t w = elem_bytes(field);
    int64_t b = (int64_t)(BG_NOALLOC_SCRATCH_BYTES / (2 * (size_t)n * d * w + w + 4));   // ignores the rounding
    while (b > 0 && need_bytes(field, n, d, b) > BG_NOALLOC_SCRATCH_BYTES) --b;
    return b;
}

int bg_amplitudes_host_noalloc(int field, int n, int d, int64_t batch, const void* host_momenta,
                               const void* host_polarisations, void* host_out, uint32_t* host_status,
                               cudaStream_t stream)
{
    if (!shape_ok(field, n, d) || batch < 0) return BG_ERR_ARG;
    if (batch == 0) return BG_OK;
    if (!host_momenta || !host_polarisations || !host_out) return BG_ERR_ARG;
    if (batch > bg_noalloc_max_batch(field, n, d)) return BG_ERR_TOO_LARGE;
    unsigned char* base = nullptr;
    int rc = scratch_base(&base);                   // first call on this device: cudaGetSymbolAddress
    if (rc != BG_OK) return rc;

    const size_t w = elem_bytes(field);
    const size_t in_bytes = (size_t)batch * n * d * w, in_slot = round256(in_bytes);
    unsigned char* dm = base;
    unsigned char* dp = dm + in_slot;
    unsigned char* dout = dp + in_slot;
    uint32_t* dst = reinterpret_cast<uint32_t*>(dout + round256((size_t)batch * w));

    cudaError_t e = cudaMemcpyAsync(dm, host_momenta, in_bytes, cudaMemcpyHostToDevice, stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dp, host_polarisations, in_bytes, cudaMemcpyHostToDevice, stream);
    if (e != cudaSuccess) { cudaGetLastError(); return BG_ERR_CUDA; }
    // the existing device entry point does the work: same kernel selection, same kernels, same results
    rc = bg_amplitudes_status(field, n, d, batch, dm, dp, dout, host_status ? dst : nullptr, stream);
    if (rc == BG_OK) {
        e = cudaMemcpyAsync(host_out, dout, (size_t)batch * w, cudaMemcpyDeviceToHost, stream);
        if (e == cudaSuccess && host_status)
            e = cudaMemcpyAsync(host_status, dst, (size_t)batch * 4, cudaMemcpyDeviceToHost, stream);
        if (e != cudaSuccess) rc = BG_ERR_CUDA;
    }
    // wait also after a failed enqueue: the copies already queued read the caller's host arrays
    if (cudaStreamSynchronize(stream) != cudaSuccess) rc = BG_ERR_CUDA;
    if (rc == BG_ERR_CUDA) cudaGetLastError();
    return rc;
}

}  // extern "C"
