// oo_sort_static.cu — oo_sort_queries_static: row a1 (Morton order of the queries) for callers that must not allocate.
//
// Who that is: code that runs where device allocation is forbidden or impossible — a render loop that was given a fixed
// memory budget and no allocator after start-up, a plug-in inside a host application that owns the whole device heap, a
// real-time thread for which cudaMalloc's implicit device-wide synchronisation is a missed frame, or a process whose memory
// pool is already carved up and that has nothing left to hand to oo_reserve.  oo_sort_queries needs about 13 bytes of
// scratch per query from oo_reserve (= cudaMalloc); this variant runs the SAME kernels (launch_morton_sort, oo_sort.cu) on
// scratch that is part of the library image instead: one file-scope __device__ array, sized for OO_SORT_STATIC_MAX_QUERIES.
//
// What that costs: every GPU on which this translation unit's module gets loaded holds the array (13,643,776 bytes) from then
// until the process exits, whether or not the entry point is ever called again.
//
// The array's name below is a device symbol.  In HOST code `g_sort_scratch` is only a handle for the runtime, not an address a
// kernel may dereference, so the host side asks the runtime for the device address (cudaGetSymbolAddress) once per device,
// with that device current, and hands that pointer to the launcher.
#include <atomic>
#include <cstdarg>
#include <cstdio>

#include "oo_internal.h"

namespace {

constexpr uint64_t kMaxQueries = OO_SORT_STATIC_MAX_QUERIES;
constexpr uint64_t kKeyWords = kMaxQueries;   // one u32 per query in each of the three per-query arrays
// scratch layout in 32-bit words: keys_a | keys_b | idx_a | hist (the (digit, tile) table + the digit totals of three passes);
// every part starts on a multiple of 64 words = 256 bytes because kMaxQueries is one
constexpr uint64_t kHistWords = (kMaxQueries / 4096) * 1024 + 3 * 1024;
constexpr uint64_t kScratchWords = 3 * kKeyWords + kHistWords;
static_assert(kMaxQueries % 4096 == 0, "the histogram size below assumes whole 4096-key tiles at the maximum");
static_assert(kScratchWords * 4 == 13643776, "the size the header and the README state");

static __device__ __align__(256) uint32_t g_sort_scratch[kScratchWords];

// device address of g_sort_scratch per device ordinal; 0 = not asked yet.  The address never changes for the life of the
// process, so two threads that race through the set-up store the same value.
constexpr int kMaxOrdinals = 64;
std::atomic<uintptr_t> g_scratch_addr[kMaxOrdinals];

oo_status report(char* err, size_t cap, oo_status st, const char* fmt, ...) {
    if (err && cap) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(err, cap, fmt, ap);
        va_end(ap);
    }
    return st;
}

}  // namespace

extern "C" OO_API oo_status oo_sort_queries_static(const float* d_x, uint64_t n, uint32_t* d_perm_out, void* cuda_stream,
                                                   char* err_msg, size_t err_cap) {
    if (err_msg && err_cap) err_msg[0] = 0;
    if (n > kMaxQueries)
        return report(err_msg, err_cap, OO_ERR_UNSUPPORTED,
                      "oo_sort_queries_static: n = %llu exceeds OO_SORT_STATIC_MAX_QUERIES = %llu (the built-in scratch is fixed; "
                      "larger batches need oo_reserve + oo_sort_queries)",
                      (unsigned long long)n, (unsigned long long)kMaxQueries);
    if (n && (!d_x || !d_perm_out)) return report(err_msg, err_cap, OO_ERR_INVALID_ARG, "oo_sort_queries_static: NULL argument");

    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return report(err_msg, err_cap, OO_ERR_CUDA, "oo_sort_queries_static: cudaGetDevice: %s", cudaGetErrorString(e));
    // set-up, once per device: the device address of the array on the CURRENT device (this is also what makes the runtime load
    // the module that holds it on that device)
    uintptr_t addr = (dev >= 0 && dev < kMaxOrdinals) ? g_scratch_addr[dev].load(std::memory_order_acquire) : 0;
    if (!addr) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_sort_scratch);
        if (e != cudaSuccess || !p) {
            if (e != cudaSuccess) cudaGetLastError();   // not sticky: leave nothing pending on the caller's thread
            return report(err_msg, err_cap, OO_ERR_CUDA, "oo_sort_queries_static: cudaGetSymbolAddress on device %d: %s", dev,
                          e != cudaSuccess ? cudaGetErrorString(e) : "null address");
        }
        addr = (uintptr_t)p;
        if (dev >= 0 && dev < kMaxOrdinals) g_scratch_addr[dev].store(addr, std::memory_order_release);
    }
    if (n == 0) return OO_OK;   // a call with n = 0 is the way to do the set-up ahead of time

    uint32_t* base = reinterpret_cast<uint32_t*>(addr);
    uint32_t* keys_a = base;
    uint32_t* keys_b = base + kKeyWords;
    uint32_t* idx_a = base + 2 * kKeyWords;
    uint32_t* hist = base + 3 * kKeyWords;
    // The array still holds whatever the previous call left.  Keys, indices and the (digit, tile) table are overwritten for this
    // call's n before they are read; the digit totals are accumulated with atomics and must start at zero — launch_morton_sort
    // clears them with a cudaMemsetAsync on the caller's stream in front of the first kernel.
    const int k = oo::launch_morton_sort(d_x, n, keys_a, keys_b, idx_a, d_perm_out, hist, (cudaStream_t)cuda_stream);
    e = cudaPeekAtLastError();
    if (k < 0 || e != cudaSuccess) {
        if (e != cudaSuccess) cudaGetLastError();
        return report(err_msg, err_cap, OO_ERR_CUDA, "oo_sort_queries_static: launch failed: %s", e != cudaSuccess ? cudaGetErrorString(e) : "launcher error");
    }
    return OO_OK;
}
