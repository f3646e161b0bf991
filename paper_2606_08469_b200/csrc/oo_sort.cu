// oo_sort.cu — row a1: Morton pre-sort of the queries (BASELINE.json north_star; not in the paper).
//
// key = 30-bit Morton code of clamp(floor(x*1024), 0, 1023): bit b of q_x -> key bit 3b, q_y -> 3b+1, q_z -> 3b+2 (the
// octant convention of the tree, so sorted order walks the octree depth-first).  Stable LSD radix sort, 4 passes of 8
// bits, hand written: per pass a histogram kernel, a single-block exclusive scan, and a stable scatter in which every
// warp owns a contiguous chunk and ranks its items 32 at a time with __match_any_sync against running per-warp digit
// counters in shared memory.  Ties keep the original order, so the permutation is unique.
#include "oo_device.cuh"

namespace oo {

constexpr int kSortThreads = 256;                 // 8 warps per block
constexpr int kChunk = 2048;                      // items per warp

__device__ __forceinline__ uint32_t spread3(uint32_t v) {   // 10 bits -> every third bit
    v = (v | (v << 16)) & 0x030000FFu;
    v = (v | (v << 8)) & 0x0300F00Fu;
    v = (v | (v << 4)) & 0x030C30C3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}

__global__ void morton_key_kernel(const float* __restrict__ x, uint64_t n, uint32_t* __restrict__ keys) {
    const uint64_t t = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x;
    if (t >= n) return;
    const int qx = quantise(__ldg(x + 3 * t), 1024.0f, 1023), qy = quantise(__ldg(x + 3 * t + 1), 1024.0f, 1023),
              qz = quantise(__ldg(x + 3 * t + 2), 1024.0f, 1023);
    keys[t] = spread3((uint32_t)qx) | (spread3((uint32_t)qy) << 1) | (spread3((uint32_t)qz) << 2);
}

// hist[digit * n_chunks + chunk] = number of keys of that digit in the chunk
__global__ void __launch_bounds__(kSortThreads) radix_hist_kernel(const uint32_t* __restrict__ keys, uint64_t n,
                                                                  uint32_t shift, uint32_t n_chunks, uint32_t* __restrict__ hist) {
    __shared__ uint32_t cnt[kSortThreads / 32][256];
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t chunk = blockIdx.x * (kSortThreads / 32) + warp;
    for (int d = lane; d < 256; d += 32) cnt[warp][d] = 0;
    __syncwarp();
    if (chunk < n_chunks) {
        const uint64_t base = (uint64_t)chunk * kChunk;
        for (int it = 0; it < kChunk / 32; ++it) {
            const uint64_t i = base + it * 32 + lane;
            if (i < n) atomicAdd(&cnt[warp][(keys[i] >> shift) & 255u], 1u);
        }
        __syncwarp();
        for (int d = lane; d < 256; d += 32) hist[(size_t)d * n_chunks + chunk] = cnt[warp][d];
    }
}

// in-place exclusive scan of `len` counters by one block
__global__ void __launch_bounds__(1024) scan_kernel(uint32_t* __restrict__ data, uint32_t len) {
    __shared__ uint32_t part[1024];
    const uint32_t per = (len + 1023) / 1024;
    const uint32_t lo = min(threadIdx.x * per, len), hi = min(lo + per, len);
    uint32_t s = 0;
    for (uint32_t i = lo; i < hi; ++i) s += data[i];
    part[threadIdx.x] = s;
    __syncthreads();
    for (uint32_t off = 1; off < 1024; off <<= 1) {
        uint32_t v = threadIdx.x >= off ? part[threadIdx.x - off] : 0;
        __syncthreads();
        part[threadIdx.x] += v;
        __syncthreads();
    }
    uint32_t run = part[threadIdx.x] - s;
    for (uint32_t i = lo; i < hi; ++i) {
        const uint32_t v = data[i];
        data[i] = run;
        run += v;
    }
}

// stable scatter: offsets[digit * n_chunks + chunk] = first output position of that (digit, chunk)
__global__ void __launch_bounds__(kSortThreads) radix_scatter_kernel(const uint32_t* __restrict__ keys_in,
                                                                     const uint32_t* __restrict__ idx_in, uint64_t n,
                                                                     uint32_t shift, uint32_t n_chunks,
                                                                     const uint32_t* __restrict__ offsets,
                                                                     uint32_t* __restrict__ keys_out, uint32_t* __restrict__ idx_out) {
    __shared__ uint32_t pos[kSortThreads / 32][256];
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t chunk = blockIdx.x * (kSortThreads / 32) + warp;
    if (chunk >= n_chunks) return;
    for (int d = lane; d < 256; d += 32) pos[warp][d] = offsets[(size_t)d * n_chunks + chunk];
    __syncwarp();
    const uint64_t base = (uint64_t)chunk * kChunk;
    const uint32_t lt = (1u << lane) - 1u;
    for (int it = 0; it < kChunk / 32; ++it) {
        const uint64_t i = base + it * 32 + lane;
        const bool live = i < n;
        const uint32_t active = __ballot_sync(0xffffffffu, live);
        if (live) {
            const uint32_t key = keys_in[i];
            const uint32_t id = idx_in ? idx_in[i] : (uint32_t)i;
            const uint32_t d = (key >> shift) & 255u;
            const uint32_t peers = __match_any_sync(active, d);
            const uint32_t rank = __popc(peers & lt);
            const uint32_t dst = pos[warp][d] + rank;
            keys_out[dst] = key;
            idx_out[dst] = id;
            __syncwarp(active);
            if (rank == 0) pos[warp][d] += __popc(peers);
        }
        __syncwarp();
    }
}

size_t morton_sort_hist_ints(uint64_t n) {
    const uint64_t chunks = (n + kChunk - 1) / kChunk;
    return (size_t)(chunks ? chunks : 1) * 256;
}

int launch_morton_sort(const float* x, uint64_t n, uint32_t* keys_a, uint32_t* keys_b, uint32_t* idx_a, uint32_t* perm_out,
                       uint32_t* hist, cudaStream_t stream) {
    if (n == 0) return 0;
    int launches = 0;
    morton_key_kernel<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(x, n, keys_a);
    ++launches;
    const uint32_t n_chunks = (uint32_t)((n + kChunk - 1) / kChunk);
    const unsigned blocks = (n_chunks + kSortThreads / 32 - 1) / (kSortThreads / 32);
    uint32_t* kin = keys_a;
    uint32_t* kout = keys_b;
    const uint32_t* iin = nullptr;
    uint32_t* iout = idx_a;
    for (int pass = 0; pass < 4; ++pass) {
        const uint32_t shift = 8 * pass;
        radix_hist_kernel<<<blocks, kSortThreads, 0, stream>>>(kin, n, shift, n_chunks, hist);
        scan_kernel<<<1, 1024, 0, stream>>>(hist, n_chunks * 256);
        radix_scatter_kernel<<<blocks, kSortThreads, 0, stream>>>(kin, iin, n, shift, n_chunks, hist, kout, iout);
        launches += 3;
        uint32_t* t = kin; kin = kout; kout = t;
        iin = iout;
        iout = (iout == idx_a) ? perm_out : idx_a;
    }
    return launches;   // 4 passes: the last scatter wrote perm_out
}

}  // namespace oo
