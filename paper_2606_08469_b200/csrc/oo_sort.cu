// oo_sort.cu — row a1: Morton pre-sort of the queries (BASELINE.json north_star; not in the paper).
//
// key = 30-bit Morton code of clamp(floor(x*1024), 0, 1023): bit b of q_x -> key bit 3b, q_y -> 3b+1, q_z -> 3b+2 (the
// octant convention of the tree, so sorted order walks the octree depth-first).  Stable LSD radix sort, 3 passes of 10
// bits, hand written: per pass a per-tile histogram kernel (4096 keys per block; the first one also makes the keys), an
// exclusive scan with one block per digit (digit totals come from the histogram kernel's atomics), and a stable scatter in which every warp keeps 512 consecutive keys in registers and ranks
// them 32 at a time with __match_any_sync against warp-private digit counters in shared memory.  Ties keep the original
// order, so the permutation is unique.  9 launches.
#include "oo_device.cuh"

namespace oo {

constexpr int kSortThreads = 256;                 // 8 warps per block
constexpr int kItems = 16;                        // keys per thread
constexpr int kWarpChunk = 32 * kItems;           // 512 consecutive keys per warp
constexpr int kTile = kSortThreads * kItems;      // 4096 keys per block
constexpr int kBits = 10;                         // digit width: 30-bit keys = 3 passes
constexpr int kDigits = 1 << kBits;
constexpr int kPasses = 3;
constexpr int kDPT = kDigits / kSortThreads;      // digits per thread in the per-digit loops

__device__ __forceinline__ uint32_t spread3(uint32_t v) {   // 10 bits -> every third bit
    v = (v | (v << 16)) & 0x030000FFu;
    v = (v | (v << 8)) & 0x0300F00Fu;
    v = (v | (v << 4)) & 0x030C30C3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}

__device__ __forceinline__ uint32_t morton_of(const float* __restrict__ x, uint64_t i) {
    const int qx = quantise(__ldg(x + 3 * i), 1024.0f, 1023), qy = quantise(__ldg(x + 3 * i + 1), 1024.0f, 1023),
              qz = quantise(__ldg(x + 3 * i + 2), 1024.0f, 1023);
    return spread3((uint32_t)qx) | (spread3((uint32_t)qy) << 1) | (spread3((uint32_t)qz) << 2);
}

// hist[digit * n_tiles + tile] = number of keys of that digit in the tile; tot[digit] += the same (digit totals of
// the pass).  FIRST: the keys are made here (from x) and written out, so there is no separate key kernel.
template <bool FIRST>
__global__ void __launch_bounds__(kSortThreads) radix_hist_kernel(const float* __restrict__ x, uint32_t* __restrict__ keys,
                                                                  uint64_t n, uint32_t shift, uint32_t n_tiles,
                                                                  uint32_t* __restrict__ hist, uint32_t* __restrict__ tot) {
    __shared__ uint32_t cnt[kDigits];
#pragma unroll
    for (int k = 0; k < kDPT; ++k) cnt[threadIdx.x + k * kSortThreads] = 0;
    __syncthreads();
    const uint64_t base = (uint64_t)blockIdx.x * kTile;
#pragma unroll 4
    for (int it = 0; it < kItems; ++it) {
        const uint64_t i = base + (uint64_t)it * kSortThreads + threadIdx.x;
        if (i < n) {
            uint32_t key;
            if constexpr (FIRST) {
                key = morton_of(x, i);
                keys[i] = key;
            } else {
                key = keys[i];
            }
            atomicAdd(&cnt[(key >> shift) & (kDigits - 1)], 1u);
        }
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kDPT; ++k) {
        const uint32_t d = threadIdx.x + k * kSortThreads, c = cnt[d];
        hist[(size_t)d * n_tiles + blockIdx.x] = c;
        if (c) atomicAdd(&tot[d], c);
    }
}

// Exclusive scan of hist in (digit, tile) order, in place: block d scans row d and adds the total of all smaller digits.
__global__ void __launch_bounds__(kSortThreads) scan_kernel(uint32_t* __restrict__ hist, const uint32_t* __restrict__ tot,
                                                            uint32_t n_tiles) {
    __shared__ uint32_t red[kSortThreads / 32];
    __shared__ uint32_t part[kSortThreads];
    const uint32_t d = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t s = 0;
    for (uint32_t k = threadIdx.x; k < d; k += kSortThreads) s += tot[k];
#pragma unroll
    for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) red[warp] = s;
    uint32_t* row = hist + (size_t)d * n_tiles;
    const uint32_t per = (n_tiles + kSortThreads - 1) / kSortThreads;
    const uint32_t lo = min(threadIdx.x * per, n_tiles), hi = min(lo + per, n_tiles);
    uint32_t mine = 0;
    for (uint32_t i = lo; i < hi; ++i) mine += row[i];
    part[threadIdx.x] = mine;
    __syncthreads();
    uint32_t base = 0;
#pragma unroll
    for (int w = 0; w < kSortThreads / 32; ++w) base += red[w];
    for (uint32_t off = 1; off < kSortThreads; off <<= 1) {
        const uint32_t v = threadIdx.x >= off ? part[threadIdx.x - off] : 0;
        __syncthreads();
        part[threadIdx.x] += v;
        __syncthreads();
    }
    uint32_t run = base + part[threadIdx.x] - mine;
    for (uint32_t i = lo; i < hi; ++i) {
        const uint32_t v = row[i];
        row[i] = run;
        run += v;
    }
}

// Stable scatter of one tile: offsets[digit * n_tiles + tile] = first output position of that (digit, tile).  Warp w owns
// the 512 consecutive keys [tile*4096 + 512 w, +512) and keeps them in registers: it ranks them 32 at a time with
// __match_any_sync against its private digit counters (rank among equal digits in index order), the block then turns the
// counters into per-warp start positions, and every key goes to start + rank.
__global__ void __launch_bounds__(kSortThreads) radix_scatter_kernel(const uint32_t* __restrict__ keys_in,
                                                                     const uint32_t* __restrict__ idx_in, uint64_t n,
                                                                     uint32_t shift, uint32_t n_tiles,
                                                                     const uint32_t* __restrict__ offsets,
                                                                     uint32_t* __restrict__ keys_out, uint32_t* __restrict__ idx_out) {
    __shared__ uint32_t pos[kSortThreads / 32][kDigits];
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int w = 0; w < kSortThreads / 32; ++w)
#pragma unroll
        for (int k = 0; k < kDPT; ++k) pos[w][threadIdx.x + k * kSortThreads] = 0;
    __syncthreads();
    const uint64_t base = (uint64_t)blockIdx.x * kTile + (uint64_t)warp * kWarpChunk;
    const uint32_t lt = (1u << lane) - 1u;
    uint32_t key[kItems], rank[kItems];
#pragma unroll
    for (int it = 0; it < kItems; ++it) {
        const uint64_t i = base + it * 32 + lane;
        key[it] = i < n ? keys_in[i] : 0xFFFFFFFFu;
    }
#pragma unroll
    for (int it = 0; it < kItems; ++it) {
        const uint64_t i = base + it * 32 + lane;
        const bool live = i < n;
        const uint32_t active = __ballot_sync(0xffffffffu, live);
        if (live) {
            const uint32_t d = (key[it] >> shift) & (kDigits - 1);
            const uint32_t peers = __match_any_sync(active, d);
            const uint32_t r = __popc(peers & lt);
            rank[it] = pos[warp][d] + r;
            __syncwarp(active);
            if (r == 0) pos[warp][d] += __popc(peers);
        }
        __syncwarp();
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kDPT; ++k) {   // per digit: tile offset, then the warps in order
        const uint32_t d = threadIdx.x + k * kSortThreads;
        uint32_t run = offsets[(size_t)d * n_tiles + blockIdx.x];
#pragma unroll
        for (int w = 0; w < kSortThreads / 32; ++w) {
            const uint32_t c = pos[w][d];
            pos[w][d] = run;
            run += c;
        }
    }
    __syncthreads();
#pragma unroll
    for (int it = 0; it < kItems; ++it) {
        const uint64_t i = base + it * 32 + lane;
        if (i < n) {
            const uint32_t dst = pos[warp][(key[it] >> shift) & (kDigits - 1)] + rank[it];
            keys_out[dst] = key[it];
            idx_out[dst] = idx_in ? idx_in[i] : (uint32_t)i;
        }
    }
}

// scratch ints: the (digit, tile) table + one row of digit totals per pass
size_t morton_sort_hist_ints(uint64_t n) {
    const uint64_t tiles = (n + kTile - 1) / kTile;
    return (size_t)(tiles ? tiles : 1) * kDigits + (size_t)kPasses * kDigits;
}

int launch_morton_sort(const float* x, uint64_t n, uint32_t* keys_a, uint32_t* keys_b, uint32_t* idx_a, uint32_t* perm_out,
                       uint32_t* hist, cudaStream_t stream) {
    if (n == 0) return 0;
    int launches = 0;
    const uint32_t n_tiles = (uint32_t)((n + kTile - 1) / kTile);
    uint32_t* tot = hist + (size_t)n_tiles * kDigits;
    cudaMemsetAsync(tot, 0, sizeof(uint32_t) * kPasses * kDigits, stream);
    uint32_t* kin = keys_a;
    uint32_t* kout = keys_b;
    const uint32_t* iin = nullptr;
    // three passes: the index arrays alternate so that the last scatter writes perm_out
    uint32_t* iout = perm_out;
    for (int pass = 0; pass < kPasses; ++pass) {
        const uint32_t shift = kBits * pass;
        uint32_t* t = tot + pass * kDigits;
        if (pass == 0) radix_hist_kernel<true><<<n_tiles, kSortThreads, 0, stream>>>(x, kin, n, shift, n_tiles, hist, t);
        else radix_hist_kernel<false><<<n_tiles, kSortThreads, 0, stream>>>(nullptr, kin, n, shift, n_tiles, hist, t);
        scan_kernel<<<kDigits, kSortThreads, 0, stream>>>(hist, t, n_tiles);
        radix_scatter_kernel<<<n_tiles, kSortThreads, 0, stream>>>(kin, iin, n, shift, n_tiles, hist, kout, iout);
        launches += 3;
        uint32_t* tk = kin; kin = kout; kout = tk;
        iin = iout;
        iout = (iout == idx_a) ? perm_out : idx_a;
    }
    return launches;   // odd number of passes starting at perm_out: the last scatter wrote perm_out
}

// =====================================================================================================================
// OO_PRESORT_BIN (a1'): ONE stable radix pass on the top kBits bits of the Morton key (the cell at depth 3 plus one bit)
// that moves the QUERIES, not (key, index) pairs.  Same per-tile histogram and scan as above; the scatter below ranks
// its tile exactly like radix_scatter_kernel, then sorts the tile locally in shared memory so that global writes are runs
// (all queries of one digit in a tile are consecutive in the output): x, n and wo are staged through a 48 KB buffer, one
// array at a time, read back in sorted order and written with consecutive threads on consecutive floats.  A direct
// scatter of 4-byte stores to 1024 open buckets made DRAM read-modify-write partial sectors (measured on B200, 2^22
// incoherent queries: 313 MB read + 263 MB written, 387 us; this version moves the algorithmic ~320 MB).
// inv[i] = position of query i in the binned arrays (written in query order, coalesced): unbin_kernel uses it to bring the
// RGB back to the caller's order with coalesced stores.
// =====================================================================================================================
struct BinPayload {
    const float *x, *nrm, *wo, *extra;
    uint32_t n_extra;
    float *sx, *sn, *sw, *se;
};
constexpr uint32_t kBinSmemBytes = (kSortThreads / 32) * kDigits * 4 + kTile * 4 + kTile * 2 + kDigits * 4 + kTile * 3 * 4 + 64;

__global__ void __launch_bounds__(kSortThreads) bin_scatter_kernel(const uint32_t* __restrict__ keys_in, uint64_t n, uint32_t shift,
                                                                   uint32_t n_tiles, const uint32_t* __restrict__ offsets,
                                                                   const BinPayload B, uint32_t* __restrict__ inv) {
    extern __shared__ __align__(16) uint32_t sm[];
    uint32_t(*pos)[kDigits] = (uint32_t(*)[kDigits])sm;              // [8][1024] per-warp digit counters, then start positions
    uint32_t* s_src = sm + (kSortThreads / 32) * kDigits;            // [4096] tile-local source index at each sorted position
    uint32_t* s_delta = s_src + kTile;                               // [1024] global position - tile-local sorted position
    float* s_pay = (float*)(s_delta + kDigits);                      // [4096*3] one staged array
    uint16_t* s_dig = (uint16_t*)(s_pay + kTile * 3);                // [4096] digit at each sorted position
    uint32_t* s_warp = (uint32_t*)(s_dig + kTile);                   // [8] warp totals of the digit scan
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int w = 0; w < kSortThreads / 32; ++w)
#pragma unroll
        for (int k = 0; k < kDPT; ++k) pos[w][threadIdx.x + k * kSortThreads] = 0;
    __syncthreads();
    const uint64_t tile_base = (uint64_t)blockIdx.x * kTile;
    const uint32_t tile_n = (uint32_t)(n - tile_base < (uint64_t)kTile ? n - tile_base : (uint64_t)kTile);
    const uint32_t wbase = warp * kWarpChunk;
    const uint32_t lt = (1u << lane) - 1u;
    uint32_t dig[kItems], rank[kItems];
#pragma unroll
    for (int it = 0; it < kItems; ++it) {
        const uint32_t li = wbase + it * 32 + lane;
        dig[it] = li < tile_n ? (keys_in[tile_base + li] >> shift) & (kDigits - 1) : 0u;
    }
#pragma unroll
    for (int it = 0; it < kItems; ++it) {
        const bool live = wbase + it * 32 + lane < tile_n;
        const uint32_t active = __ballot_sync(0xffffffffu, live);
        if (live) {
            const uint32_t peers = __match_any_sync(active, dig[it]);
            const uint32_t r = __popc(peers & lt);
            rank[it] = pos[warp][dig[it]] + r;
            __syncwarp(active);
            if (r == 0) pos[warp][dig[it]] += __popc(peers);
        }
        __syncwarp();
    }
    __syncthreads();
    {   // exclusive scan of the tile's digit counts in digit order; thread t owns digits 4t .. 4t+3
        uint32_t cnt[kDPT], mine = 0;
#pragma unroll
        for (int k = 0; k < kDPT; ++k) {
            uint32_t c = 0;
#pragma unroll
            for (int w = 0; w < kSortThreads / 32; ++w) c += pos[w][threadIdx.x * kDPT + k];
            cnt[k] = c;
            mine += c;
        }
        uint32_t incl = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= (uint32_t)o) incl += v;
        }
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        uint32_t run = incl - mine;
        for (uint32_t w = 0; w < warp; ++w) run += s_warp[w];
#pragma unroll
        for (int k = 0; k < kDPT; ++k) {
            const uint32_t d = threadIdx.x * kDPT + k;
            s_delta[d] = offsets[(size_t)d * n_tiles + blockIdx.x] - run;
            uint32_t r = run;
#pragma unroll
            for (int w = 0; w < kSortThreads / 32; ++w) {
                const uint32_t c = pos[w][d];
                pos[w][d] = r;
                r += c;
            }
            run += cnt[k];
        }
    }
    __syncthreads();
#pragma unroll
    for (int it = 0; it < kItems; ++it) {
        const uint32_t li = wbase + it * 32 + lane;
        if (li < tile_n) {
            const uint32_t lp = pos[warp][dig[it]] + rank[it];
            s_src[lp] = li;
            s_dig[lp] = (uint16_t)dig[it];
            inv[tile_base + li] = lp + s_delta[dig[it]];
        }
    }
    __syncthreads();
    const float* src[3] = {B.x, B.nrm, B.wo};
    float* dst[3] = {B.sx, B.sn, B.sw};
    const uint32_t nf = tile_n * 3;
#pragma unroll 1
    for (int a = 0; a < 3; ++a) {
        const float* g = src[a] + tile_base * 3;
        for (uint32_t f = threadIdx.x; f < nf; f += kSortThreads) s_pay[f] = __ldg(g + f);
        __syncthreads();
        float* o = dst[a];
        for (uint32_t f = threadIdx.x; f < nf; f += kSortThreads) {
            const uint32_t lp = f / 3u, k = f - 3u * lp;
            o[(size_t)(lp + s_delta[s_dig[lp]]) * 3 + k] = s_pay[3u * s_src[lp] + k];
        }
        __syncthreads();
    }
    if (B.n_extra) {   // extras: gathered straight from the tile's own rows (L1-resident), written in runs
        const uint32_t ne = B.n_extra, nfe = tile_n * ne;
        for (uint32_t f = threadIdx.x; f < nfe; f += kSortThreads) {
            const uint32_t lp = f / ne, k = f - ne * lp;
            B.se[(size_t)(lp + s_delta[s_dig[lp]]) * ne + k] = __ldg(B.extra + (tile_base + s_src[lp]) * ne + k);
        }
    }
}

// out[i][c] = binned[inv[i]][c]: the RGB of the binned queries back in the caller's order, coalesced stores
__global__ void __launch_bounds__(256) unbin_kernel(const float* __restrict__ binned, const uint32_t* __restrict__ inv, uint64_t n,
                                                    uint32_t od, float* __restrict__ out) {
    const uint64_t total = n * od;
    for (uint64_t f = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; f < total; f += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t i = f / od;
        const uint32_t c = (uint32_t)(f - i * od);
        out[f] = __ldg(binned + (size_t)__ldg(inv + i) * od + c);
    }
}

int launch_bin_queries(const QueryParams& Q, uint32_t* keys, uint32_t* hist, float* sx, float* sn, float* sw, float* se,
                       uint32_t* inv, cudaStream_t stream) {
    if (Q.n == 0) return 0;
    static bool attr = false;
    if (!attr) {
        cudaFuncSetAttribute(bin_scatter_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kBinSmemBytes);
        attr = true;
    }
    const uint32_t n_tiles = (uint32_t)((Q.n + kTile - 1) / kTile);
    uint32_t* tot = hist + (size_t)n_tiles * kDigits;
    cudaMemsetAsync(tot, 0, sizeof(uint32_t) * kDigits, stream);
    constexpr uint32_t shift = 30 - kBits;
    radix_hist_kernel<true><<<n_tiles, kSortThreads, 0, stream>>>(Q.x, keys, Q.n, shift, n_tiles, hist, tot);
    scan_kernel<<<kDigits, kSortThreads, 0, stream>>>(hist, tot, n_tiles);
    const BinPayload B{Q.x, Q.nrm, Q.wo, Q.extra, Q.n_extra, sx, sn, sw, se};
    bin_scatter_kernel<<<n_tiles, kSortThreads, kBinSmemBytes, stream>>>(keys, Q.n, shift, n_tiles, hist, B, inv);
    return 3;
}

int launch_unbin(const float* binned, const uint32_t* inv, uint64_t n, uint32_t out_dim, float* out, int n_sms, cudaStream_t stream) {
    if (n == 0) return 0;
    const uint64_t blocks = (n * out_dim + 255) / 256;
    const uint64_t cap = (uint64_t)n_sms * 16;
    unbin_kernel<<<(unsigned)(blocks < cap ? blocks : cap), 256, 0, stream>>>(binned, inv, n, out_dim, out);
    return 1;
}

}  // namespace oo
