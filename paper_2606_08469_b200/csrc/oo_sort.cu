// oo_sort.cu — row a1: Morton pre-sort of the queries (BASELINE.json north_star; not in the paper).
//
// key = 30-bit Morton code of clamp(floor(x*1024), 0, 1023): bit b of q_x -> key bit 3b, q_y -> 3b+1, q_z -> 3b+2 (the
// octant convention of the tree, so sorted order walks the octree depth-first).  Stable LSD radix sort, 3 passes of 10
// bits, hand written: per pass a per-tile histogram kernel (4096 keys per block; the first one also makes the keys), an
// exclusive scan with one block per digit (digit totals come from the histogram kernel's atomics), and a stable scatter in which every warp keeps 512 consecutive keys in registers and ranks
// them 32 at a time with __match_any_sync against warp-private digit counters in shared memory.  Ties keep the original
// order, so the permutation is unique.  9 launches.
#include "oo_device.cuh"
#include "oo_tc_ptx.cuh"

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
template <bool FIRST, int THREADS>
__global__ void __launch_bounds__(THREADS) radix_hist_kernel(const float* __restrict__ x, uint32_t* __restrict__ keys, uint64_t n,
                                                             uint32_t shift, uint32_t n_tiles, uint32_t* __restrict__ hist,
                                                             uint32_t* __restrict__ tot) {
    // THREADS threads share one 4096-key tile: 256 for the sort's later passes (many tiles in flight anyway), 1024 where the
    // pass runs alone in front of the query and a tile's 16 dependent rounds per thread would be the critical path
    constexpr int ITEMS = kTile / THREADS;
    __shared__ uint32_t cnt[kDigits];
    for (int d = threadIdx.x; d < kDigits; d += THREADS) cnt[d] = 0;
    __syncthreads();
    const uint64_t base = (uint64_t)blockIdx.x * kTile;
#pragma unroll 4
    for (int it = 0; it < ITEMS; ++it) {
        const uint64_t i = base + (uint64_t)it * THREADS + threadIdx.x;
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

    for (int d = threadIdx.x; d < kDigits; d += THREADS) {
        const uint32_t c = cnt[d];
        hist[(size_t)d * n_tiles + blockIdx.x] = c;
        if (c) atomicAdd(&tot[d], c);
    }
}

// The counting pass of OO_PRESORT_BIN: as radix_hist_kernel<true> on the top digit, but every thread takes FOUR consecutive
// queries with three 16-byte loads (a 4096-query tile starts 16-byte aligned when x does) and stores their keys with one:
// a quarter of the load/store instructions of the 4-byte version (24.5 -> ? us on 2^22 queries).  1024 threads = one tile.
// stat: the coherence sample of OO_PRESORT_AUTO (this kernel sees the caller's order when a call is binned): distinct depth-4
// cells (top 12 key bits) among the FIRST query of each lane of warp 0, i.e. 32 queries at stride 4.
__global__ void __launch_bounds__(1024) bin_hist_kernel(const float* __restrict__ x, uint32_t* __restrict__ keys, uint64_t n,
                                                        uint32_t n_tiles, uint32_t* __restrict__ hist, uint32_t* __restrict__ tot,
                                                        unsigned long long* stat, uint32_t stat_seq) {
    constexpr uint32_t shift = 30 - kBits;
    __shared__ uint32_t cnt[kDigits];
    cnt[threadIdx.x] = 0;
    __syncthreads();
    const uint64_t i0 = (uint64_t)blockIdx.x * kTile + 4ull * threadIdx.x;
    uint32_t key[4] = {0, 0, 0, 0};
    if (i0 + 3 < n && (((uintptr_t)x) & 15u) == 0) {
        const float4* p = reinterpret_cast<const float4*>(x + 3 * i0);
        const float4 a = __ldg(p), b = __ldg(p + 1), c = __ldg(p + 2);
        const float v[12] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w, c.x, c.y, c.z, c.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int qx = quantise(v[3 * k], 1024.0f, 1023), qy = quantise(v[3 * k + 1], 1024.0f, 1023), qz = quantise(v[3 * k + 2], 1024.0f, 1023);
            key[k] = spread3((uint32_t)qx) | (spread3((uint32_t)qy) << 1) | (spread3((uint32_t)qz) << 2);
            atomicAdd(&cnt[key[k] >> shift], 1u);
        }
        *reinterpret_cast<uint4*>(keys + i0) = make_uint4(key[0], key[1], key[2], key[3]);
    } else {
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (i0 + k < n) {
                key[k] = morton_of(x, i0 + k);
                keys[i0 + k] = key[k];
                atomicAdd(&cnt[key[k] >> shift], 1u);
            }
    }
    if (stat && threadIdx.x < 32 && (uint64_t)blockIdx.x * kTile + 127u < n) {      // warp 0, all of its 128 queries exist
        const uint32_t peers = __match_any_sync(0xffffffffu, key[0] >> 18);
        const bool leader = (uint32_t)(__ffs(peers) - 1) == threadIdx.x;
        const uint32_t distinct = __popc(__ballot_sync(0xffffffffu, leader));
        if (threadIdx.x == 0)      // one slot of the device sample array per block (see stat_sample_warp)
            *(volatile unsigned long long*)(stat + (blockIdx.x % kStatSlots)) =
                ((unsigned long long)(stat_seq & ((1u << kStatSeqBits) - 1u)) << 44) | (1ull << 32) | distinct;
    }
    __syncthreads();
    const uint32_t c = cnt[threadIdx.x];
    hist[(size_t)threadIdx.x * n_tiles + blockIdx.x] = c;
    if (c) atomicAdd(&tot[threadIdx.x], c);
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
        if (pass == 0) radix_hist_kernel<true, kSortThreads><<<n_tiles, kSortThreads, 0, stream>>>(x, kin, n, shift, n_tiles, hist, t);
        else radix_hist_kernel<false, kSortThreads><<<n_tiles, kSortThreads, 0, stream>>>(nullptr, kin, n, shift, n_tiles, hist, t);
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
// OO_PRESORT_BIN (a1'): ONE counting pass on the top kBits bits of the Morton key (the cell at depth 3 plus one bit) that
// moves the QUERIES, not (key, index) pairs.  Same per-tile histogram and scan as above.  The scatter below gives every
// query of its tile a rank inside its digit with a shared-memory atomic (the order inside a bin is whatever the atomics
// return: nothing downstream depends on it, every query is evaluated on its own and inv brings its RGB home), turns the
// ranks into a tile-local sorted order, and copies x, n and wo out of shared memory in that order, consecutive threads on
// consecutive floats, so that global writes are whole runs (all queries of one digit in a tile are consecutive in the
// output).  The tile's three arrays (3 x 48 KB) arrive by three bulk asynchronous copies issued before the ranking starts.
// A direct scatter of 4-byte stores to 1024 open buckets made DRAM read-modify-write partial sectors (measured on B200,
// 2^22 incoherent queries: 313 MB read + 263 MB written, 387 us); staging one array at a time through registers 140 us.
// inv[i] = position of query i in the binned arrays (written in query order, coalesced): unbin_kernel uses it to bring the
// RGB back to the caller's order with coalesced stores.
// =====================================================================================================================
struct BinPayload {
    const float *x, *nrm, *wo, *extra;   // nrm may be nullptr (oo_encode): that array is then skipped
    uint32_t n_extra;
    float *sx, *sn, *sw, *se;
    uint32_t* idx;                       // optional: idx[binned position] = query index (oo_encode stores rows at it)
    const float* disp;                   // optional per-query disparity d^ (full query, OO_LOOKUP_SHIFTED) and its binned copy
    float* sdisp;
};
constexpr int kBinThreads = 512;
constexpr int kBinItems = kTile / kBinThreads;      // 8 queries per thread
constexpr int kBinDPT = kDigits / kBinThreads;      // 2 digits per thread in the scan
// one payload array at a time: 48 KB + destination / source maps + digit tables = 80 KB, so TWO blocks share an SM and one
// block's copy-out overlaps the other's loads and ranking (all three arrays resident: 176 KB, one block per SM, 88 us)
constexpr uint32_t kBinSmemBytes = kTile * 3 * 4 + kTile * 4 + kTile * 2 + kDigits * 4 * 2 + (kBinThreads / 32) * 4 + 16;

__global__ void __launch_bounds__(kBinThreads, 2) bin_scatter_kernel(const uint32_t* __restrict__ keys_in, uint64_t n, uint32_t shift,
                                                                     uint32_t n_tiles, const uint32_t* __restrict__ offsets,
                                                                     const BinPayload B, uint32_t* __restrict__ inv,
                                                                     uint32_t* __restrict__ tot_to_clear) {
    extern __shared__ __align__(128) uint8_t smem_raw[];
    float* s_pay = (float*)smem_raw;                                 // [4096*3] one of x, n, wo of the tile as it lies in memory
    uint32_t* s_dst = (uint32_t*)(s_pay + kTile * 3);                // [4096] global position of each sorted position
    uint32_t* s_cnt = s_dst + kTile;                                 // [1024] digit counts, then tile-local start positions
    uint32_t* s_delta = s_cnt + kDigits;                             // [1024] global position - tile-local sorted position
    uint32_t* s_warp = s_delta + kDigits;                            // [16] warp totals of the digit scan
    uint64_t* s_bar = (uint64_t*)(s_warp + kBinThreads / 32);
    uint16_t* s_src = (uint16_t*)(s_bar + 2);                        // [4096] tile-local source row of each sorted position
    const uint32_t tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint64_t tile_base = (uint64_t)blockIdx.x * kTile;
    const uint32_t tile_n = (uint32_t)(n - tile_base < (uint64_t)kTile ? n - tile_base : (uint64_t)kTile);
    const uint32_t nf = tile_n * 3;
    const float* g[3] = {B.x + tile_base * 3, B.nrm ? B.nrm + tile_base * 3 : nullptr, B.wo + tile_base * 3};
    float* out[3] = {B.sx, B.sn, B.sw};
    const uint32_t bar = smem_u32(s_bar);
    // bulk copies need 16-byte aligned addresses and sizes; anything else takes the plain loop
    const bool bulk = (tile_n & 3u) == 0 && ((((uintptr_t)g[0]) | ((uintptr_t)g[1]) | ((uintptr_t)g[2])) & 15u) == 0;
    if (tid == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // the digit totals of this call have been consumed by the scan: clear them for the next call's counting pass
    if (blockIdx.x == 0 && tot_to_clear)
        for (uint32_t d = tid; d < (uint32_t)kDigits; d += kBinThreads) tot_to_clear[d] = 0;
    // the tile's global start per digit (two strided loads per thread) and its keys are requested first: neither depends on
    // anything, and both were exposed latencies in front of the scan and the ranking (20 % + 15 % of the stall samples)
    uint32_t goff[kBinDPT];
#pragma unroll
    for (int k = 0; k < kBinDPT; ++k) goff[k] = __ldg(offsets + (size_t)(tid * kBinDPT + k) * n_tiles + blockIdx.x);
    uint32_t dig[kBinItems], rank[kBinItems];
#pragma unroll
    for (int it = 0; it < kBinItems; ++it) {
        const uint32_t li = it * kBinThreads + tid;
        dig[it] = li < tile_n ? (__ldg(keys_in + tile_base + li) >> shift) & (kDigits - 1) : 0u;
    }
#pragma unroll
    for (int k = 0; k < kBinDPT; ++k) s_cnt[tid + k * kBinThreads] = 0;
    __syncthreads();
    // load array a of the tile into the payload buffer: one bulk asynchronous copy (completes on the mbarrier), or the plain loop
    auto load = [&](int a) {
        if (bulk) {
            if (tid == 0) {
                mbar_expect_tx(bar, nf * 4u);
                bulk_g2s(smem_u32(s_pay), g[a], nf * 4u, bar);
            }
        } else {
            for (uint32_t f = tid; f < nf; f += kBinThreads) s_pay[f] = __ldg(g[a] + f);
        }
    };
    load(0);
#pragma unroll
    for (int it = 0; it < kBinItems; ++it)
        if (it * kBinThreads + tid < tile_n) rank[it] = atomicAdd(&s_cnt[dig[it]], 1u);
    __syncthreads();
    {   // exclusive scan of the tile's digit counts in digit order; thread t owns digits 2t, 2t+1
        uint32_t cnt[kBinDPT], mine = 0;
#pragma unroll
        for (int k = 0; k < kBinDPT; ++k) {
            cnt[k] = s_cnt[tid * kBinDPT + k];
            mine += cnt[k];
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
        for (int k = 0; k < kBinDPT; ++k) {
            const uint32_t d = tid * kBinDPT + k;
            s_delta[d] = goff[k] - run;
            s_cnt[d] = run;
            run += cnt[k];
        }
    }
    __syncthreads();
#pragma unroll
    for (int it = 0; it < kBinItems; ++it) {
        const uint32_t li = it * kBinThreads + tid;
        if (li < tile_n) {
            const uint32_t lp = s_cnt[dig[it]] + rank[it];
            const uint32_t dst = lp + s_delta[dig[it]];
            s_dst[lp] = dst;
            s_src[lp] = (uint16_t)li;
            inv[tile_base + li] = dst;
        }
    }
    uint32_t phase = 0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (!g[a]) continue;
        if (a > 0) {
            // every thread has read the previous array out of the buffer (generic proxy) before the next bulk copy (async proxy)
            // overwrites it
            fence_async_smem();
            __syncthreads();
            load(a);
        }
        __syncthreads();           // s_dst / s_src (a == 0) or the plain-loop load are visible
        if (bulk) {
            mbar_wait(bar, phase);
            phase ^= 1;
        }
        float* o = out[a];
#pragma unroll 4
        for (uint32_t f = tid; f < nf; f += kBinThreads) {
            const uint32_t p = f / 3u, k = f - 3u * p;
            o[(size_t)s_dst[p] * 3 + k] = s_pay[3u * s_src[p] + k];
        }
    }
    if (B.idx)
        for (uint32_t p = tid; p < tile_n; p += kBinThreads) B.idx[s_dst[p]] = (uint32_t)tile_base + s_src[p];
    if (B.disp)
        for (uint32_t p = tid; p < tile_n; p += kBinThreads) B.sdisp[s_dst[p]] = __ldg(B.disp + tile_base + s_src[p]);
    if (B.n_extra) {   // extras: gathered straight from the tile's own rows, written in runs
        const uint32_t ne = B.n_extra, nfe = tile_n * ne;
        for (uint32_t f = tid; f < nfe; f += kBinThreads) {
            const uint32_t p = f / ne, k = f - ne * p;
            B.se[(size_t)s_dst[p] * ne + k] = __ldg(B.extra + (tile_base + s_src[p]) * ne + k);
        }
    }
}

// out[i][c] = binned[inv[i]][c]: the RGB of the binned queries back in the caller's order, coalesced stores.  A block owns
// 1024 consecutive queries so that everything inside it is 32-bit arithmetic with a compile-time divisor.
constexpr int kUnbinQueries = 1024;
template <int OD>
__global__ void __launch_bounds__(256) unbin_kernel(const float* __restrict__ binned, const uint32_t* __restrict__ inv, uint64_t n,
                                                    uint32_t od_rt, float* __restrict__ out) {
    const uint32_t od = OD ? (uint32_t)OD : od_rt;
    const uint64_t q0 = (uint64_t)blockIdx.x * kUnbinQueries;
    const uint32_t nq = (uint32_t)(n - q0 < (uint64_t)kUnbinQueries ? n - q0 : (uint64_t)kUnbinQueries);
    const uint32_t* iv = inv + q0;
    float* o = out + q0 * od;
#pragma unroll 4
    for (uint32_t f = threadIdx.x; f < nq * od; f += 256) {
        const uint32_t i = f / od, c = f - i * od;
        o[f] = __ldg(binned + (size_t)__ldg(iv + i) * od + c);
    }
}

// bin_tot: kDigits ints that are ZERO on entry (the caller clears them once when it allocates them; the scatter kernel of every
// call clears them again after the scan has consumed them, so no call needs a memset of its own; a call whose scan or scatter
// launch is rejected restores the zeros with a memset before it reports the failure)
int launch_bin_queries(const QueryParams& Q, uint32_t* keys, uint32_t* hist, uint32_t* bin_tot, float* sx, float* sn, float* sw, float* se,
                       uint32_t* inv, uint32_t* idx, float* sdisp, cudaStream_t stream) {
    if (Q.n == 0) return 0;
    static std::atomic<uint64_t> opted{0};
    if (!opt_in_smem(opted, (const void*)bin_scatter_kernel, (int)kBinSmemBytes)) return kLaunchCudaError;
    const uint32_t n_tiles = (uint32_t)((Q.n + kTile - 1) / kTile);
    constexpr uint32_t shift = 30 - kBits;
    bin_hist_kernel<<<n_tiles, 1024, 0, stream>>>(Q.x, keys, Q.n, n_tiles, hist, bin_tot, Q.stat, Q.stat_seq);
    if (cudaPeekAtLastError() != cudaSuccess) return kLaunchCudaError;      // nothing was enqueued: the totals are still zero
    scan_kernel<<<kDigits, kSortThreads, 0, stream>>>(hist, bin_tot, n_tiles);
    bool rejected = cudaPeekAtLastError() != cudaSuccess;
    if (!rejected) {
        const BinPayload B{Q.x, Q.nrm, Q.wo, Q.extra, Q.extra ? Q.n_extra : 0u, sx, sn, sw, se, idx, sdisp ? Q.disparity : nullptr, sdisp};
        bin_scatter_kernel<<<n_tiles, kBinThreads, kBinSmemBytes, stream>>>(keys, Q.n, shift, n_tiles, hist, B, inv, bin_tot);
        rejected = cudaPeekAtLastError() != cudaSuccess;
    }
    if (rejected) {
        // the counting kernel is enqueued and will add this call's counts to bin_tot, but the kernel that clears them is not:
        // clear them behind it, or every later binned call on this context would scan stale totals and scatter out of bounds.
        // (The rejected launch's error stays pending for the caller's report: a call that succeeds does not reset it.)
        cudaMemsetAsync(bin_tot, 0, sizeof(uint32_t) * kDigits, stream);
        return kLaunchCudaError;
    }
    return 3;
}

int launch_unbin(const float* binned, const uint32_t* inv, uint64_t n, uint32_t out_dim, float* out, int, cudaStream_t stream) {
    if (n == 0) return 0;
    const unsigned grid = (unsigned)((n + kUnbinQueries - 1) / kUnbinQueries);
    if (out_dim == 3) unbin_kernel<3><<<grid, 256, 0, stream>>>(binned, inv, n, out_dim, out);
    else unbin_kernel<0><<<grid, 256, 0, stream>>>(binned, inv, n, out_dim, out);
    return 1;
}

}  // namespace oo
