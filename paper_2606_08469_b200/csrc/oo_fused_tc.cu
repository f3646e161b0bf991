// oo_fused_tc.cu — fused encode + MLP on 5th-generation tensor cores (OO_PATH_FUSED_TC).
//
// One warpgroup (128 threads) owns a tile of 128 queries end to end; thread t is query row t and TMEM lane t.
//   gather (registers, fp32)  ->  fp16 row into the A tile in shared memory (UMMA K-major canonical layout)
//   -> tcgen05.mma.kind::f16 M=128 N=64 K=16 steps issued by ONE thread, accumulator in TMEM (64 fp32 columns)
//   -> tcgen05.commit -> mbarrier -> every thread tcgen05.ld's its own row -> ReLU -> fp16 -> back into the A tile
//   -> next layer ... -> output layer (N=16) -> exp -> RGB.
// Features and activations never touch HBM.  A block holds two such warpgroups sharing the descent tables and the weight
// image; several blocks per SM overlap the memory-bound gather of one tile with the tensor/epilogue phase of others.
//
// Shared-memory operand layout (no swizzle, K-major): 16-byte chunk c (8 consecutive K) of row r is at
//   base + c * (rows*16) + r*16,  i.e. core matrices (8 rows x 16 B) are contiguous, SBO = 128 B, LBO = rows*16 B.
// A warp writing chunk c of its 32 rows therefore writes 512 contiguous bytes (no bank conflicts).
#include <cstdio>
#include <cstdlib>

#include "oo_device.cuh"
#include "oo_tc_ptx.cuh"

namespace oo {

namespace {

constexpr int kTileRows = 128;

}  // namespace

// The tensor-core weight image (built by oo_upload_mlp, MlpParams::image_tc): per layer chunk-major [K/8][N][8] halves:
//   layer 0: K = k1, N = 64;  layers 1..H-1: K = 64, N = 64;  output: K = 64, N = 16 (rows >= out_dim zero).
//
// ONE persistent block per SM with NWG warpgroups: the descent tables and the weight image are staged once per SM and
// shared; every warpgroup owns an A tile, 64 TMEM columns, an mbarrier and a query staging buffer into which the NEXT
// tile's (x, n, wo, extra, index) are prefetched with cp.async while the current tile is gathered and decoded, so the
// cold HBM latency of the query stream is hidden behind the previous tile.
template <int L, int F, bool F32, int NWG, int MINB, bool DBG>
__global__ void __launch_bounds__(NWG * 128, MINB) fused_tc_kernel(const __grid_constant__ TreeParams T,
                                                                const __grid_constant__ MlpParams M,
                                                                const __grid_constant__ QueryParams Q,
                                                                float* __restrict__ rgb, uint32_t n_tiles) {
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t dense_bytes = (T.dense_ints * 4 + 127) & ~127u;
    const uint32_t a_chunks = (M.k1 > 64 ? M.k1 : 64) / 8;
    const uint32_t a_bytes = a_chunks * kTileRows * 16;
    const uint32_t q_words = 10 + Q.n_extra;                         // x3 n3 wo3 index extras, each [128] words
    const uint32_t q_bytes = q_words * kTileRows * 4;
    int32_t* s_dense = (int32_t*)smem;
    uint8_t* s_w = smem + dense_bytes;
    uint8_t* s_tiles = s_w + ((M.image_tc_bytes + 127) & ~127u);
    uint64_t* s_bar = (uint64_t*)(s_tiles + NWG * (a_bytes + q_bytes));
    uint32_t* s_tmem = (uint32_t*)(s_bar + NWG);

    const uint32_t wg = threadIdx.x >> 7, row = threadIdx.x & 127, warp = threadIdx.x >> 5;
    {
        const uint4* s = (const uint4*)T.dense;
        uint4* d = (uint4*)s_dense;
        for (uint32_t i = threadIdx.x; i < T.dense_ints / 4; i += NWG * 128) d[i] = __ldg(s + i);
        s = (const uint4*)M.image_tc;
        d = (uint4*)s_w;
        for (uint32_t i = threadIdx.x; i < M.image_tc_bytes / 16; i += NWG * 128) d[i] = __ldg(s + i);
    }
    if (threadIdx.x < NWG) mbar_init(smem_u32(&s_bar[threadIdx.x]), 1);
    if (threadIdx.x == 0) asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    constexpr uint32_t kTmemCols = NWG * 64 <= 64 ? 64 : NWG * 64 <= 128 ? 128 : NWG * 64 <= 256 ? 256 : 512;
    if (warp == 0) {
        tmem_alloc(smem_u32(s_tmem), kTmemCols);
        tmem_relinquish();
    }
    fence_async_smem();          // the weight image was written with generic stores and is read by the tensor core
    fence_before_sync();
    __syncthreads();
    fence_after_sync();
    const uint32_t tmem_d = *s_tmem + wg * 64;                       // this warpgroup's 64 accumulator columns
    const uint32_t tmem_lane = tmem_d + ((row & ~31u) << 16);        // this warp's 32 lanes
    uint8_t* s_a = s_tiles + wg * (a_bytes + q_bytes);
    float* s_q = (float*)(s_a + a_bytes) + row;                      // word k of my row: s_q[k * 128]
    const uint32_t a_addr = smem_u32(s_a), w_addr = smem_u32(s_w), bar = smem_u32(&s_bar[wg]), q_addr = smem_u32(s_q);
    const uint32_t a_lbo = kTileRows * 16;                           // 2048 B between K chunks of the A tile
    uint32_t phase = 0;
    const bool leader_warp = row < 32;                               // warp 0 of the warpgroup issues the MMAs (one elected lane)
    constexpr uint32_t idesc_h = instr_desc(128, 64), idesc_o = instr_desc(128, 16);
    const uint32_t tile_stride = gridDim.x * NWG;

    // prefetch one tile's query rows into the staging buffer: 4-byte cp.async per word (rows are 12-byte packed)
    auto prefetch = [&](uint32_t tile) {
        const uint64_t t = (uint64_t)tile * kTileRows + row;
        const uint64_t tt = t < Q.n ? t : Q.n - 1;
        const uint32_t qi = Q.perm ? __ldg(Q.perm + tt) : (uint32_t)tt;
        const float* px = Q.x + (size_t)qi * 3;
        const float* pn = Q.nrm + (size_t)qi * 3;
        const float* pw = Q.wo + (size_t)qi * 3;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            cp_async4(q_addr + (k) * 512, px + k);
            cp_async4(q_addr + (3 + k) * 512, pn + k);
            cp_async4(q_addr + (6 + k) * 512, pw + k);
        }
        for (uint32_t k = 0; k < Q.n_extra; ++k) cp_async4(q_addr + (10 + k) * 512, Q.extra + (size_t)qi * Q.n_extra + k);
        s_q[9 * 128] = __uint_as_float(qi);
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    uint32_t tile = blockIdx.x * NWG + wg;
    if (tile < n_tiles) prefetch(tile);
#ifdef OO_PROFILE_PHASES
    long long t_gather = 0, t_mlp = 0, t_wait = 0, t_q = 0; int n_done = 0;
    const long long t_begin = clock64();
#endif
    for (; tile < n_tiles; tile += tile_stride) {
        // ------------------------------------------------------------------ this tile's query (prefetched into s_q)
        float x[3], w[3];
        const bool valid = (uint64_t)tile * kTileRows + row < Q.n;
#ifdef OO_PROFILE_PHASES
        const long long t0 = clock64();
#endif
        asm volatile("cp.async.wait_group 0;" ::: "memory");
#ifdef OO_PROFILE_PHASES
        const long long t0b = clock64();
#endif
#pragma unroll
        for (int k = 0; k < 3; ++k) { x[k] = s_q[k * 128]; w[k] = s_q[(6 + k) * 128]; }
        // ------------------------------------------------------------------ gather: one query per thread
        Encoded<L, F, F32> e;
        locate<L, F, F32>(T, s_dense, x, w, e);
        uint64_t dbg_row = 0;
        if constexpr (DBG) {             // where this query's index rows go: its own index (binned queries: out_idx's)
            const uint64_t t = (uint64_t)tile * kTileRows + row;
            dbg_row = Q.out_idx ? Q.out_idx[t < Q.n ? t : Q.n - 1] : __float_as_uint(s_q[9 * 128]);
        }
        const auto dbg = make_dbg<DBG>(Q, L, dbg_row, valid);
        uint8_t* a_row = s_a + row * 16;
        constexpr int NB = (F * (F32 ? 4 : 2) == 16) ? (L < 4 ? L : 4) : (F * (F32 ? 4 : 2) == 32 ? 2 : 1);   // levels per load batch (<= 64 data registers)
#pragma unroll
        for (int l0 = 0; l0 < L; l0 += NB) {
            float h[NB][F];
            if (l0 + NB <= L) {
                gather_levels<F, F32, NB>(&T.lv[l0], &e.slot[l0], e.uv, h, dbg, l0);
            } else {     // ragged last batch: one level at a time
#pragma unroll
                for (int b = 0; b < NB; ++b)
                    if (l0 + b < L) {
                        gather_level<F, F32>(T.lv[l0 + b], e.slot[l0 + b], e.uv, h[b], dbg, l0 + b);
                    }
            }
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const int l = l0 + b;
                if (l >= L) break;
                if constexpr (F % 8 == 0) {
#pragma unroll
                    for (int v = 0; v < F / 8; ++v)
                        *(uint4*)(a_row + (l * (F / 8) + v) * a_lbo) =
                            make_uint4(pack_half2(h[b][8 * v], h[b][8 * v + 1]), pack_half2(h[b][8 * v + 2], h[b][8 * v + 3]),
                                       pack_half2(h[b][8 * v + 4], h[b][8 * v + 5]), pack_half2(h[b][8 * v + 6], h[b][8 * v + 7]));
                } else {   // F == 4: half a chunk
                    *(uint2*)(a_row + ((l * 4) / 8) * a_lbo + ((l * 4) % 8) * 2) = make_uint2(pack_half2(h[b][0], h[b][1]), pack_half2(h[b][2], h[b][3]));
                }
            }
        }
        uint32_t qi;
        {   // attributes + zero padding up to k1 (n, extras and the query index are read from the staging buffer only now,
            // so that they do not occupy registers during the gather)
            float v[24];
#pragma unroll
            for (int k = 0; k < 24; ++k) v[k] = 0.0f;
            constexpr int lead = (L * F) % 8;            // 0 or 4: position of n inside its chunk
#pragma unroll
            for (int k = 0; k < 3; ++k) { v[lead + k] = s_q[(3 + k) * 128]; v[lead + 3 + k] = w[k]; }
#pragma unroll
            for (int k = 0; k < OO_MAX_EXTRA; ++k)
                if ((uint32_t)k < Q.n_extra) v[lead + 6 + k] = s_q[(10 + k) * 128];
            qi = __float_as_uint(s_q[9 * 128]);
            constexpr int c0 = (L * F) / 8;
            const uint32_t c_end = M.k1 / 8;
            if constexpr (lead == 0) {
                *(uint4*)(a_row + c0 * a_lbo) = make_uint4(pack_half2(v[0], v[1]), pack_half2(v[2], v[3]), pack_half2(v[4], v[5]), pack_half2(v[6], v[7]));
            } else {
                *(uint2*)(a_row + c0 * a_lbo + 8) = make_uint2(pack_half2(v[4], v[5]), pack_half2(v[6], v[7]));
            }
            if (c0 + 1 < c_end)
                *(uint4*)(a_row + (c0 + 1) * a_lbo) = make_uint4(pack_half2(v[8], v[9]), pack_half2(v[10], v[11]), pack_half2(v[12], v[13]), pack_half2(v[14], v[15]));
            if (c0 + 2 < c_end)
                *(uint4*)(a_row + (c0 + 2) * a_lbo) = make_uint4(pack_half2(v[16], v[17]), pack_half2(v[18], v[19]), pack_half2(v[20], v[21]), pack_half2(v[22], v[23]));
        }
        // the staging buffer is free again: prefetch the next tile's queries behind this tile's MLP phase
        if (tile + tile_stride < n_tiles) prefetch(tile + tile_stride);
#ifdef OO_PROFILE_PHASES
        const long long t1 = clock64();
        long long tw = 0;
#endif
        // ------------------------------------------------------------------ hidden layers
        uint32_t w_off = 0;
        for (uint32_t layer = 0; layer < M.n_hidden; ++layer) {
            const uint32_t kt_n = (layer == 0 ? M.k1 : 64u) >> 4;
            fence_async_smem();          // my A-tile stores -> visible to the tensor core
            fence_before_sync();
            named_bar(1 + wg, 128);
            if (leader_warp) {
                fence_after_sync();
                umma_group<8>(tmem_d, smem_desc(a_addr, a_lbo, 128), (2 * a_lbo) >> 4, smem_desc(w_addr + w_off, 1024, 128), 2048 >> 4, idesc_h,
                              kt_n, bar);
            }
            w_off += kt_n * 2 * 1024;
#ifdef OO_PROFILE_PHASES
            const long long tw0 = clock64();
            mbar_wait(bar, phase);
            tw += clock64() - tw0;
#else
            mbar_wait(bar, phase);
#endif
            phase ^= 1;
            fence_after_sync();
            // epilogue: my row of D -> ReLU -> fp16 -> my row of the next A tile
#pragma unroll
            for (int half = 0; half < 2; ++half) {
                uint32_t r[32];
                tmem_ld32(tmem_lane + half * 32, r);
                tmem_wait_ld();
#pragma unroll
                for (int c = 0; c < 4; ++c)
                    *(uint4*)(a_row + (half * 4 + c) * a_lbo) =
                        make_uint4(pack_half2_relu(__uint_as_float(r[8 * c]), __uint_as_float(r[8 * c + 1])),
                                   pack_half2_relu(__uint_as_float(r[8 * c + 2]), __uint_as_float(r[8 * c + 3])),
                                   pack_half2_relu(__uint_as_float(r[8 * c + 4]), __uint_as_float(r[8 * c + 5])),
                                   pack_half2_relu(__uint_as_float(r[8 * c + 6]), __uint_as_float(r[8 * c + 7])));
            }
        }
        // ------------------------------------------------------------------ output layer (N = 16, K = 64)
        fence_async_smem();
        fence_before_sync();
        named_bar(1 + wg, 128);
        if (leader_warp) {
            fence_after_sync();
            umma_group<4>(tmem_d, smem_desc(a_addr, a_lbo, 128), (2 * a_lbo) >> 4, smem_desc(w_addr + w_off, 256, 128), 512 >> 4, idesc_o, 4u, bar);
        }
        mbar_wait(bar, phase);
        phase ^= 1;
        fence_after_sync();
        uint32_t o[4];
        tmem_ld4(tmem_lane, o);
        tmem_wait_ld();
        if (valid) {
#pragma unroll
            for (uint32_t c = 0; c < 4; ++c)
                if (c < M.out_dim) {
                    const float z = __uint_as_float(o[c]);
                    rgb[(size_t)qi * M.out_dim + c] = M.out_act == OO_ACT_EXP ? fast_exp(z) : z;
                }
        }
        // the next tile's MMA overwrites D: order every thread's TMEM loads before the next barrier
        fence_before_sync();
#ifdef OO_PROFILE_PHASES
        const long long t2 = clock64();
        t_q += t0b - t0; t_gather += t1 - t0b; t_mlp += t2 - t1; t_wait += tw; ++n_done;
#endif
    }
#ifdef OO_PROFILE_PHASES
    if (blockIdx.x == 3 && (threadIdx.x & 31) == 0 && n_done)
        printf("wg %u warp %u tiles %d total %lld qwait %lld gather %lld mlp %lld (mma-wait %lld) per tile\n", wg, warp & 3, n_done,
               (clock64() - t_begin) / n_done, t_q / n_done, t_gather / n_done, t_mlp / n_done, t_wait / n_done);
#endif
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();
    if (warp == 0) tmem_dealloc(*s_tmem, kTmemCols);
}

// ---------------------------------------------------------------------------------------------------------------------
#define OO_TC_SHAPES(X)                                                        \
    X(1, 8, false) X(2, 8, false) X(3, 8, false) X(4, 8, false) X(5, 8, false) \
    X(2, 16, false) X(3, 16, false) X(4, 16, false) X(5, 16, false)            \
    X(2, 4, true) X(4, 4, true)

bool tc_shape_supported(uint32_t L, uint32_t F, bool f32) {
#define X(l, f, t) if (L == l && F == f && f32 == t) return true;
    OO_TC_SHAPES(X)
#undef X
    return false;
}

template <int NWG, int MINB, bool DBG>
static int launch_tc_nwg(const TreeParams& T, const MlpParams& M, const QueryParams& Q, float* rgb, int n_sms, uint32_t smem,
                         cudaStream_t stream) {
    const uint64_t n_tiles = (Q.n + kTileRows - 1) / kTileRows;
    const uint64_t blocks = (n_tiles + NWG - 1) / NWG;
    const unsigned grid = (unsigned)(blocks < (uint64_t)n_sms * MINB ? blocks : (uint64_t)n_sms * MINB);
#define X(l, f, t)                                                                                                        \
    if (T.n_levels == l && T.F == f && (T.f32 != 0) == t) {                                                               \
        static std::atomic<uint64_t> opted{0};                                                                            \
        if (!opt_in_smem(opted, (const void*)fused_tc_kernel<l, f, t, NWG, MINB, DBG>, 227 * 1024)) return kLaunchCudaError; \
        fused_tc_kernel<l, f, t, NWG, MINB, DBG><<<grid, NWG * 128, smem, stream>>>(T, M, Q, rgb, (uint32_t)n_tiles);     \
        return 1;                                                                                                         \
    }
    OO_TC_SHAPES(X)
#undef X
    return -1;
}

// Largest warpgroup count per SM-resident block whose shared memory fits (6, else 4); -1 if the shape has no instance.
template <bool DBG>
static int launch_fused_tc_impl(const TreeParams& T, const MlpParams& M, const QueryParams& Q, float* rgb, int n_sms, cudaStream_t stream) {
    if (Q.n == 0) return 0;
    if (M.out_dim > 4 || !M.image_tc) return -1;
    const uint32_t a_chunks = (M.k1 > 64 ? M.k1 : 64) / 8;
    const uint32_t per_wg = a_chunks * kTileRows * 16 + (10 + Q.n_extra) * kTileRows * 4;
    const uint32_t fixed = ((T.dense_ints * 4 + 127) & ~127u) + ((M.image_tc_bytes + 127) & ~127u) + 64 + 64;
    const uint32_t limit = 227 * 1024;
    // residency: measured on config 1 (B200): 3 warpgroups x 2 blocks/SM 72.9 us, 6 x 1 75.4 us, 5 x 1 78.6 us, 4 x 1 80.7 us
    if (2 * (fixed + 3 * per_wg + 1024) <= 228 * 1024) return launch_tc_nwg<3, 2, DBG>(T, M, Q, rgb, n_sms, fixed + 3 * per_wg, stream);
    if (fixed + 6 * per_wg <= limit) return launch_tc_nwg<6, 1, DBG>(T, M, Q, rgb, n_sms, fixed + 6 * per_wg, stream);
    if (fixed + 4 * per_wg <= limit) return launch_tc_nwg<4, 1, DBG>(T, M, Q, rgb, n_sms, fixed + 4 * per_wg, stream);
    return -1;
}

// dbg: the instances with the index sink compiled in (oo_query_debug)
int launch_fused_tc(const TreeParams& T, const MlpParams& M, const QueryParams& Q, float* rgb, int n_sms, cudaStream_t stream, bool dbg) {
    return dbg ? launch_fused_tc_impl<true>(T, M, Q, rgb, n_sms, stream) : launch_fused_tc_impl<false>(T, M, Q, rgb, n_sms, stream);
}

}  // namespace oo
