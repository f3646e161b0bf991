// oo_full_fused.cuh — the paper's full query in ONE launch: 8-neighbour / vertex-map / shifted-direction gather
// (oo_full.cuh) -> fp16 row in tensor memory -> tcgen05.mma decoder of width W = 64 or 128 -> RGB.
//
// Same skeleton as oo_fused_tm.cu (A operand of every layer in TMEM, weights in shared memory, accumulator in TMEM, the
// epilogue writes the next A over accumulator columns already read), generalised in two directions:
//   * W = 128: D is 128 columns and A 64, so a tile with an accumulator of its own needs 192 TMEM columns and only TWO fit an SM.
//     Either the accumulators are shared (NSLOT < NTEAM, below: the product form, four one-part teams over two slots), or, to keep the
//     gather phase populated, a tile is worked by a TEAM of KS x 128 threads: part p of the team gathers the levels
//     l = p (mod KS) of the same 128 queries (levels are independent channels, Eq. 11) and writes them to its rows of A
//     (a warp may touch TMEM lanes 32*(warp%4)..+32, so part p's warp 4p+i shares lanes with warp i); the epilogue's
//     32-column chunks are split the same way.  All parts walk the whole descent (one load per level and neighbour).
//   * runtime level count, runtime attribute layout (Eq. 12 or [n | wo | extra]).
// TMEM columns of one team, S = W + max(W/2, k1/2):
//   even layer:  A at [W, W + K/2)    D at [0, W)
//   odd  layer:  A at [0, W/2)        D at [W/2, 3W/2)
// even epilogue: chunk c: ld D[32c, +32) -> st A'[16c, +16);  odd: ld D[W/2 + 32c, +32) -> st A'[W + 16c, +16), c descending.
#pragma once
#include "oo_full.cuh"
#include "oo_tc_ptx.cuh"

namespace oo {

// NSLOT < NTEAM: the accumulators are shared as in fused_tm_kernel (oo_fused_tm.cuh).  A team owns an A region of team_cols = max(W/2, k1/2)
// columns; D (W columns) lives in one of NSLOT slots taken before the tile's first MMA and given back when its output has been read:
// A of team t at [t * team_cols, +team_cols), D slot s at [NTEAM * team_cols + W * s, +W).  The full query spends three quarters of a tile
// in its gather, so four one-part teams share two slots (4 x 64 + 2 x 128 = 512 columns) and no thread walks a descent it does not gather from.
template <int F, bool F32, bool VERTEX, bool TRI8, bool SHIFTED, int W, int KS, int NTEAM, bool DBG, int NSLOT = NTEAM>
__global__ void __launch_bounds__(NTEAM* KS * 128, 1)
    fused_full_kernel(const __grid_constant__ TreeParams T, const __grid_constant__ MlpParams M,
                      const __grid_constant__ QueryParams Q, const __grid_constant__ FullMode mode, float* __restrict__ rgb,
                      uint32_t n_tiles, uint32_t team_cols) {
    constexpr int NJ = TRI8 ? 8 : 1;
    constexpr int TEAM_THREADS = KS * 128;
    constexpr int NCHUNK = W / 32;
    constexpr int CPP = (NCHUNK + KS - 1) / KS;                       // epilogue chunks per part
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t dense_bytes = (T.dense_ints * 4 + 127) & ~127u;
    const uint32_t q_words = 11 + Q.n_extra;                         // x3 n3 wo3 index disparity extras, each [128] words
    const uint32_t q_bytes = q_words * 128 * 4;
    int32_t* s_dense = (int32_t*)smem;
    uint8_t* s_w = smem + dense_bytes;
    uint8_t* s_stage = s_w + ((M.image_tc_bytes + 127) & ~127u);
    uint64_t* s_bar = (uint64_t*)(s_stage + NTEAM * q_bytes);
    uint32_t* s_tmem = (uint32_t*)(s_bar + NTEAM);
    constexpr bool DYN = NSLOT < NTEAM;
    uint32_t* s_free = s_tmem + 1;                               // DYN: bit s set = D slot s is free
    uint32_t* s_slot = s_free + 1;                               // [NTEAM] the slot a team's tile holds
    uint32_t* s_rel = s_slot + NTEAM;                            // [NTEAM] warps of part 0 that are done with the slot

    const uint32_t team = threadIdx.x / TEAM_THREADS, part = (threadIdx.x >> 7) % KS, row = threadIdx.x & 127,
                   warp = threadIdx.x >> 5;
    {
        const uint4* s = (const uint4*)T.dense;
        uint4* d = (uint4*)s_dense;
        for (uint32_t i = threadIdx.x; i < T.dense_ints / 4; i += blockDim.x) d[i] = __ldg(s + i);
        s = (const uint4*)M.image_tc;
        d = (uint4*)s_w;
        for (uint32_t i = threadIdx.x; i < M.image_tc_bytes / 16; i += blockDim.x) d[i] = __ldg(s + i);
    }
    if (threadIdx.x < NTEAM) {
        mbar_init(smem_u32(&s_bar[threadIdx.x]), 1);
        s_rel[threadIdx.x] = 0;
    }
    if (threadIdx.x == 0) *s_free = (1u << NSLOT) - 1u;
    if (threadIdx.x == 0) asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if (warp == 0) {
        tmem_alloc(smem_u32(s_tmem), 512);
        tmem_relinquish();
    }
    fence_async_smem();
    fence_before_sync();
    __syncthreads();
    fence_after_sync();
    const uint32_t tmem_team = *s_tmem + team * team_cols;
    const uint32_t lane_off = (row & ~31u) << 16;
    const uint32_t tmem_d0 = *s_tmem + NTEAM * team_cols;            // DYN: D slot 0
    uint32_t tmem_d = tmem_d0;                                       // DYN: the D slot of the current tile
    // columns of the A operand / the accumulator of a layer of the given parity (warp-uniform)
    auto col_a = [&](bool odd) -> uint32_t { return DYN ? tmem_team : tmem_team + (odd ? 0u : (uint32_t)W); };
    auto col_d = [&](bool odd) -> uint32_t { return DYN ? tmem_d : tmem_team + (odd ? (uint32_t)(W / 2) : 0u); };
    float* s_q = (float*)(s_stage + team * q_bytes) + row;            // word k of my row: s_q[k * 128]
    const uint32_t w_addr = smem_u32(s_w), bar = smem_u32(&s_bar[team]), q_addr = smem_u32(s_q);
    uint32_t phase = 0;
    const bool leader_warp = part == 0 && row < 32;
    constexpr uint32_t idesc_h = instr_desc(128, W), idesc_o = instr_desc(128, 16);
    const uint32_t tile_stride = gridDim.x * NTEAM;
    const uint32_t L = T.n_levels, LF = L * F;

    auto prefetch = [&](uint32_t tile) {      // part 0 only
        const uint64_t t = (uint64_t)tile * 128 + row;
        const uint64_t tt = t < Q.n ? t : Q.n - 1;
        const uint32_t qi = Q.perm ? __ldg(Q.perm + tt) : (uint32_t)tt;
        const float* px = Q.x + (size_t)qi * 3;
        const float* pn = Q.nrm + (size_t)qi * 3;
        const float* pw = Q.wo + (size_t)qi * 3;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            cp_async4(q_addr + (k)*512, px + k);
            cp_async4(q_addr + (3 + k) * 512, pn + k);
            cp_async4(q_addr + (6 + k) * 512, pw + k);
        }
        if constexpr (SHIFTED) cp_async4(q_addr + 10 * 512, Q.disparity + qi);
        for (uint32_t k = 0; k < Q.n_extra; ++k) cp_async4(q_addr + (11 + k) * 512, Q.extra + (size_t)qi * Q.n_extra + k);
        s_q[9 * 128] = __uint_as_float(qi);
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    uint32_t tile = team * gridDim.x + blockIdx.x;        // the partial last round spreads one tile per SM (see oo_fused_tm.cu)
    if (tile < n_tiles && part == 0) prefetch(tile);
    bool sample = Q.stat != nullptr;
    for (; tile < n_tiles; tile += tile_stride) {
        const bool valid = (uint64_t)tile * 128 + row < Q.n;
        if (part == 0) asm volatile("cp.async.wait_group 0;" ::: "memory");
        if constexpr (KS > 1) named_bar(1 + team, TEAM_THREADS);     // the staged queries are visible to every part
        float x[3], w[3], wl[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) { x[k] = s_q[k * 128]; w[k] = s_q[(6 + k) * 128]; }
        if (sample) {                        // OO_PRESORT_AUTO: the first tile of every team
            if (part == 0 && team == 0) stat_sample_warp(Q, blockIdx.x * 4 + (warp & 3u), x[0], x[1], x[2]);
            sample = false;
        }
        if (mode.lookup == OO_LOOKUP_WO) {
#pragma unroll
            for (int a = 0; a < 3; ++a) wl[a] = w[a];
        } else {
            const float n[3] = {s_q[3 * 128], s_q[4 * 128], s_q[5 * 128]};
            mirror_dir(n, w, wl);
        }
        const float disp = SHIFTED ? s_q[10 * 128] : 0.0f;
        OctaUV uv{0.0f, 0.0f};
        if constexpr (!SHIFTED) uv = octa_project(wl[0], wl[1], wl[2]);
        // ------------------------------------------------------------------ gather -> A0 in TMEM (layer 0 is even)
        const uint32_t a0 = col_a(false) + lane_off;
        {
            Station<NJ> st;
            station_init<NJ>(T, s_dense, x, st);
            FullDebug dbg{nullptr, nullptr};
            if constexpr (DBG) {         // oo_query_debug: this query's [L][NJ] slot and [L][NJ][3] index rows (binned: out_idx's)
                const uint64_t t = (uint64_t)tile * 128 + row;
                const uint64_t r = Q.out_idx ? Q.out_idx[t < Q.n ? t : Q.n - 1] : __float_as_uint(s_q[9 * 128]);
                if (valid && Q.dbg_slot) dbg.slot = Q.dbg_slot + r * L * NJ;
                if (valid && Q.dbg_texel) dbg.cell = Q.dbg_texel + r * L * NJ * 3;
            }
            for (uint32_t l = 0; l < L; ++l) {
                const bool mine = KS == 1 || (l % KS) == part;
                float h[F];
                full_level<F, F32, VERTEX, TRI8, SHIFTED>(T.lv[l], s_dense, x, wl, uv, disp, st, mine, h, (int)l, dbg);
                if (mine) {
                    if constexpr (F % 8 == 0) {
#pragma unroll
                        for (int v = 0; v < F / 8; ++v)
                            tmem_st4(a0 + (l * F) / 2 + 4 * v, pack_half2(h[8 * v], h[8 * v + 1]), pack_half2(h[8 * v + 2], h[8 * v + 3]),
                                     pack_half2(h[8 * v + 4], h[8 * v + 5]), pack_half2(h[8 * v + 6], h[8 * v + 7]));
                    } else {   // F == 4
                        tmem_st2(a0 + l * 2, pack_half2(h[0], h[1]), pack_half2(h[2], h[3]));
                    }
                }
            }
        }
        uint32_t qi = 0;
        if (part == 0) {   // attributes (Eq. 12 or [n | wo | extra]) + zero padding up to k1, 4 halves per store
            float e[13], v[32];
#pragma unroll
            for (int k = 0; k < 13; ++k) e[k] = (uint32_t)k < Q.n_extra ? s_q[(11 + k) * 128] : 0.0f;
            const bool paper = mode.attrs_paper != 0;
            float wr[3];
            const float n[3] = {s_q[3 * 128], s_q[4 * 128], s_q[5 * 128]};
            mirror_dir(n, w, wr);
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                v[k] = paper ? x[k] : n[k];
                v[3 + k] = paper ? wr[k] : w[k];
                v[6 + k] = paper ? n[k] : e[k];
            }
#pragma unroll
            for (int k = 9; k < 19; ++k) v[k] = paper ? e[k - 9] : e[k - 6];
#pragma unroll
            for (int k = 19; k < 32; ++k) v[k] = 0.0f;
            qi = __float_as_uint(s_q[9 * 128]);
            const uint32_t chunks = (M.k1 - LF) / 4;
#pragma unroll
            for (int c = 0; c < 8; ++c)
                if ((uint32_t)c < chunks)
                    tmem_st2(a0 + LF / 2 + 2 * c, pack_half2(v[4 * c], v[4 * c + 1]), pack_half2(v[4 * c + 2], v[4 * c + 3]));
        }
        // ------------------------------------------------------------------ hidden layers
        uint32_t w_off = 0;
        for (uint32_t layer = 0; layer < M.n_hidden; ++layer) {
            const uint32_t kt_n = (layer == 0 ? M.k1 : (uint32_t)W) >> 4;
            const bool odd = layer & 1u;
            // the issuing warp forms the layer's operand addresses ahead of the barrier (see oo_fused_tm.cuh): between the barrier and the
            // first tcgen05.mma only the issue itself is left on the tile's critical path
            if constexpr (DYN) {
                if (layer == 0 && leader_warp) {      // lane 0 takes a free D slot (see fused_tm_kernel) and tells its warp and the team
                    uint32_t got = 0;
                    if ((threadIdx.x & 31u) == 0) {
                        got = 0xffffffffu;
                        while (got == 0xffffffffu) {
                            const uint32_t m = *(volatile uint32_t*)s_free;
                            if (m) {
                                const uint32_t b = (uint32_t)__ffs((int)m) - 1u;
                                if (atomicAnd(s_free, ~(1u << b)) & (1u << b)) got = b;
                            } else {
                                __nanosleep(20);
                            }
                        }
                        *(volatile uint32_t*)&s_slot[team] = got;
                    }
                    tmem_d = tmem_d0 + (uint32_t)W * __shfl_sync(0xffffffffu, got, 0);
                }
            }
            uint32_t mma_d = col_d(odd), mma_a = col_a(odd);
            uint64_t mma_b = smem_desc(w_addr + w_off, 16 * W, 128);
            if (leader_warp) asm volatile("" : "+r"(mma_d), "+r"(mma_a), "+l"(mma_b));
            tmem_wait_st();              // my part of A is in TMEM
            fence_before_sync();
            named_bar(1 + team, TEAM_THREADS);
            if constexpr (DYN) {
                if (layer == 0 && !leader_warp) tmem_d = tmem_d0 + (uint32_t)W * *(volatile uint32_t*)&s_slot[team];
            }
            if (leader_warp) {
                fence_after_sync();
                umma_group_ts<8>(mma_d, mma_a, mma_b, (32 * W) >> 4, idesc_h, kt_n, bar);
            }
            if (layer == 0 && part == 0 && tile + tile_stride < n_tiles) prefetch(tile + tile_stride);   // staging is free now
            w_off += kt_n * 32 * W;
            mbar_wait(bar, phase);
            phase ^= 1;
            fence_after_sync();
            // epilogue: my row of D -> ReLU -> fp16 -> my row of the next layer's A (over columns of D already read)
            const uint32_t d_base = col_d(odd) + lane_off;
            const uint32_t a_base = col_a(!odd) + lane_off;
            if constexpr (KS == 1) {
#pragma unroll
                for (int i = 0; i < NCHUNK; ++i) {
                    const uint32_t c = odd ? (uint32_t)(NCHUNK - 1 - i) : (uint32_t)i;
                    uint32_t r[32], p[16];
                    tmem_ld32(d_base + 32 * c, r);
                    tmem_wait_ld();
#pragma unroll
                    for (int k = 0; k < 16; ++k) p[k] = pack_half2_relu(__uint_as_float(r[2 * k]), __uint_as_float(r[2 * k + 1]));
                    tmem_st16(a_base + 16 * c, p);
                }
            } else {
                uint32_t p[CPP][16];
#pragma unroll
                for (int i = 0; i < CPP; ++i) {
                    const uint32_t c = part + (uint32_t)i * KS;
                    if (c < (uint32_t)NCHUNK) {
                        uint32_t r[32];
                        tmem_ld32(d_base + 32 * c, r);
                        tmem_wait_ld();
#pragma unroll
                        for (int k = 0; k < 16; ++k) p[i][k] = pack_half2_relu(__uint_as_float(r[2 * k]), __uint_as_float(r[2 * k + 1]));
                    }
                }
                fence_before_sync();
                named_bar(1 + team, TEAM_THREADS);       // every part has read its chunks of D
                fence_after_sync();
#pragma unroll
                for (int i = 0; i < CPP; ++i) {
                    const uint32_t c = part + (uint32_t)i * KS;
                    if (c < (uint32_t)NCHUNK) tmem_st16(a_base + 16 * c, p[i]);
                }
            }
        }
        // ------------------------------------------------------------------ output layer (N = 16, K = W)
        const bool odd = M.n_hidden & 1u;
        uint32_t out_d = col_d(odd), out_a = col_a(odd);
        uint64_t out_b = smem_desc(w_addr + w_off, 256, 128);
        if (leader_warp) asm volatile("" : "+r"(out_d), "+r"(out_a), "+l"(out_b));
        tmem_wait_st();
        fence_before_sync();
        named_bar(1 + team, TEAM_THREADS);
        if (leader_warp) {
            fence_after_sync();
            umma_group_ts<W / 16>(out_d, out_a, out_b, 512 >> 4, idesc_o, (uint32_t)(W / 16), bar);
        }
        mbar_wait(bar, phase);
        phase ^= 1;
        fence_after_sync();
        if (part == 0) {
            uint32_t o[4];
            tmem_ld4(col_d(odd) + lane_off, o);
            tmem_wait_ld();
            if constexpr (DYN) {      // part 0's four warps are the last readers of the slot
                fence_before_sync();
                __syncwarp();
                if ((threadIdx.x & 31u) == 0 && (atomicAdd(&s_rel[team], 1u) & 3u) == 3u) atomicOr(s_free, 1u << ((tmem_d - tmem_d0) / (uint32_t)W));
            }
            if (valid) {
#pragma unroll
                for (uint32_t c = 0; c < 4; ++c)
                    if (c < M.out_dim) {
                        const float z = __uint_as_float(o[c]);
                        rgb[(size_t)qi * M.out_dim + c] = M.out_act == OO_ACT_EXP ? fast_exp(z) : z;
                    }
            }
        }
        // no barrier here: the next tile's gather writes A0 at [W, ...), which neither the output accumulator ([0,16) or
        // [W/2, W/2+16)) nor anything still in flight overlaps (every thread has seen the output MMA complete)
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem_dealloc(*s_tmem, 512);
}

// ---------------------------------------------------------------------------------------------------------------------
template <int F, bool F32, bool VERTEX, bool TRI8, bool SHIFTED, int W, int KS, int NTEAM, bool DBG, int NSLOT = NTEAM>
static int launch_full_inst(const TreeParams& T, const MlpParams& M, const QueryParams& Q, const FullModeH& mode, float* rgb,
                            int n_sms, uint32_t team_cols, cudaStream_t stream) {
    const uint64_t n_tiles = (Q.n + 127) / 128;
    const uint64_t blocks = (n_tiles + NTEAM - 1) / NTEAM;
    const unsigned grid = (unsigned)(blocks < (uint64_t)n_sms ? blocks : (uint64_t)n_sms);
    const uint32_t smem = ((T.dense_ints * 4 + 127) & ~127u) + ((M.image_tc_bytes + 127) & ~127u) + NTEAM * (11 + Q.n_extra) * 128 * 4 + 256;
    if (smem > 227 * 1024) return -1;
    auto kern = fused_full_kernel<F, F32, VERTEX, TRI8, SHIFTED, W, KS, NTEAM, DBG, NSLOT>;
    static std::atomic<uint64_t> opted{0};
    if (!opt_in_smem(opted, (const void*)kern, 227 * 1024)) return kLaunchCudaError;
    kern<<<grid, NTEAM * KS * 128, smem, stream>>>(T, M, Q, mode, rgb, (uint32_t)n_tiles, team_cols);
    return 1;
}

#define OO_FULL_MODES(X, f, t) \
    X(f, t, false, false, false) X(f, t, false, false, true) X(f, t, false, true, false) X(f, t, false, true, true) \
    X(f, t, true, false, false) X(f, t, true, false, true) X(f, t, true, true, false) X(f, t, true, true, true)

// dispatch over (F, dtype, vertex, tri8, shifted) for a fixed (W, KS, NTEAM)
template <int W, int KS, int NTEAM, bool DBG, int NSLOT = NTEAM>
static int launch_full_w(const TreeParams& T, const MlpParams& M, const QueryParams& Q, const FullModeH& mode, float* rgb,
                         int n_sms, uint32_t team_cols, cudaStream_t stream) {
    const bool vertex = T.vertex != 0, tri8 = mode.tri8 != 0, shifted = mode.lookup == OO_LOOKUP_SHIFTED;
#define X(f, t, v, s8, sh)                                                                                 \
    if (T.F == f && (T.f32 != 0) == t && vertex == v && tri8 == s8 && shifted == sh)                       \
        return launch_full_inst<f, t, v, s8, sh, W, KS, NTEAM, DBG, NSLOT>(T, M, Q, mode, rgb, n_sms, team_cols, stream);
    OO_FULL_MODES(X, 4, true)
    OO_FULL_MODES(X, 8, false)
    OO_FULL_MODES(X, 16, false)
#undef X
    return -1;
}

}  // namespace oo
