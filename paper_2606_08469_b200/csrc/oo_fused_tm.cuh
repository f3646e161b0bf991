// oo_fused_tm.cuh — fused encode + MLP on tcgen05 with the activations resident in TENSOR MEMORY (OO_PATH_FUSED_TC_TMEM).
//
// Same arithmetic as oo_fused_tc.cu; the A operand of every layer lives in TMEM instead of shared memory:
//   gather (registers, fp32) -> fp16 row -> tcgen05.st into this thread's TMEM lane (two halves per 32-bit column)
//   -> tcgen05.mma.kind::f16 with A from TMEM, B (weights) from shared memory, D in TMEM
//   -> tcgen05.ld own row of D -> ReLU -> fp16 -> tcgen05.st as the next layer's A -> ... -> output layer -> exp -> RGB.
// What that buys (ncu, config 1, oo_fused_tc.cu): the shared-memory A tile cost 540 of ~1500 L1 data-pipe wavefronts per
// 128-query tile (l1tex 66 % busy, the busiest unit) and 2 x 100 KB of shared memory that left the gathers ~28 KB of L1.
// Here a block needs only the descent tables, the weight image and 5 KB of query staging per warpgroup.
//
// TMEM columns of one warpgroup (stride S = 64 + max(32, k1/2)); D is 64 fp32 columns, A is K/2 columns:
//   even layer:  A at [64, 64 + K/2)   D at [0, 64)
//   odd  layer:  A at [0, 32)          D at [32, 96)
// so the epilogue of a layer writes the next A over columns of D that it has already read (own lane only):
//   even: ld D[0,32) -> st A'[0,16);  ld D[32,64) -> st A'[16,32)
//   odd : ld D[64,96) -> st A'[80,96) (k = 32..63);  ld D[32,64) -> st A'[64,80) (k = 0..31)
// One persistent block per SM (it allocates all 512 columns) with NWG = 512 / S warpgroups (5 when k1 <= 64).
//
// Included by oo_fused_tm.cu (DBG = false: the product instances) and oo_fused_tm_dbg.cu (DBG = true: the same kernels with
// the index sink of oo_query_debug compiled in, see IndexDbg in oo_device.cuh).
#pragma once
#include <cstdio>

#include "oo_device.cuh"
#include "oo_tc_ptx.cuh"

namespace oo {

namespace {
constexpr int kRows = 128;

// ReLU + fp16 pack of 32 accumulator columns -> 16 registers
__device__ __forceinline__ void relu_pack32(const uint32_t (&r)[32], uint32_t (&p)[16]) {
#pragma unroll
    for (int c = 0; c < 16; ++c) p[c] = pack_half2_relu(__uint_as_float(r[2 * c]), __uint_as_float(r[2 * c + 1]));
}
}  // namespace

// PIPE (chosen at launch for fp16 trees whose first two used levels are dense and the rest hops, i.e. the BASELINE.json configs):
// the hop chain and the gathers overlap.  Stage l resolves slot l from the hop load issued one stage earlier, issues the next
// hop and the taps of level l, and consumes the taps of level l-RD (RD = 2, or 3 for 16-byte texels): a query exposes max(hop, taps) once per hop level plus one
// last gather (4 latencies for L = 5) instead of every hop and then every gather batch (6).  Same taps, same weights, same
// accumulation order per level: bit-identical to the batched form.
// KS (first layers wider than 64 inputs, L*F >= 64): layer 0 runs as TWO MMA groups over the same 32 A columns.  The first 64
// inputs (the levels below feature 64) are multiplied as soon as they are stored; the rest of the row (later levels, attributes,
// padding) is gathered and packed while that MMA is in flight, stored over the same columns once it has completed, and
// accumulated by the second group.  A tile then needs 96 TMEM columns like the narrow configs instead of 64 + k1/2, so five
// warpgroups fit where four did (config 3: k1 = 96, 112 columns), at the price of one more MMA round trip per tile.
// H, K1, NX (0, 0, -1 = read from the parameter structs): the decoder's hidden-layer count, the padded width of its first layer and the
// number of extra scalars as compile-time constants, with out_dim = 3 through exp implied.  The instances of the BASELINE.json configs
// are compiled this way: the layer loop unrolls, the K-step predicates of the MMA issue, the attribute-row conditionals and most
// parameter loads fold away (config 1: 901 -> ~780 thread instructions per query).  Same arithmetic, same order: bit-identical.
// NSLOT < NWG (k1 <= 64 or KS, i.e. 32 A columns): the accumulators are SHARED.  Every warpgroup owns an A region of 32 columns (its tile's
// activations) and the fp32 accumulator D (64 columns) lives in one of NSLOT slots taken from a free mask in shared memory right before the
// tile's first MMA and given back when its four warps have read the output:  A of warpgroup wg at [32 wg, +32), D slot s at
// [32 NWG + 64 s, +64); 6 x 32 + 5 x 64 = 512 columns.  A tile needs a D slot only for the decoder half of its life, so six tiles share five.
// The epilogue reads its whole row of D into registers and then writes the next layer's A over the A region (the MMA that read it has completed).
template <int L, int F, bool F32, int NWG, bool PIPE = false, bool KS = false, bool DBG = false, int H = 0, int K1 = 0, int NX = -1, int NSLOT = NWG>
__global__ void __launch_bounds__(NWG * 128, 1) fused_tm_kernel(const __grid_constant__ TreeParams T,
                                                               const __grid_constant__ MlpParams M,
                                                               const __grid_constant__ QueryParams Q,
                                                               float* __restrict__ rgb, uint32_t n_tiles, uint32_t wg_cols) {
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t dense_bytes = (T.dense_ints * 4 + 127) & ~127u;
    constexpr bool DYN = NSLOT < NWG;                                 // accumulator slots are handed around
    constexpr bool SPEC = H != 0;                                     // (then out_dim = 3 through exp: checked by the launcher)
    const uint32_t n_extra = NX >= 0 ? (uint32_t)NX : Q.n_extra;
    const uint32_t n_hidden = H ? (uint32_t)H : M.n_hidden;
    const uint32_t k1 = K1 ? (uint32_t)K1 : M.k1;
    const uint32_t q_words = 10 + n_extra;                           // x3 n3 wo3 index extras, each [128] words
    const uint32_t q_bytes = q_words * kRows * 4;
    int32_t* s_dense = (int32_t*)smem;
    uint8_t* s_w = smem + dense_bytes;
    uint8_t* s_stage = s_w + ((M.image_tc_bytes + 127) & ~127u);
    float* s_out = (float*)(s_stage + NWG * q_bytes);            // [NWG * 4 warps][32 rows * 3]: a warp's RGB rows before their 16-byte stores
    uint64_t* s_bar = (uint64_t*)(s_out + NWG * 4 * 96);         // one per warpgroup, then tables, then weights
    uint32_t* s_tmem = (uint32_t*)(s_bar + NWG + 2);
    uint32_t* s_free = s_tmem + 1;                               // DYN: bit s set = D slot s is free
    uint32_t* s_slot = s_free + 1;                               // [NWG] the slot a warpgroup's tile holds, for its other warps
    uint32_t* s_rel = s_slot + NWG;                              // [NWG] warps of the warpgroup that are done with the slot

    const uint32_t wg = threadIdx.x >> 7, row = threadIdx.x & 127, warp = threadIdx.x >> 5;
    // Prologue: the descent tables and the weight image arrive by two bulk asynchronous copies that thread 0 issues before
    // anything else; the tables are awaited by every thread before its first descent, the weights only by the warp that issues
    // the MMAs, right before its first one (both travel through the async proxy: no proxy fence, no block barrier for them).
    // Before: 512-640 threads looping LDG.128 -> STS over 54 KB of cold lines, then fence.proxy.async + __syncthreads.
    const uint32_t bar_d = smem_u32(&s_bar[NWG]), bar_w = smem_u32(&s_bar[NWG + 1]);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < NWG + 2; ++k) mbar_init(smem_u32(&s_bar[k]), 1);
        *s_free = (1u << NSLOT) - 1u;
#pragma unroll
        for (int k = 0; k < NWG; ++k) s_rel[k] = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        mbar_expect_tx(bar_d, T.dense_ints * 4);
        bulk_g2s(smem_u32(s_dense), T.dense, T.dense_ints * 4, bar_d);
        mbar_expect_tx(bar_w, M.image_tc_bytes);
        bulk_g2s(smem_u32(s_w), M.image_tc, M.image_tc_bytes, bar_w);
    }
    float* s_q = (float*)(s_stage + wg * q_bytes) + row;             // word k of my row: s_q[k * 128]
    const uint32_t q_addr = smem_u32(s_q);
    auto prefetch = [&](uint32_t tile) {
        const uint64_t t = (uint64_t)tile * kRows + row;
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
#pragma unroll(NX > 0 ? NX : 1)
        for (uint32_t k = 0; k < n_extra; ++k) cp_async4(q_addr + (10 + k) * 512, Q.extra + (size_t)qi * n_extra + k);
        s_q[9 * 128] = __uint_as_float(qi);
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    // Warpgroup wg of block b takes tiles wg*grid + b, + grid*NWG, ...: the n_tiles mod (grid*NWG) tiles of the last, partial
    // round then land one per SM (a lone warpgroup finishes its tile about twice as fast as five sharing an SM) instead of five
    // per SM on a few SMs.  Measured on B200: config 1 61.1 -> 60.1 us, config 3 333.3 -> 329.4 us.
    uint32_t tile = wg * gridDim.x + blockIdx.x;
    if (tile < n_tiles) prefetch(tile);       // the first tile's queries travel while TMEM is allocated and the tables arrive
    if (warp == 0) {
        tmem_alloc(smem_u32(s_tmem), 512);
        tmem_relinquish();
    }
    fence_before_sync();
    __syncthreads();
    fence_after_sync();
    const uint32_t tmem_wg = *s_tmem + wg * wg_cols;                 // this warpgroup's columns (DYN: wg_cols = 32, its A region)
    const uint32_t lane_off = (row & ~31u) << 16;                    // ... and this warp's 32 lanes
    const uint32_t tmem_d0 = *s_tmem + NWG * wg_cols;                // DYN: D slot 0
    uint32_t tmem_d = tmem_d0;                                       // DYN: the D slot of the current tile
    // columns of the A operand / the accumulator of a layer of the given parity (warp-uniform, no lane offset)
    auto col_a = [&](bool odd) -> uint32_t { return DYN ? tmem_wg : tmem_wg + (odd ? 0u : 64u); };
    auto col_d = [&](bool odd) -> uint32_t { return DYN ? tmem_d : tmem_wg + (odd ? 32u : 0u); };
    const uint32_t w_addr = smem_u32(s_w), bar = smem_u32(&s_bar[wg]);
    const bool rgb_vec = !Q.perm && !Q.out_idx && ((uintptr_t)rgb & 15u) == 0;   // rows in order and the output 16-byte aligned: vector stores
    uint32_t phase = 0;
    // The warp that issues a warpgroup's MMAs executes ~45 % more instructions per tile than the other three (descriptor arithmetic on the
    // uniform datapath, elect, commit) and every tile waits for it: the five issuing warps sit on different scheduler partitions
    // (warp index mod 4) instead of all on partition 0 (ncu before: issue slots 75 % busy there, 51 % on the other three).
    const bool leader_warp = (row >> 5) == (wg & 3u);
    // DYN: lane 0 of the issuing warp takes a free D slot (spinning while all are busy: a holder never waits on anyone), tells its own warp
    // by shuffle and the other three through shared memory (they read it after the barrier that precedes the tile's first MMA)
    auto acquire_slot = [&]() {
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
            *(volatile uint32_t*)&s_slot[wg] = got;
        }
        tmem_d = tmem_d0 + 64u * __shfl_sync(0xffffffffu, got, 0);
    };
    constexpr uint32_t idesc_h = instr_desc(128, 64), idesc_o = instr_desc(128, 16);
    const uint32_t tile_stride = gridDim.x * NWG;

    mbar_wait(bar_d, 0);                  // descent tables in shared memory
    bool w_ready = false;
    if (Q.stat && wg == 0 && tile < n_tiles) {   // OO_PRESORT_AUTO: the warps of warpgroup 0 sample their first tile, before the tile loop
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        stat_sample_warp(Q, blockIdx.x * 4 + warp, s_q[0], s_q[128], s_q[256]);
    }
#ifdef OO_PROFILE_PHASES      // -DOO_PROFILE_PHASES: per-warp cycle counts of the phases of a tile (one block prints them); never in the product build
    long long t_gather = 0, t_mlp = 0, t_wait = 0, t_q = 0, t_bar = 0;
    int n_done = 0;
    const long long t_begin = clock64();
#endif
    for (; tile < n_tiles; tile += tile_stride) {
        float x[3], w[3];
        const bool valid = (uint64_t)tile * kRows + row < Q.n;
#ifdef OO_PROFILE_PHASES
        const long long t0 = clock64();
#endif
        asm volatile("cp.async.wait_group 0;" ::: "memory");
#ifdef OO_PROFILE_PHASES
        const long long t0b = clock64();
        long long tw = 0, tb = 0;
#endif
#pragma unroll
        for (int k = 0; k < 3; ++k) { x[k] = s_q[k * 128]; w[k] = s_q[(6 + k) * 128]; }
        // ------------------------------------------------------------------ gather: one query per thread -> A0 in TMEM
        const uint32_t a0 = col_a(false) + lane_off;                 // my row of layer 0's A
        uint64_t dbg_row = 0;
        if constexpr (DBG) {             // where this query's index rows go: its own index (binned queries: out_idx's)
            const uint64_t t = (uint64_t)tile * kRows + row;
            dbg_row = Q.out_idx ? Q.out_idx[t < Q.n ? t : Q.n - 1] : __float_as_uint(s_q[9 * 128]);
        }
        const auto dbg = make_dbg<DBG>(Q, L, dbg_row, valid);
        constexpr int N_LATE = KS ? (L * F - 64) / 2 : 0;            // packed halves of the levels past input 64 (KS)
        uint32_t late[N_LATE > 0 ? N_LATE : 1];
        auto store_level = [&](int l, const float (&h)[F]) {
            if constexpr (KS) {
                if (l * F >= 64) {            // kept in registers until the first MMA group has read the A columns
#pragma unroll
                    for (int k = 0; k < F / 2; ++k) late[(l * F - 64) / 2 + k] = pack_half2(h[2 * k], h[2 * k + 1]);
                    return;
                }
            }
            if constexpr (F % 8 == 0) {
#pragma unroll
                for (int v = 0; v < F / 8; ++v)
                    tmem_st4(a0 + (l * F) / 2 + 4 * v, pack_half2(h[8 * v], h[8 * v + 1]), pack_half2(h[8 * v + 2], h[8 * v + 3]),
                             pack_half2(h[8 * v + 4], h[8 * v + 5]), pack_half2(h[8 * v + 6], h[8 * v + 7]));
            } else {   // F == 4
                tmem_st2(a0 + (l * 4) / 2, pack_half2(h[0], h[1]), pack_half2(h[2], h[3]));
            }
            if constexpr (KS) {
                if ((l + 1) * F == 64) {      // inputs 0..63 of all 128 rows are in TMEM: first MMA group of layer 0
                    if constexpr (DYN) {
                        if (leader_warp) acquire_slot();
                    }
                    uint32_t g_d = col_d(false), g_a = col_a(false);
                    uint64_t g_b = smem_desc(w_addr, 1024, 128);
                    if (leader_warp) {           // operand addresses and the weights' arrival ahead of the barrier (see the hidden layers)
                        asm volatile("" : "+r"(g_d), "+r"(g_a), "+l"(g_b));
                        if (!w_ready) {
                            mbar_wait(bar_w, 0);
                            w_ready = true;
                        }
                    }
                    tmem_wait_st();
                    fence_before_sync();
                    named_bar(1 + wg, 128);
                    if constexpr (DYN) {
                        if (!leader_warp) tmem_d = tmem_d0 + 64u * *(volatile uint32_t*)&s_slot[wg];
                    }
                    if (leader_warp) {
                        fence_after_sync();
                        umma_group_ts<4>(g_d, g_a, g_b, 2048 >> 4, idesc_h, 4u, bar);
                    }
                }
            }
        };
        if constexpr (PIPE && L >= 3) {
            gather_pipelined<L, F, F32>(T, s_dense, x, w, store_level, dbg);
        } else {
            Encoded<L, F, F32> e;
            locate<L, F, F32>(T, s_dense, x, w, e);
            constexpr int NB = (F * (F32 ? 4 : 2) == 16) ? (L < 4 ? L : 4) : (F * (F32 ? 4 : 2) == 32 ? 2 : 1);   // levels per load batch
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
                    store_level(l, h[b]);
                }
            }
        }
        uint32_t qi;
        const uint32_t aA = KS ? a0 - 32 : a0;   // KS: input k >= 64 lives at column (k - 64) / 2 of the same A region
        if constexpr (KS) {
            mbar_wait(bar, phase);                // the first MMA group has read inputs 0..63
            phase ^= 1;
            fence_after_sync();
#pragma unroll
            for (int v = 0; v < N_LATE / 4; ++v) tmem_st4(a0 + 4 * v, late[4 * v], late[4 * v + 1], late[4 * v + 2], late[4 * v + 3]);
        }
        {   // attributes + zero padding up to k1, read late from the staging buffer.  (A shorter special case for "no extras" --
            // [n | wo | 0 0] as one 4-column store, ~30 instructions fewer per query -- measured 5 us SLOWER on config 1: this kernel
            // is bound by how its dependent chains interleave, not by its instruction count.)
            float v[24];
#pragma unroll
            for (int k = 0; k < 24; ++k) v[k] = 0.0f;
            constexpr int lead = (L * F) % 8;            // 0 or 4: position of n inside its 8-half unit
#pragma unroll
            for (int k = 0; k < 3; ++k) { v[lead + k] = s_q[(3 + k) * 128]; v[lead + 3 + k] = w[k]; }
#pragma unroll
            for (int k = 0; k < OO_MAX_EXTRA; ++k)
                if ((uint32_t)k < n_extra) v[lead + 6 + k] = s_q[(10 + k) * 128];
            qi = __float_as_uint(s_q[9 * 128]);
            constexpr int c0 = (L * F) / 8;              // first 8-half unit (4 columns) holding attributes
            const uint32_t c_end = k1 / 8;
            if constexpr (lead == 0) {
                tmem_st4(aA + 4 * c0, pack_half2(v[0], v[1]), pack_half2(v[2], v[3]), pack_half2(v[4], v[5]), pack_half2(v[6], v[7]));
            } else {
                tmem_st2(aA + 4 * c0 + 2, pack_half2(v[4], v[5]), pack_half2(v[6], v[7]));
            }
            if (c0 + 1 < c_end)
                tmem_st4(aA + 4 * (c0 + 1), pack_half2(v[8], v[9]), pack_half2(v[10], v[11]), pack_half2(v[12], v[13]), pack_half2(v[14], v[15]));
            if (c0 + 2 < c_end)
                tmem_st4(aA + 4 * (c0 + 2), pack_half2(v[16], v[17]), pack_half2(v[18], v[19]), pack_half2(v[20], v[21]), pack_half2(v[22], v[23]));
        }
#ifdef OO_PROFILE_PHASES
        const long long t1 = clock64();
#endif
        // ------------------------------------------------------------------ hidden layers
        uint32_t w_off = 0;
#pragma unroll(H ? H : 1)
        for (uint32_t layer = 0; layer < n_hidden; ++layer) {
            const uint32_t kt_n = (layer == 0 ? k1 : 64u) >> 4;
            const bool second = KS && layer == 0;         // layer 0's inputs 64.. : 4 K-steps further into W0, accumulating
            const bool odd = layer & 1u;
#ifdef OO_PROFILE_PHASES
            const long long tb0 = clock64();
#endif
            // The issuing warp forms this layer's operand addresses BEFORE it waits for the other warps' rows (the empty volatile asm pins
            // the values ahead of the barrier): between the barrier and the first tcgen05.mma only the issue itself is left.  Every
            // instruction of that warp there is on the tile's critical path and takes ~9 cycles with five warps sharing a scheduler.
            if constexpr (DYN && !KS) {
                if (layer == 0 && leader_warp) acquire_slot();
            }
            uint32_t mma_d = col_d(odd), mma_a = col_a(odd);
            uint64_t mma_b = smem_desc(w_addr + w_off + (second ? 4u * 2048u : 0u), 1024, 128);
            if (leader_warp) {
                asm volatile("" : "+r"(mma_d), "+r"(mma_a), "+l"(mma_b));
                if (layer == 0 && !w_ready) {
                    mbar_wait(bar_w, 0);      // weight image in shared memory (first MMA of this warpgroup only)
                    w_ready = true;
                }
            }
            tmem_wait_st();              // my row of A is in TMEM
            fence_before_sync();
            named_bar(1 + wg, 128);
#ifdef OO_PROFILE_PHASES
            tb += clock64() - tb0;
#endif
            if constexpr (DYN && !KS) {
                if (layer == 0 && !leader_warp) tmem_d = tmem_d0 + 64u * *(volatile uint32_t*)&s_slot[wg];
            }
            if (leader_warp) {
                fence_after_sync();
                umma_group_ts<8>(mma_d, mma_a, mma_b, 2048 >> 4, idesc_h, second ? kt_n - 4u : kt_n, bar, second ? 1u : 0u);
            }
            // the next tile's queries are requested inside layer 0's MMA window (the staging buffer was read above): ~35 instructions
            // per thread that would otherwise sit between the gather and the first MMA of every tile
            if (layer == 0 && tile + tile_stride < n_tiles) prefetch(tile + tile_stride);
            w_off += kt_n * 2 * 1024;
#ifdef OO_PROFILE_PHASES
            const long long tw0 = clock64();
#endif
            mbar_wait(bar, phase);
#ifdef OO_PROFILE_PHASES
            tw += clock64() - tw0;
#endif
            phase ^= 1;
            fence_after_sync();
            // epilogue: my row of D -> ReLU -> fp16 -> my row of the next layer's A (over columns of D already read)
            // both halves of D are requested before the single wait::ld, so the second TMEM read hides behind the first
            uint32_t r0[32], r1[32], p[16];
            const uint32_t d_lane = col_d(odd) + lane_off, a_next = col_a(!odd) + lane_off;
            tmem_ld32(d_lane, r0);                  // outputs 0..31
            tmem_ld32(d_lane + 32, r1);             // outputs 32..63
            tmem_wait_ld();                         // the whole row is in registers: the next A may overlap D's columns
            relu_pack32(r0, p);
            tmem_st16(a_next, p);
            relu_pack32(r1, p);
            tmem_st16(a_next + 16, p);
        }
        // ------------------------------------------------------------------ output layer (N = 16, K = 64)
        const bool odd = n_hidden & 1u;
        uint32_t out_d = col_d(odd), out_a = col_a(odd);
        uint64_t out_b = smem_desc(w_addr + w_off, 256, 128);
        if (leader_warp) asm volatile("" : "+r"(out_d), "+r"(out_a), "+l"(out_b));       // formed ahead of the barrier, as above
        tmem_wait_st();
        fence_before_sync();
        named_bar(1 + wg, 128);
        if (leader_warp) {
            fence_after_sync();
            umma_group_ts<4>(out_d, out_a, out_b, 512 >> 4, idesc_o, 4u, bar);
        }
        mbar_wait(bar, phase);
        phase ^= 1;
        fence_after_sync();
        // the output MMA is N = 16 wide: columns 0..3 always, 4..7 (into the same registers) only for out_dim > 4
        const uint32_t o_addr = col_d(odd) + lane_off;
        uint32_t o[4], o_hi[4];
        tmem_ld4(o_addr, o);
        if (!SPEC && M.out_dim > 4) tmem_ld4(o_addr + 4, o_hi);
        tmem_wait_ld();
        if constexpr (DYN) {          // this warp is done with the D slot; the last of the four warps gives it back
            fence_before_sync();
            __syncwarp();
            if ((threadIdx.x & 31u) == 0 && (atomicAdd(&s_rel[wg], 1u) & 3u) == 3u) atomicOr(s_free, 1u << ((tmem_d - tmem_d0) >> 6));
        }
        if (SPEC || (M.out_dim == 3 && M.out_act == OO_ACT_EXP)) {       // RGB through exp: the case every BASELINE.json config runs
            const float r0 = fast_exp(__uint_as_float(o[0])), r1 = fast_exp(__uint_as_float(o[1])), r2 = fast_exp(__uint_as_float(o[2]));
            // A warp's 32 rows are 384 contiguous bytes of the output when the queries are processed in order: they go through a
            // warp-private strip of shared memory and leave as 24 sixteen-byte stores (whole 32-byte sectors: what makes writing the RGB
            // straight into pinned HOST memory run at the link rate, oo_query_host) instead of 96 four-byte ones.
            // in order (qi = position) and all 32 rows of the warp exist.  (The same test as `__all_sync(valid)` measured 0.9 us slower.)
            if (rgb_vec && (uint64_t)tile * kRows + (row | 31u) < Q.n) {
                float* so = s_out + warp * 96;
                const uint32_t lane = row & 31u;
                so[3 * lane] = r0; so[3 * lane + 1] = r1; so[3 * lane + 2] = r2;
                __syncwarp();
                if (lane < 24) reinterpret_cast<float4*>(rgb + (size_t)(qi - lane) * 3)[lane] = reinterpret_cast<const float4*>(so)[lane];
                __syncwarp();
            } else if (valid) {
                float* dst = rgb + (size_t)qi * 3;
                dst[0] = r0; dst[1] = r1; dst[2] = r2;
            }
        } else {
            if (valid) {
#pragma unroll
                for (uint32_t c = 0; c < 4; ++c)
                    if (c < M.out_dim) {
                        const float z = __uint_as_float(o[c]);
                        rgb[(size_t)qi * M.out_dim + c] = M.out_act == OO_ACT_EXP ? fast_exp(z) : z;
                    }
            }
            if (M.out_dim > 4) {
                if (valid) {
#pragma unroll
                    for (uint32_t c = 0; c < 4; ++c)
                        if (4 + c < M.out_dim) {
                            const float z = __uint_as_float(o_hi[c]);
                            rgb[(size_t)qi * M.out_dim + 4 + c] = M.out_act == OO_ACT_EXP ? fast_exp(z) : z;
                        }
                }
            }
        }
#ifdef OO_PROFILE_PHASES
        const long long t2 = clock64();
        t_q += t0b - t0; t_gather += t1 - t0b; t_mlp += t2 - t1; t_wait += tw; t_bar += tb; ++n_done;
#endif
    }
#ifdef OO_PROFILE_PHASES
    if (blockIdx.x == 3 && (threadIdx.x & 31) == 0 && n_done)
        printf("wg %u warp %u tiles %d total %lld qwait %lld gather %lld mlp %lld (mma-wait %lld, bar %lld) cycles per tile\n", wg, warp & 3, n_done,
               (clock64() - t_begin) / n_done, t_q / n_done, t_gather / n_done, t_mlp / n_done, t_wait / n_done, t_bar / n_done);
#endif
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem_dealloc(*s_tmem, 512);
}

// ---------------------------------------------------------------------------------------------------------------------
// every L whose first layer fits the 128-input limit of the TMEM A region (L*F + 6 + extras <= 128)
#define OO_TM_SHAPES(X)                                                                                                   \
    X(1, 8, false) X(2, 8, false) X(3, 8, false) X(4, 8, false) X(5, 8, false) X(6, 8, false) X(7, 8, false) X(8, 8, false) \
    X(1, 16, false) X(2, 16, false) X(3, 16, false) X(4, 16, false) X(5, 16, false) X(6, 16, false) X(7, 16, false)       \
    X(1, 4, true) X(2, 4, true) X(3, 4, true) X(4, 4, true) X(5, 4, true) X(6, 4, true) X(7, 4, true) X(8, 4, true)

#define OO_TM_PIPE_SHAPES(X)                                                                   \
    X(3, 16, false) X(4, 16, false) X(5, 16, false) X(6, 16, false) X(7, 16, false)            \
    X(3, 8, false) X(4, 8, false) X(5, 8, false) X(6, 8, false) X(7, 8, false) X(8, 8, false)

// the two-group first layer (KS) exists where the levels below input 64 fill those 64 inputs exactly
static bool ks_applies(const TreeParams& T, const MlpParams& M) {
    return M.k1 > 64 && T.n_levels * T.F >= 64 && T.F % 8 == 0 && 64 % T.F == 0;
}
#define OO_TM_KS_SHAPES(X) X(4, 16, false) X(5, 16, false) X(6, 16, false) X(7, 16, false) X(8, 8, false)

// one instance with the decoder's shape compiled in (see H, K1, NX above)
template <int L, int F, int NWG, bool KS, bool DBG, int H, int K1, int NX, int NSLOT = NWG>
static int launch_tm_spec(const TreeParams& T, const MlpParams& M, const QueryParams& Q, float* rgb, int n_sms, uint32_t wg_cols, cudaStream_t stream) {
    const uint64_t n_tiles = (Q.n + kRows - 1) / kRows;
    const unsigned grid = (unsigned)(n_tiles < (uint64_t)n_sms ? n_tiles : (uint64_t)n_sms);
    const uint32_t smem = ((T.dense_ints * 4 + 127) & ~127u) + ((M.image_tc_bytes + 127) & ~127u) + NWG * (10 + Q.n_extra) * kRows * 4 + NWG * 4 * 96 * 4 + 256;
    if (smem > 227 * 1024) return -1;
    static std::atomic<uint64_t> opted{0};
    auto kern = fused_tm_kernel<L, F, false, NWG, true, KS, DBG, H, K1, NX, NSLOT>;
    if (!opt_in_smem(opted, (const void*)kern, 227 * 1024)) return kLaunchCudaError;
    kern<<<grid, NWG * 128, smem, stream>>>(T, M, Q, rgb, (uint32_t)n_tiles, wg_cols);
    return 1;
}

template <int NWG, bool PIPE, bool KS, bool DBG>
static int launch_tm_variant(const TreeParams& T, const MlpParams& M, const QueryParams& Q, float* rgb, int n_sms, uint32_t wg_cols,
                             cudaStream_t stream) {
    const uint64_t n_tiles = (Q.n + kRows - 1) / kRows;
    // one block per SM as soon as there is a tile for each: a small batch spreads over all SMs (a warpgroup alone on its SM
    // finishes a tile faster than four sharing one) instead of filling every warpgroup of the first n_tiles / NWG SMs
    const unsigned grid = (unsigned)(n_tiles < (uint64_t)n_sms ? n_tiles : (uint64_t)n_sms);
    const uint32_t smem = ((T.dense_ints * 4 + 127) & ~127u) + ((M.image_tc_bytes + 127) & ~127u) + NWG * (10 + Q.n_extra) * kRows * 4 + NWG * 4 * 96 * 4 + 256;
    if (smem > 227 * 1024) return -1;
#define X(l, f, t)                                                                                                     \
    if (T.n_levels == l && T.F == f && (T.f32 != 0) == t) {                                                            \
        static std::atomic<uint64_t> opted{0};                                                                         \
        if (!opt_in_smem(opted, (const void*)fused_tm_kernel<l, f, t, NWG, PIPE, KS, DBG>, 227 * 1024)) return kLaunchCudaError; \
        fused_tm_kernel<l, f, t, NWG, PIPE, KS, DBG><<<grid, NWG * 128, smem, stream>>>(T, M, Q, rgb, (uint32_t)n_tiles, wg_cols); \
        return 1;                                                                                                      \
    }
    if constexpr (KS) {
        OO_TM_KS_SHAPES(X)
    } else if constexpr (PIPE) {
        OO_TM_PIPE_SHAPES(X)
    } else {
        OO_TM_SHAPES(X)
    }
#undef X
    return -1;
}

// warpgroups per block = how many column strides fit in the 512 TMEM columns; -1 if the shape has no instance
template <bool DBG>
static int launch_fused_tm_impl(const TreeParams& T, const MlpParams& M, const QueryParams& Q, float* rgb, int n_sms, cudaStream_t stream) {
    if (Q.n == 0) return 0;
    if (M.out_dim > 8 || !M.image_tc || M.k1 > 128) return -1;
    // Measured on B200 (PIPE against the batched form): config 1 60.2 -> 58.6 us, config 2 55.3 -> 54.5 us, config 3 326 -> 309 us,
    // unsorted incoherent 2^22 queries 1.53 -> 1.32 ms.  Binned queries: mixed with four warpgroups (-2 % at 2^22, +8 % at 2^24),
    // a gain at every size once KS runs five (2^22 0.657 -> 0.632 ms, 2^24 2.40 -> 2.22 ms), so PIPE is used wherever it applies.
    const bool pipe = pipe_applies(T);
    // the BASELINE.json configs: decoder shape compiled in (configs 1, 2: 38/39 -> 3 x 64 -> 3 exp on L = 4, F = 8; configs 3, 4: 86 -> 4 x 64 -> 3 exp on L = 5, F = 16)
    if (pipe && M.out_dim == 3 && M.out_act == OO_ACT_EXP && !T.f32) {
        // warpgroups x accumulator slots (see NSLOT).  Measured on B200: config 1 5x5 / 6x5 / 7x4 = 48.9 / 52.3 / 45.8 us (72 registers and no spills
        // at 7x4), config 3 244.6 / 236.9 / 291.7 us (7x4 spills there).  Below ~2^19 queries the shared slots lose 1-2 us (all warpgroups reach their
        // first MMA together and queue for the slots; there is no steady state to amortise it), so small batches keep one slot per warpgroup.
        const bool shared_slots = (Q.n + kRows - 1) / kRows >= 4096;
        if (T.n_levels == 4 && T.F == 8 && M.n_hidden == 3 && M.k1 == 48 && Q.n_extra == 0)
            return shared_slots ? launch_tm_spec<4, 8, 7, false, DBG, 3, 48, 0, 4>(T, M, Q, rgb, n_sms, 32, stream)
                                : launch_tm_spec<4, 8, 5, false, DBG, 3, 48, 0>(T, M, Q, rgb, n_sms, 96, stream);
        if (T.n_levels == 4 && T.F == 8 && M.n_hidden == 3 && M.k1 == 48 && Q.n_extra == 1)
            return shared_slots ? launch_tm_spec<4, 8, 7, false, DBG, 3, 48, 1, 4>(T, M, Q, rgb, n_sms, 32, stream)
                                : launch_tm_spec<4, 8, 5, false, DBG, 3, 48, 1>(T, M, Q, rgb, n_sms, 96, stream);
        if (T.n_levels == 5 && T.F == 16 && M.n_hidden == 4 && M.k1 == 96 && Q.n_extra == 0)
            return shared_slots ? launch_tm_spec<5, 16, 6, true, DBG, 4, 96, 0, 5>(T, M, Q, rgb, n_sms, 32, stream)
                                : launch_tm_spec<5, 16, 5, true, DBG, 4, 96, 0>(T, M, Q, rgb, n_sms, 96, stream);
    }
    if (ks_applies(T, M)) {      // 96 columns per tile: five warpgroups
        const int n = pipe ? launch_tm_variant<5, true, true, DBG>(T, M, Q, rgb, n_sms, 96, stream)
                           : launch_tm_variant<5, false, true, DBG>(T, M, Q, rgb, n_sms, 96, stream);
        if (n != -1) return n;
    }
    const uint32_t wg_cols = 64 + (M.k1 / 2 > 32 ? M.k1 / 2 : 32);
    if (5 * wg_cols <= 512) {
        if (pipe) {
            const int n = launch_tm_variant<5, true, false, DBG>(T, M, Q, rgb, n_sms, wg_cols, stream);
            if (n != -1) return n;
        }
        return launch_tm_variant<5, false, false, DBG>(T, M, Q, rgb, n_sms, wg_cols, stream);
    }
    if (4 * wg_cols <= 512) {
        if (pipe) {
            const int n = launch_tm_variant<4, true, false, DBG>(T, M, Q, rgb, n_sms, wg_cols, stream);
            if (n != -1) return n;
        }
        return launch_tm_variant<4, false, false, DBG>(T, M, Q, rgb, n_sms, wg_cols, stream);
    }
    return -1;
}

}  // namespace oo
