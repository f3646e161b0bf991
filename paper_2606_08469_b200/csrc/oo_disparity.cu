// oo_disparity.cu — the disparity predictor g_psi of Eq. 7 in one launch: multi-resolution hash-grid
// encoding of the position (trilinear over the eight vertices of the containing cell, per level) -> [e(x) | w_r] -> a
// 2 x 64 ReLU MLP on tcgen05 -> d^ = exp(z).  Readings of what the paper leaves open: DESIGN.md §14 (A25-A30).
//
// Structure = oo_fused_tm.cu's: one persistent block per SM, 5 warpgroups, a warpgroup owns a 128-query tile, thread = row =
// TMEM lane.  The A operand of every layer lives in tensor memory (two halves per 32-bit column), the weight image
// (UMMA K-major canonical layout) in shared memory, D in TMEM; the epilogue of a layer writes the next layer's A over
// columns of D it has already read.  TMEM columns of one warpgroup (stride 96):
//   even layer:  A at [64, 64 + K/2)   D at [0, 64)
//   odd  layer:  A at [0, 32)          D at [32, 96)
// Gather: per level 8 independent 4-byte loads (one entry = two fp16 features); the tables of the default predictor
// total 3 MB and stay in L2, so the phase is bound by load issue and latency, not by HBM.
#include <cstdio>
#include <type_traits>

#include "oo_device.cuh"
#include "oo_full.cuh"
#include "oo_tc_ptx.cuh"

namespace oo {

namespace {
constexpr int kRows = 128;
constexpr int kNWG = 5;
constexpr uint32_t kWgCols = 96;
constexpr uint32_t kPrimeY = 2654435761u, kPrimeZ = 805459861u;

__device__ __forceinline__ void relu_pack32(const uint32_t (&r)[32], uint32_t (&p)[16]) {
#pragma unroll
    for (int c = 0; c < 16; ++c) p[c] = pack_half2_relu(__uint_as_float(r[2 * c]), __uint_as_float(r[2 * c + 1]));
}

// One level of the hash grid at position x (already clamped to [0,1]^3).  The cell decision is taken in fp32 exactly as
// DESIGN.md §14 states it: p = fl(x * N), c0 = min(floor(p), N - 1), t = p - c0 (exact).
template <bool HASHED>
__device__ __forceinline__ void grid_level(const GridLevel& lv, const float (&x)[3], float& f0, float& f1) {
    uint32_t c[3];
    float t[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float p = __fmul_rn(x[a], lv.scale);
        const float fl = fminf(floorf(p), (float)lv.n_max);
        c[a] = (uint32_t)fl;
        t[a] = __fsub_rn(p, fl);
    }
    uint32_t ix[2], iy[2], iz[2], idx[8];
    ix[0] = c[0];
    ix[1] = c[0] + 1;
    if constexpr (HASHED) {        // hashed level: xor of the per-axis products (mod 2^32), reduced to the table
        iy[0] = c[1] * kPrimeY;
        iy[1] = iy[0] + kPrimeY;
        iz[0] = c[2] * kPrimeZ;
        iz[1] = iz[0] + kPrimeZ;
#pragma unroll
        for (int k = 0; k < 8; ++k) idx[k] = (ix[k & 1] ^ iy[(k >> 1) & 1] ^ iz[k >> 2]) & lv.mask;
    } else {                       // dense level: vertex (i,j,k) owns entry i + (N+1)(j + (N+1)k)
        iy[0] = c[1] * lv.stride;
        iy[1] = iy[0] + lv.stride;
        iz[0] = c[2] * lv.stride * lv.stride;
        iz[1] = iz[0] + lv.stride * lv.stride;
#pragma unroll
        for (int k = 0; k < 8; ++k) idx[k] = ix[k & 1] + iy[(k >> 1) & 1] + iz[k >> 2];
    }
    uint32_t v[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = __ldg(lv.table + idx[k]);
    const float wx[2] = {1.0f - t[0], t[0]}, wy[2] = {1.0f - t[1], t[1]}, wz[2] = {1.0f - t[2], t[2]};
    f0 = 0.0f;
    f1 = 0.0f;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const float w = wx[k & 1] * wy[(k >> 1) & 1] * wz[k >> 2];
        const float2 e = __half22float2(*reinterpret_cast<const __half2*>(&v[k]));
        f0 = fmaf(w, e.x, f0);
        f1 = fmaf(w, e.y, f1);
    }
}
}  // namespace

__global__ void __launch_bounds__(kNWG * 128, 1) disparity_kernel(const __grid_constant__ GridParams G, const __grid_constant__ MlpParams M,
                                                                   const __grid_constant__ QueryParams Q, float* __restrict__ disparity,
                                                                   float* __restrict__ features, uint32_t n_tiles) {
    extern __shared__ __align__(128) uint8_t smem[];
    uint8_t* s_w = smem;
    uint64_t* s_bar = (uint64_t*)(s_w + ((M.image_tc_bytes + 127) & ~127u));
    uint32_t* s_tmem = (uint32_t*)(s_bar + kNWG);

    const uint32_t wg = threadIdx.x >> 7, row = threadIdx.x & 127, warp = threadIdx.x >> 5;
    stage_to_smem(s_w, M.image_tc, M.image_tc_bytes);
    if (threadIdx.x < kNWG) mbar_init(smem_u32(&s_bar[threadIdx.x]), 1);
    if (threadIdx.x == 0) asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if (warp == 0) {
        tmem_alloc(smem_u32(s_tmem), 512);
        tmem_relinquish();
    }
    fence_async_smem();          // the weight image was written with generic stores and is read by the tensor core
    fence_before_sync();
    __syncthreads();
    fence_after_sync();
    const uint32_t tmem_wg = *s_tmem + wg * kWgCols;
    const uint32_t tmem_lane = tmem_wg + ((row & ~31u) << 16);
    const uint32_t w_addr = smem_u32(s_w), bar = smem_u32(&s_bar[wg]);
    uint32_t phase = 0;
    const bool leader_warp = row < 32;
    constexpr uint32_t idesc_h = instr_desc(128, 64), idesc_o = instr_desc(128, 16);
    const uint32_t n_lv = G.n_levels;

    for (uint32_t tile = wg * gridDim.x + blockIdx.x; tile < n_tiles; tile += gridDim.x * kNWG) {
        const uint64_t t = (uint64_t)tile * kRows + row;
        const bool valid = t < Q.n;
        const uint64_t qi = valid ? t : Q.n - 1;
        float x[3], n[3], wo[3], wr[3];
        load3(Q.x, qi, x);
        load3(Q.nrm, qi, n);
        load3(Q.wo, qi, wo);
#pragma unroll
        for (int a = 0; a < 3; ++a) x[a] = fminf(fmaxf(x[a], 0.0f), 1.0f);      // A16
        mirror_dir(n, wo, wr);
        // ------------------------------------------------------------------ hash-grid features -> A0 (even layer: columns 64..)
        const uint32_t a0 = tmem_lane + 64;
        // Levels in batches of 4, 2, 1 within the dense prefix and within the hashed rest: all loads of a batch are issued
        // before its first TMEM store (whose asm statement orders memory operations and would otherwise serialise the
        // levels), and a batch has no branch on the level kind.
        auto batch = [&](auto hashed, auto nb, uint32_t g0) {
            constexpr uint32_t NB = decltype(nb)::value;
            float f0[NB], f1[NB];
#pragma unroll
            for (uint32_t b = 0; b < NB; ++b) grid_level<decltype(hashed)::value>(G.lv[g0 + b], x, f0[b], f1[b]);
#pragma unroll
            for (uint32_t b = 0; b < NB; ++b) {
                tmem_st1(a0 + g0 + b, pack_half2(f0[b], f1[b]));
                if (features && valid) {
                    features[qi * (2 * n_lv) + 2 * (g0 + b)] = f0[b];
                    features[qi * (2 * n_lv) + 2 * (g0 + b) + 1] = f1[b];
                }
            }
        };
        auto span = [&](auto hashed, uint32_t g, uint32_t end) {
            for (; g + 4 <= end; g += 4) batch(hashed, std::integral_constant<uint32_t, 4>{}, g);
            if (g + 2 <= end) { batch(hashed, std::integral_constant<uint32_t, 2>{}, g); g += 2; }
            if (g < end) batch(hashed, std::integral_constant<uint32_t, 1>{}, g);
        };
        if (G.n_dense <= n_lv) {                      // dense levels first, hashed after (any increasing resolution schedule)
            span(std::false_type{}, 0u, G.n_dense);
            span(std::true_type{}, G.n_dense, n_lv);
        } else {                                      // arbitrary order: one level at a time
            for (uint32_t g = 0; g < n_lv; ++g) {
                if (G.lv[g].mask) batch(std::true_type{}, std::integral_constant<uint32_t, 1>{}, g);
                else batch(std::false_type{}, std::integral_constant<uint32_t, 1>{}, g);
            }
        }
        tmem_st1(a0 + n_lv, pack_half2(wr[0], wr[1]));
        tmem_st1(a0 + n_lv + 1, pack_half2(wr[2], 0.0f));
        for (uint32_t c = n_lv + 2; c < M.k1 / 2; ++c) tmem_st1(a0 + c, 0u);
        // ------------------------------------------------------------------ hidden layers
        uint32_t w_off = 0;
        for (uint32_t layer = 0; layer < M.n_hidden; ++layer) {
            const uint32_t kt_n = (layer == 0 ? M.k1 : 64u) >> 4;
            const bool odd = layer & 1u;
            // operand addresses formed by the issuing warp ahead of the barrier (see oo_fused_tm.cuh)
            uint32_t mma_d = tmem_wg + (odd ? 32u : 0u), mma_a = tmem_wg + (odd ? 0u : 64u);
            uint64_t mma_b = smem_desc(w_addr + w_off, 1024, 128);
            if (leader_warp) asm volatile("" : "+r"(mma_d), "+r"(mma_a), "+l"(mma_b));
            tmem_wait_st();
            fence_before_sync();
            named_bar(1 + wg, 128);
            if (leader_warp) {
                fence_after_sync();
                umma_group_ts<4>(mma_d, mma_a, mma_b, 2048 >> 4, idesc_h, kt_n, bar);
            }
            w_off += kt_n * 2 * 1024;
            mbar_wait(bar, phase);
            phase ^= 1;
            fence_after_sync();
            uint32_t r[32], p[16];
            if (!odd) {
                tmem_ld32(tmem_lane, r);
                tmem_wait_ld();
                relu_pack32(r, p);
                tmem_st16(tmem_lane, p);
                tmem_ld32(tmem_lane + 32, r);
                tmem_wait_ld();
                relu_pack32(r, p);
                tmem_st16(tmem_lane + 16, p);
            } else {
                tmem_ld32(tmem_lane + 64, r);
                tmem_wait_ld();
                relu_pack32(r, p);
                tmem_st16(tmem_lane + 80, p);
                tmem_ld32(tmem_lane + 32, r);
                tmem_wait_ld();
                relu_pack32(r, p);
                tmem_st16(tmem_lane + 64, p);
            }
        }
        // ------------------------------------------------------------------ output layer (N = 16 rows of which one is real)
        const bool odd = M.n_hidden & 1u;
        uint32_t out_d = tmem_wg + (odd ? 32u : 0u), out_a = tmem_wg + (odd ? 0u : 64u);
        uint64_t out_b = smem_desc(w_addr + w_off, 256, 128);
        if (leader_warp) asm volatile("" : "+r"(out_d), "+r"(out_a), "+l"(out_b));
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
        uint32_t o[4];
        tmem_ld4(tmem_lane + (odd ? 32u : 0u), o);
        tmem_wait_ld();
        if (valid) disparity[qi] = fast_exp(__uint_as_float(o[0]));
        // the next tile's A0 stores land in columns this tile's output MMA has finished reading (the commit covers it)
    }
    fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem_dealloc(*s_tmem, 512);
}

int launch_disparity(const GridParams& G, const MlpParams& M, const QueryParams& Q, float* disparity, float* features, int n_sms,
                     cudaStream_t stream) {
    if (Q.n == 0) return 0;
    if (!M.image_tc || M.k1 > 64 || M.out_dim != 1 || M.width != 64 || 2 * G.n_levels + 3 != M.in_dim) return -1;
    const uint64_t n_tiles = (Q.n + kRows - 1) / kRows;
    const uint64_t blocks = (n_tiles + kNWG - 1) / kNWG;
    const unsigned grid = (unsigned)(blocks < (uint64_t)n_sms ? blocks : (uint64_t)n_sms);
    const uint32_t smem = ((M.image_tc_bytes + 127) & ~127u) + 128;
    if (smem > 64 * 1024) return -1;
    static std::atomic<uint64_t> opted{0};
    if (!opt_in_smem(opted, (const void*)disparity_kernel, 64 * 1024)) return kLaunchCudaError;
    disparity_kernel<<<grid, kNWG * 128, smem, stream>>>(G, M, Q, disparity, features, (uint32_t)n_tiles);
    return 1;
}

}  // namespace oo
