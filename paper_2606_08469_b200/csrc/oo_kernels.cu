// oo_kernels.cu — CUDA kernels of liboo (sm_100a): atlas border padding, encode (generic + specialised), the
// stand-alone MLP kernel, and the fused encode+MLP kernel on mma.sync tiles.  The tcgen05 variant is in oo_fused_tc.cu.
#include "oo_device.cuh"

namespace oo {

// =====================================================================================================================
// Upload-time re-layout: dst[slot][jj][ii] = src[slot][wrap(jj-1, ii-1)] for jj, ii in [0, R+2).  a5: a tap
// outside the map continues on the neighbouring octahedron face = point reflection about the crossed edge's midpoint.
// One thread per 16-byte vector of the destination.
// =====================================================================================================================
__global__ void pad_atlas_kernel(const uint4* __restrict__ src, uint4* __restrict__ dst, uint64_t slots, uint32_t R,
                                 uint32_t vec_per_texel) {
    const uint32_t Rp = R + 2;
    const uint64_t per_map = (uint64_t)Rp * Rp * vec_per_texel;
    const uint64_t total = slots * per_map;
    for (uint64_t t = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; t < total; t += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t slot = t / per_map;
        uint32_t r = (uint32_t)(t - slot * per_map);
        const uint32_t v = r % vec_per_texel;
        r /= vec_per_texel;
        int i = (int)(r % Rp) - 1, j = (int)(r / Rp) - 1;
        const int Ri = (int)R;
        if (i < 0) { i = 0; j = Ri - 1 - j; } else if (i >= Ri) { i = Ri - 1; j = Ri - 1 - j; }
        if (j < 0) { j = 0; i = Ri - 1 - i; } else if (j >= Ri) { j = Ri - 1; i = Ri - 1 - i; }
        dst[t] = src[((slot * R + (uint32_t)j) * R + (uint32_t)i) * vec_per_texel + v];
    }
}

int launch_pad_atlas(const void* src, void* dst, uint64_t slots, uint32_t R, uint32_t texel_bytes, cudaStream_t stream) {
    if (slots == 0) return 0;
    const uint32_t vpt = texel_bytes / 16;
    const uint64_t total = slots * (uint64_t)(R + 2) * (R + 2) * vpt;
    const uint64_t blocks = (total + 255) / 256;
    const unsigned grid = (unsigned)(blocks < 148ull * 32 ? blocks : 148ull * 32);
    pad_atlas_kernel<<<grid, 256, 0, stream>>>((const uint4*)src, (uint4*)dst, slots, R, vpt);
    return 1;
}

// =====================================================================================================================
// Upload-time tying of vertex-stored maps (f2, P:125 / Fig. 3 caption: "the edge vertices are shared along adjacent faces").
// On the unfolded octahedron the outer edge of the (R+1) x (R+1) vertex grid is the four lower-hemisphere face edges met
// twice, mirrored about each side's midpoint, and the four corners are all the -z pole: stored vertices (0, c) and (0, R-c),
// (R, c) and (R, R-c), (r, 0) and (R-r, 0), (r, R) and (R-r, R) are one vertex each.  The library's copy gives every such
// pair the value of the member with the smaller index along its side (the corners that of vertex (0, 0)), so that the
// barycentric interpolant is continuous across the seam whatever the owner stored; *changed counts the vertices rewritten.
// One thread per boundary vertex of one map.
// =====================================================================================================================
__global__ void tie_vertex_borders_kernel(uint4* __restrict__ maps, uint64_t slots, uint32_t R, uint32_t vec_per_texel,
                                          unsigned long long* __restrict__ changed) {
    const uint32_t n = R, Rp = R + 1;
    const uint64_t total = slots * 4ull * n;
    for (uint64_t t = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; t < total; t += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t slot = t / (4ull * n);
        const uint32_t b = (uint32_t)(t - slot * 4ull * n), e = b / n, i = b - e * n;
        // the 4n boundary vertices, each once: side 0 (0, i), side 1 (i, n), side 2 (n, n - i), side 3 (n - i, 0), i = 0..n-1
        const uint32_t r = e == 0 ? 0u : e == 1 ? i : e == 2 ? n : n - i;
        const uint32_t c = e == 0 ? i : e == 1 ? n : e == 2 ? n - i : 0u;
        uint32_t sr = r, sc = c;
        const bool corner = (r == 0 || r == n) && (c == 0 || c == n);
        if (corner) { sr = 0; sc = 0; }
        else if ((r == 0 || r == n) && 2 * c > n) sc = n - c;
        else if ((c == 0 || c == n) && 2 * r > n) sr = n - r;
        if (sr == r && sc == c) continue;
        uint4* dst = maps + ((slot * Rp + r) * Rp + c) * vec_per_texel;
        const uint4* src = maps + ((slot * Rp + sr) * Rp + sc) * vec_per_texel;
        bool diff = false;
        for (uint32_t v = 0; v < vec_per_texel; ++v) {
            const uint4 a = src[v], o = dst[v];
            diff |= (a.x != o.x) | (a.y != o.y) | (a.z != o.z) | (a.w != o.w);
            dst[v] = a;
        }
        if (diff) atomicAdd(changed, 1ull);
    }
}

int launch_tie_vertex_borders(void* maps, uint64_t slots, uint32_t R, uint32_t texel_bytes, unsigned long long* changed, cudaStream_t stream) {
    if (slots == 0) return 0;
    const uint64_t total = slots * 4ull * R;
    const uint64_t blocks = (total + 255) / 256;
    const unsigned grid = (unsigned)(blocks < 148ull * 32 ? blocks : 148ull * 32);
    tie_vertex_borders_kernel<<<grid, 256, 0, stream>>>((uint4*)maps, slots, R, texel_bytes / 16, changed);
    return 1;
}

// =====================================================================================================================
// Generic encode: any tree, any (F, dtype) with 16/32/64-byte texels.  Plain child-table descent per level.
// One thread per query.  Slow by design; it is the fallback and a cross-check of the specialised kernels.
// =====================================================================================================================
__global__ void __launch_bounds__(256) encode_generic_kernel(const __grid_constant__ TreeParams T,
                                                             const __grid_constant__ QueryParams Q,
                                                             const __grid_constant__ EncodeOut O, uint32_t tree_depth) {
    const uint64_t t = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x;
    if (t >= Q.n) return;
    const uint64_t qi = Q.perm ? Q.perm[t] : t;
    const uint64_t oi = Q.out_idx ? Q.out_idx[t] : qi;          // where this query's rows go (binned queries: its own index)
    float x[3], w[3];
    load3(Q.x, qi, x);
    load3(Q.wo, qi, w);
    const float scale = (float)(1u << tree_depth);
    const int qmax = (int)(1u << tree_depth) - 1;
    const int qx = quantise(x[0], scale, qmax), qy = quantise(x[1], scale, qmax), qz = quantise(x[2], scale, qmax);
    const OctaUV uv = octa_project(w[0], w[1], w[2]);
    const uint32_t L = T.n_levels, F = T.F, LF = L * F;
    for (uint32_t l = 0; l < L; ++l) {
        const LevelParams& lv = T.lv[l];
        const int node = descend_plain(T.child, qx, qy, qz, (int)tree_depth, (int)lv.depth);
        const int slot = node >= 0 ? __ldg(T.map_slot + node) : -1;
        const Tap tp = level_tap(uv, lv.half_r, lv.off);
        if (O.slot) O.slot[oi * L + l] = slot;
        if (O.texel) {
            O.texel[(oi * L + l) * 2] = (int16_t)tp.i0;
            O.texel[(oi * L + l) * 2 + 1] = (int16_t)tp.j0;
        }
        if (!O.features) continue;
        const float w00 = (1.0f - tp.fx) * (1.0f - tp.fy), w10 = tp.fx * (1.0f - tp.fy), w01 = (1.0f - tp.fx) * tp.fy,
                    w11 = tp.fx * tp.fy;
        const uint8_t* p = nullptr;
        if (slot >= 0)
            p = lv.atlas + (uint64_t)slot * lv.map_bytes + (int64_t)((tp.j0 * (int)lv.Rp + tp.i0) * (int)T.texel_bytes);
        for (uint32_t c = 0; c < F; ++c) {
            float h = 0.0f;
            if (slot >= 0) {
                if (T.f32) {
                    const float* a = (const float*)p;
                    const float* b = (const float*)(p + lv.row_bytes);
                    h = fmaf(w00, a[c], h);
                    h = fmaf(w10, a[F + c], h);
                    h = fmaf(w01, b[c], h);
                    h = fmaf(w11, b[F + c], h);
                } else {
                    const __half* a = (const __half*)p;
                    const __half* b = (const __half*)(p + lv.row_bytes);
                    h = fmaf(w00, __half2float(a[c]), h);
                    h = fmaf(w10, __half2float(a[F + c]), h);
                    h = fmaf(w01, __half2float(b[c]), h);
                    h = fmaf(w11, __half2float(b[F + c]), h);
                }
            }
            if (T.f32) ((float*)O.features)[oi * LF + l * F + c] = h;
            else ((__half*)O.features)[oi * LF + l * F + c] = __float2half_rn(h);
        }
    }
}

int launch_encode_generic(const TreeParams& T, const QueryParams& Q, const EncodeOut& O, uint32_t tree_max_depth,
                          cudaStream_t stream) {
    if (Q.n == 0) return 0;
    const unsigned grid = (unsigned)((Q.n + 255) / 256);
    encode_generic_kernel<<<grid, 256, 0, stream>>>(T, Q, O, tree_max_depth);
    return 1;
}

// =====================================================================================================================
// Specialised encode (oo_encode fast path): hop-table descent, vector gathers, features written as 16-byte vectors.
// One thread per query; persistent-style grid-stride loop so the dense tables are staged once per block.
// =====================================================================================================================
template <int L, int F, bool F32>
__global__ void __launch_bounds__(256) encode_fast_kernel(const __grid_constant__ TreeParams T,
                                                          const __grid_constant__ QueryParams Q,
                                                          const __grid_constant__ EncodeOut O) {
    extern __shared__ __align__(16) uint8_t smem[];
    int32_t* s_dense = (int32_t*)smem;
    stage_to_smem(s_dense, T.dense, T.dense_ints * 4);
    __syncthreads();
    constexpr int TB = F * (F32 ? 4 : 2);
    bool sample = Q.stat != nullptr && threadIdx.x < 32;      // OO_PRESORT_AUTO: warp 0 of every block samples the first queries it takes
    for (uint64_t t = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; t < Q.n; t += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t qi = Q.perm ? Q.perm[t] : t;
        const uint64_t oi = Q.out_idx ? Q.out_idx[t] : qi;      // where this query's rows go (binned queries: its own index)
        float x[3], w[3];
        load3(Q.x, qi, x);
        load3(Q.wo, qi, w);
        if (sample) {
            if ((t | 31u) < Q.n) stat_sample_warp(Q, blockIdx.x, x[0], x[1], x[2]);    // warp-uniform: t | 31 is the warp's last query
            sample = false;
        }
        Encoded<L, F, F32> e;
        locate<L, F, F32>(T, s_dense, x, w, e);
#pragma unroll
        for (int l = 0; l < L; ++l) {
            const LevelParams& lv = T.lv[l];
            const Tap tp = level_tap(e.uv, lv.half_r, lv.off);
            if (O.slot) O.slot[oi * L + l] = e.slot[l];
            if (O.texel) {
                O.texel[(oi * L + l) * 2] = (int16_t)tp.i0;
                O.texel[(oi * L + l) * 2 + 1] = (int16_t)tp.j0;
            }
            if (O.features) {
                float h[F];
                gather_level<F, F32>(lv, e.slot[l], e.uv, h);
                uint8_t* dst = (uint8_t*)O.features + (oi * L + l) * TB;
                if constexpr (F32) {
#pragma unroll
                    for (int v = 0; v < F / 4; ++v)
                        ((float4*)dst)[v] = make_float4(h[4 * v], h[4 * v + 1], h[4 * v + 2], h[4 * v + 3]);
                } else {
#pragma unroll
                    for (int v = 0; v < F / 8; ++v)
                        ((uint4*)dst)[v] = make_uint4(pack_half2(h[8 * v], h[8 * v + 1]), pack_half2(h[8 * v + 2], h[8 * v + 3]),
                                                      pack_half2(h[8 * v + 4], h[8 * v + 5]), pack_half2(h[8 * v + 6], h[8 * v + 7]));
                }
            }
        }
    }
}

// The same encode for batches whose taps miss the caches (binned or incoherent queries): the fused kernel's pipelined descent
// (gather_pipelined: the hop chain overlaps the gathers, two or three levels of taps in flight per query) instead of one level
// at a time.  It costs registers, i.e. occupancy, which is what the kernel above lives on when the taps hit L1/L2 -- so the
// launcher picks per call: this one when the batch was binned or measured incoherent, the one above for coherent frames.
// Same taps, weights and accumulation order: bit-identical rows.
template <int L, int F, bool F32, bool IDX>
__global__ void __launch_bounds__(256) encode_pipe_kernel(const __grid_constant__ TreeParams T,
                                                          const __grid_constant__ QueryParams Q,
                                                          const __grid_constant__ EncodeOut O) {
    extern __shared__ __align__(16) uint8_t smem[];
    int32_t* s_dense = (int32_t*)smem;
    stage_to_smem(s_dense, T.dense, T.dense_ints * 4);
    __syncthreads();
    constexpr int TB = F * (F32 ? 4 : 2);
    bool sample = Q.stat != nullptr && threadIdx.x < 32;
    for (uint64_t t = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; t < Q.n; t += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t qi = Q.perm ? Q.perm[t] : t;
        const uint64_t oi = Q.out_idx ? Q.out_idx[t] : qi;
        float x[3], w[3];
        load3(Q.x, qi, x);
        load3(Q.wo, qi, w);
        if (sample) {
            if ((t | 31u) < Q.n) stat_sample_warp(Q, blockIdx.x, x[0], x[1], x[2]);
            sample = false;
        }
        typename DbgSel<IDX>::type dbg;          // IDX: the slot / base-texel rows are wanted too
        if constexpr (IDX) {
            dbg.slot = O.slot ? O.slot + oi * L : nullptr;
            dbg.texel = O.texel ? O.texel + oi * L * 2 : nullptr;
        }
        uint8_t* row = (uint8_t*)O.features + oi * L * TB;
        auto store = [&](int l, const float (&h)[F]) {
            if (!O.features) return;
            uint8_t* dst = row + l * TB;
            if constexpr (F32) {
#pragma unroll
                for (int v = 0; v < F / 4; ++v)
                    ((float4*)dst)[v] = make_float4(h[4 * v], h[4 * v + 1], h[4 * v + 2], h[4 * v + 3]);
            } else {
#pragma unroll
                for (int v = 0; v < F / 8; ++v)
                    ((uint4*)dst)[v] = make_uint4(pack_half2(h[8 * v], h[8 * v + 1]), pack_half2(h[8 * v + 2], h[8 * v + 3]),
                                                  pack_half2(h[8 * v + 4], h[8 * v + 5]), pack_half2(h[8 * v + 6], h[8 * v + 7]));
            }
        };
        gather_pipelined<L, F, F32>(T, s_dense, x, w, store, dbg);
    }
}

// =====================================================================================================================
// MLP input row: [h (L*F) | n | wo | extra | 0-pad] as fp16 in shared memory, row stride (k1 + 8) halves.
// The tail (attributes + padding) is written 16 bytes at a time starting at column feat_dim (a multiple of 8).
// =====================================================================================================================
__device__ __forceinline__ void write_row_tail(uint8_t* row, uint32_t feat_dim, uint32_t k1, const float (&n)[3],
                                               const float (&w)[3], const float* __restrict__ extra, uint64_t qi,
                                               uint32_t n_extra) {
    float v[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = 0.0f;
    v[0] = n[0]; v[1] = n[1]; v[2] = n[2];
    v[3] = w[0]; v[4] = w[1]; v[5] = w[2];
#pragma unroll
    for (int k = 0; k < OO_MAX_EXTRA; ++k)
        if ((uint32_t)k < n_extra) v[6 + k] = __ldg(extra + qi * n_extra + k);
    uint4* dst = (uint4*)(row + feat_dim * 2);
    dst[0] = make_uint4(pack_half2(v[0], v[1]), pack_half2(v[2], v[3]), pack_half2(v[4], v[5]), pack_half2(v[6], v[7]));
    if (k1 - feat_dim > 8)
        dst[1] = make_uint4(pack_half2(v[8], v[9]), pack_half2(v[10], v[11]), pack_half2(v[12], v[13]), pack_half2(v[14], v[15]));
    if (k1 - feat_dim > 16) dst[2] = make_uint4(0, 0, 0, 0);
}

// the same when feat_dim = 4 mod 8 (F = 4 fp32 with an odd level count): the tail starts mid-vector; halves one by one
__device__ __forceinline__ void write_row_tail_odd(uint8_t* row, uint32_t feat_dim, uint32_t k1, const float (&n)[3],
                                                   const float (&w)[3], const float* __restrict__ extra, uint64_t qi,
                                                   uint32_t n_extra) {
    __half* r = (__half*)row;
    for (uint32_t c = feat_dim; c < k1; ++c) r[c] = __float2half_rn(0.0f);
    for (int k = 0; k < 3; ++k) { r[feat_dim + k] = __float2half_rn(n[k]); r[feat_dim + 3 + k] = __float2half_rn(w[k]); }
    for (uint32_t k = 0; k < n_extra; ++k) r[feat_dim + 6 + k] = __float2half_rn(__ldg(extra + qi * n_extra + k));
}

// rgb of the warp's 32 rows: C fragments -> shared scratch -> one row per lane -> activation -> store at the query's index
__device__ __forceinline__ void store_rgb(float* s_out /* [32][8] floats, warp private */, const float (&out)[2][4],
                                          float* __restrict__ rgb, uint64_t qi, bool valid, uint32_t out_dim, uint32_t act) {
    const uint32_t lane = threadIdx.x & 31;
#pragma unroll
    for (int m = 0; m < 2; ++m) {
        const uint32_t r = m * 16 + (lane >> 2), c = (lane & 3) * 2;
        *(float2*)(s_out + r * 8 + c) = make_float2(out[m][0], out[m][1]);
        *(float2*)(s_out + (r + 8) * 8 + c) = make_float2(out[m][2], out[m][3]);
    }
    __syncwarp();
    if (valid) {
        for (uint32_t c = 0; c < out_dim; ++c) {
            float z = s_out[lane * 8 + c];
            rgb[qi * out_dim + c] = act == OO_ACT_EXP ? fast_exp(z) : z;
        }
    }
    __syncwarp();
}

// =====================================================================================================================
// Stand-alone MLP over feature rows in HBM (the unfused baseline): one warp per 32 queries.
// =====================================================================================================================
constexpr int kMlpThreads = 256;

__global__ void __launch_bounds__(kMlpThreads, 2) mlp_rows_kernel(const __grid_constant__ MlpParams M,
                                                                  const __grid_constant__ QueryParams Q,
                                                                  const void* __restrict__ features, uint32_t f32,
                                                                  float* __restrict__ rgb, uint32_t n_tiles) {
    extern __shared__ __align__(16) uint8_t smem[];
    uint8_t* s_w = smem;
    const uint32_t a_stride = (M.k1 + 8) * 2;
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint8_t* s_a = smem + M.image_bytes + warp * 32 * a_stride;
    stage_to_smem(s_w, M.image, M.image_bytes);
    __syncthreads();
    const uint32_t warps = kMlpThreads / 32;
    for (uint32_t tile = blockIdx.x * warps + warp; tile < n_tiles; tile += gridDim.x * warps) {
        const uint64_t t = (uint64_t)tile * 32 + lane;
        const bool valid = t < Q.n;
        const uint64_t tt = valid ? t : Q.n - 1;
        const uint64_t qi = Q.perm ? Q.perm[tt] : tt;
        float n[3], w[3];
        load3(Q.nrm, qi, n);
        load3(Q.wo, qi, w);
        uint8_t* row = s_a + lane * a_stride;
        const uint32_t fd = M.feat_dim;
        if (f32) {
            const float4* src = (const float4*)((const float*)features + qi * fd);
            for (uint32_t v = 0; v < fd / 8; ++v) {
                const float4 p = __ldg(src + 2 * v), q = __ldg(src + 2 * v + 1);
                ((uint4*)row)[v] = make_uint4(pack_half2(p.x, p.y), pack_half2(p.z, p.w), pack_half2(q.x, q.y), pack_half2(q.z, q.w));
            }
            if (fd & 4u) {     // odd number of 4-float levels: one more half vector
                const float4 p = __ldg(src + 2 * (fd / 8));
                *(uint2*)(row + (fd & ~7u) * 2) = make_uint2(pack_half2(p.x, p.y), pack_half2(p.z, p.w));
            }
        } else {
            const uint4* src = (const uint4*)((const __half*)features + qi * fd);
            for (uint32_t v = 0; v < fd / 8; ++v) ((uint4*)row)[v] = __ldg(src + v);
        }
        if (fd & 7u) write_row_tail_odd(row, fd, M.k1, n, w, Q.extra, qi, Q.n_extra);
        else write_row_tail(row, fd, M.k1, n, w, Q.extra, qi, Q.n_extra);
        __syncwarp();
        float out[2][4];
        warp_mlp(smem_u32(s_a), smem_u32(s_w), M.k1, M.n_hidden, out);
        __syncwarp();
        store_rgb((float*)s_a, out, rgb, qi, valid, M.out_dim, M.out_act);
    }
}

static uint32_t mlp_smem_bytes(const MlpParams& M, int threads) { return M.image_bytes + (threads / 32) * 32 * (M.k1 + 8) * 2; }

int launch_mlp_rows(const TreeParams& T, const MlpParams& M, const QueryParams& Q, const void* features, float* rgb,
                    int n_sms, cudaStream_t stream) {
    if (Q.n == 0) return 0;
    if (M.feat_dim % 4 != 0 || (M.feat_dim % 8 != 0 && !T.f32)) return -1;
    const uint32_t smem = mlp_smem_bytes(M, kMlpThreads);
    static std::atomic<uint64_t> opted{0};
    if (!opt_in_smem(opted, (const void*)mlp_rows_kernel, 200 * 1024)) return kLaunchCudaError;
    const uint64_t n_tiles = (Q.n + 31) / 32;
    const uint64_t blocks = (n_tiles + 7) / 8;
    const unsigned grid = (unsigned)(blocks < (uint64_t)n_sms * 2 ? blocks : (uint64_t)n_sms * 2);
    mlp_rows_kernel<<<grid, kMlpThreads, smem, stream>>>(M, Q, features, T.f32, rgb, (uint32_t)n_tiles);
    return 1;
}

// =====================================================================================================================
// Fused encode + MLP, mma.sync version.  Persistent blocks; every warp owns 32 queries end to end, so there is no
// block-level synchronisation inside the loop: gather (registers) -> fp16 row (shared memory, warp private) ->
// ldmatrix -> HMMA chain with register-resident activations -> RGB.  Features never touch HBM.
// =====================================================================================================================
constexpr int kFusedThreads = 256;

template <int L, int F, bool F32, bool DBG>
__global__ void __launch_bounds__(kFusedThreads, 2) fused_mma_kernel(const __grid_constant__ TreeParams T,
                                                                     const __grid_constant__ MlpParams M,
                                                                     const __grid_constant__ QueryParams Q,
                                                                     float* __restrict__ rgb, uint32_t n_tiles) {
    extern __shared__ __align__(16) uint8_t smem[];
    const uint32_t dense_bytes = (T.dense_ints * 4 + 15) & ~15u;
    int32_t* s_dense = (int32_t*)smem;
    uint8_t* s_w = smem + dense_bytes;
    const uint32_t a_stride = (M.k1 + 8) * 2;
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint8_t* s_a = s_w + M.image_bytes + warp * 32 * a_stride;
    stage_to_smem(s_dense, T.dense, T.dense_ints * 4);
    stage_to_smem(s_w, M.image, M.image_bytes);
    __syncthreads();
    constexpr uint32_t warps = kFusedThreads / 32;
    for (uint32_t tile = blockIdx.x * warps + warp; tile < n_tiles; tile += gridDim.x * warps) {
        const uint64_t t = (uint64_t)tile * 32 + lane;
        const bool valid = t < Q.n;
        const uint64_t tt = valid ? t : Q.n - 1;
        const uint64_t qi = Q.perm ? Q.perm[tt] : tt;
        float x[3], n[3], w[3];
        load3(Q.x, qi, x);
        load3(Q.nrm, qi, n);
        load3(Q.wo, qi, w);
        Encoded<L, F, F32> e;
        locate<L, F, F32>(T, s_dense, x, w, e);
        uint8_t* row = s_a + lane * a_stride;
        const auto dbg = make_dbg<DBG>(Q, L, Q.out_idx ? Q.out_idx[tt] : qi, valid);
#pragma unroll
        for (int l = 0; l < L; ++l) {
            const LevelParams& lv = T.lv[l];
            float h[F];
            gather_level<F, F32>(lv, e.slot[l], e.uv, h, dbg, l);
#pragma unroll
            for (int v = 0; v < F / 8 + (F % 8 ? 1 : 0); ++v) {
                if constexpr (F % 8 == 0) {
                    ((uint4*)(row + l * F * 2))[v] =
                        make_uint4(pack_half2(h[8 * v], h[8 * v + 1]), pack_half2(h[8 * v + 2], h[8 * v + 3]),
                                   pack_half2(h[8 * v + 4], h[8 * v + 5]), pack_half2(h[8 * v + 6], h[8 * v + 7]));
                } else {   // F == 4: 8-byte store
                    *(uint2*)(row + l * F * 2) = make_uint2(pack_half2(h[0], h[1]), pack_half2(h[2], h[3]));
                }
            }
        }
        if constexpr ((L * F) % 8 == 0) {
            write_row_tail(row, L * F, M.k1, n, w, Q.extra, qi, Q.n_extra);
        } else {   // L*F = 4 mod 8
            write_row_tail_odd(row, L * F, M.k1, n, w, Q.extra, qi, Q.n_extra);
        }
        __syncwarp();
        float out[2][4];
        warp_mlp(smem_u32(s_a), smem_u32(s_w), M.k1, M.n_hidden, out);
        __syncwarp();
        store_rgb((float*)s_a, out, rgb, qi, valid, M.out_dim, M.out_act);
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// Dispatch over the instantiated (L, F, dtype) shapes.
// ---------------------------------------------------------------------------------------------------------------------
// encode_fast_kernel (and with it OO_PATH_UNFUSED and the gate of every specialised path): every L up to OO_MAX_LEVELS for the
// three texel formats the configs and the paper use (fp16 F = 8 / 16, fp32 F = 4)
#define OO_SHAPES(X)                                                                                       \
    X(1, 8, false) X(2, 8, false) X(3, 8, false) X(4, 8, false) X(5, 8, false) X(6, 8, false) X(7, 8, false) X(8, 8, false)         \
    X(1, 16, false) X(2, 16, false) X(3, 16, false) X(4, 16, false) X(5, 16, false) X(6, 16, false) X(7, 16, false) X(8, 16, false) \
    X(1, 4, true) X(2, 4, true) X(3, 4, true) X(4, 4, true) X(5, 4, true) X(6, 4, true) X(7, 4, true) X(8, 4, true)
// fused_mma_kernel (the mma.sync fallback): the BASELINE.json shapes; other shapes fall through to OO_PATH_UNFUSED
#define OO_MMA_SHAPES(X)                                                                                   \
    X(1, 8, false) X(2, 8, false) X(3, 8, false) X(4, 8, false) X(5, 8, false)                             \
    X(2, 16, false) X(3, 16, false) X(4, 16, false) X(5, 16, false)                                        \
    X(1, 4, true) X(2, 4, true) X(3, 4, true) X(4, 4, true)

bool fast_shape_supported(uint32_t L, uint32_t F, bool f32) {
#define X(l, f, t) if (L == l && F == f && f32 == t) return true;
    OO_SHAPES(X)
#undef X
    return false;
}

// the shapes of the pipelined descent (pipe_applies: fp16 trees, two dense levels, then hops)
#define OO_ENC_PIPE_SHAPES(X)                                                                          \
    X(3, 8, false) X(4, 8, false) X(5, 8, false) X(6, 8, false) X(7, 8, false) X(8, 8, false)          \
    X(3, 16, false) X(4, 16, false) X(5, 16, false) X(6, 16, false) X(7, 16, false) X(8, 16, false)

// cache_cold: the batch was binned, or measured incoherent (OO_PRESORT_AUTO's samples): its taps miss L1/L2
int launch_encode_fast(const TreeParams& T, const QueryParams& Q, const EncodeOut& O, int n_sms, cudaStream_t stream, bool cache_cold, bool* pipelined) {
    if (pipelined) *pipelined = false;
    if (Q.n == 0) return 0;
    const uint32_t smem = T.dense_ints * 4;
    const uint64_t blocks = (Q.n + 255) / 256;
    const unsigned grid = (unsigned)(blocks < (uint64_t)n_sms * 8 ? blocks : (uint64_t)n_sms * 8);
    if (cache_cold && pipe_applies(T)) {
#define X(l, f, t)                                                                          \
    if (T.n_levels == l && T.F == f && (T.f32 != 0) == t) {                                 \
        if (O.slot || O.texel) encode_pipe_kernel<l, f, t, true><<<grid, 256, smem, stream>>>(T, Q, O);   \
        else encode_pipe_kernel<l, f, t, false><<<grid, 256, smem, stream>>>(T, Q, O);      \
        if (pipelined) *pipelined = true;                                                   \
        return 1;                                                                           \
    }
        OO_ENC_PIPE_SHAPES(X)
#undef X
    }
#define X(l, f, t)                                                                          \
    if (T.n_levels == l && T.F == f && (T.f32 != 0) == t) {                                 \
        encode_fast_kernel<l, f, t><<<grid, 256, smem, stream>>>(T, Q, O);                  \
        return 1;                                                                           \
    }
    OO_SHAPES(X)
#undef X
    return -1;
}

template <bool DBG>
static int launch_fused_mma_impl(const TreeParams& T, const MlpParams& M, const QueryParams& Q, float* rgb, int n_sms,
                                 cudaStream_t stream) {
    if (Q.n == 0) return 0;
    const uint32_t smem = ((T.dense_ints * 4 + 15) & ~15u) + mlp_smem_bytes(M, kFusedThreads);
    const uint64_t n_tiles = (Q.n + 31) / 32;
    const uint64_t blocks = (n_tiles + 7) / 8;
    const unsigned grid = (unsigned)(blocks < (uint64_t)n_sms * 2 ? blocks : (uint64_t)n_sms * 2);
#define X(l, f, t)                                                                                                   \
    if (T.n_levels == l && T.F == f && (T.f32 != 0) == t) {                                                          \
        static std::atomic<uint64_t> opted{0};                                                                       \
        if (!opt_in_smem(opted, (const void*)fused_mma_kernel<l, f, t, DBG>, 200 * 1024)) return kLaunchCudaError;   \
        fused_mma_kernel<l, f, t, DBG><<<grid, kFusedThreads, smem, stream>>>(T, M, Q, rgb, (uint32_t)n_tiles);      \
        return 1;                                                                                                    \
    }
    OO_MMA_SHAPES(X)
#undef X
    return -1;
}

// dbg: the instances with the index sink compiled in (oo_query_debug)
int launch_fused_mma(const TreeParams& T, const MlpParams& M, const QueryParams& Q, float* rgb, int n_sms, cudaStream_t stream, bool dbg) {
    return dbg ? launch_fused_mma_impl<true>(T, M, Q, rgb, n_sms, stream) : launch_fused_mma_impl<false>(T, M, Q, rgb, n_sms, stream);
}

}  // namespace oo
