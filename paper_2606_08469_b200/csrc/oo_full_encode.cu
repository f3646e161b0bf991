// oo_full_encode.cu — oo_encode_full: steps 1-3 of the paper's full query (oo_full.cuh), features written to HBM as fp32
// with the per-neighbour slot and directional index decisions as debug outputs.  One thread per query; runtime level count.
#include "oo_full.cuh"

namespace oo {

template <int F, bool F32, bool VERTEX, bool TRI8, bool SHIFTED>
__global__ void __launch_bounds__(256) encode_full_kernel(const __grid_constant__ TreeParams T,
                                                          const __grid_constant__ QueryParams Q,
                                                          const __grid_constant__ FullMode mode, float* __restrict__ features,
                                                          int32_t* __restrict__ d_slot, int16_t* __restrict__ d_cell) {
    extern __shared__ __align__(16) uint8_t smem[];
    int32_t* s_dense = (int32_t*)smem;
    stage_to_smem(s_dense, T.dense, T.dense_ints * 4);
    __syncthreads();
    constexpr int NJ = TRI8 ? 8 : 1;
    const uint32_t L = T.n_levels;
    for (uint64_t t = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; t < Q.n; t += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t qi = Q.perm ? Q.perm[t] : t;
        float x[3], w[3], wl[3];
        load3(Q.x, qi, x);
        load3(Q.wo, qi, w);
        if (mode.lookup == OO_LOOKUP_WO) {
#pragma unroll
            for (int a = 0; a < 3; ++a) wl[a] = w[a];
        } else {
            float n[3];
            load3(Q.nrm, qi, n);
            mirror_dir(n, w, wl);
        }
        const float disp = SHIFTED ? __ldg(Q.disparity + qi) : 0.0f;
        OctaUV uv{0.0f, 0.0f};
        if constexpr (!SHIFTED) uv = octa_project(wl[0], wl[1], wl[2]);
        Station<NJ> st;
        station_init<NJ>(T, s_dense, x, st);
        FullDebug dbg{d_slot ? d_slot + qi * L * NJ : nullptr, d_cell ? d_cell + qi * L * NJ * 3 : nullptr};
        for (uint32_t l = 0; l < L; ++l) {
            float h[F];
            full_level<F, F32, VERTEX, TRI8, SHIFTED>(T.lv[l], s_dense, x, wl, uv, disp, st, true, h, (int)l, dbg);
            if (features) {
                float4* dst = (float4*)(features + (qi * L + l) * F);
#pragma unroll
                for (int v = 0; v < F / 4; ++v) dst[v] = make_float4(h[4 * v], h[4 * v + 1], h[4 * v + 2], h[4 * v + 3]);
            }
        }
    }
}

#define OO_FULL_ENC_MODES(X, f, t) \
    X(f, t, false, false, false) X(f, t, false, false, true) X(f, t, false, true, false) X(f, t, false, true, true) \
    X(f, t, true, false, false) X(f, t, true, false, true) X(f, t, true, true, false) X(f, t, true, true, true)

int launch_encode_full(const TreeParams& T, const QueryParams& Q, const FullModeH& mode, float* features, int32_t* slot,
                       int16_t* cell, int n_sms, cudaStream_t stream) {
    if (Q.n == 0) return 0;
    const uint32_t smem = T.dense_ints * 4;
    const uint64_t blocks = (Q.n + 255) / 256;
    const unsigned grid = (unsigned)(blocks < (uint64_t)n_sms * 8 ? blocks : (uint64_t)n_sms * 8);
    const bool vertex = T.vertex != 0, tri8 = mode.tri8 != 0, shifted = mode.lookup == OO_LOOKUP_SHIFTED;
#define X(f, t, v, s8, sh)                                                                                           \
    if (T.F == f && (T.f32 != 0) == t && vertex == v && tri8 == s8 && shifted == sh) {                               \
        encode_full_kernel<f, t, v, s8, sh><<<grid, 256, smem, stream>>>(T, Q, mode, features, slot, cell);          \
        return 1;                                                                                                    \
    }
    OO_FULL_ENC_MODES(X, 4, true)
    OO_FULL_ENC_MODES(X, 8, false)
    OO_FULL_ENC_MODES(X, 16, false)
#undef X
    return -1;
}

}  // namespace oo
