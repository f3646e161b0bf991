// oo_full.cuh — device functions of the paper's FULL OctaOctree query:
//   f1  blend over the eight neighbouring cells, trilinear weights, non-empty indicator, renormalised   Eq. 10
//   f2  vertex-stored octahedral maps, barycentric interpolation over the containing triangle (3 taps)  Eq. 6,
//   f3  lookup direction = mirror direction w_r, optionally shifted per cell by the disparity   Eq. 8-9
//   f4  attribute vector [x | w_r | n | extras]                                                        Eq. 12
// Each piece is a template switch, so the all-off instance is the hot path of oo_device.cuh again.
//
// Descent for eight neighbours at once.  With p = x*2^d - 1/2 and k0 = floor(p), the neighbour block at depth d is
// k0 + {0,1}^3.  The ancestor at depth d-g of any of its cells lies in the neighbour block of depth d-g (floor((k0+a)/2^g)
// is floor(X -+ 2^-(g+1)) with X = x*2^(d-g), which is floor(X - 1/2) or that plus one), so the hop tables of the hot
// path serve all eight: keep the eight local node indices of the previous station, pick each neighbour's ancestor among
// them, and take ONE dependent load per neighbour and used level.  Cells outside the grid propagate as -1.
#pragma once
#include "oo_device.cuh"

namespace oo {

using FullMode = FullModeH;   // tri8 = OO_SPATIAL_TRILINEAR8, lookup = oo_lookup, attrs_paper = OO_ATTRS_PAPER

// w_r = 2 (n . wo) n - wo, fp32, one rounding per operation, in this order
__device__ __forceinline__ void mirror_dir(const float (&n)[3], const float (&w)[3], float (&r)[3]) {
    const float dot = __fadd_rn(__fadd_rn(__fmul_rn(n[0], w[0]), __fmul_rn(n[1], w[1])), __fmul_rn(n[2], w[2]));
    const float s = __fmul_rn(2.0f, dot);
#pragma unroll
    for (int a = 0; a < 3; ++a) r[a] = __fsub_rn(__fmul_rn(s, n[a]), w[a]);
}

// Directional taps of one lookup: byte offsets from the map's base and their weights.
//   texel maps : 4 taps (i0,j0) (i0+1,j0) (i0,j0+1) (i0+1,j0+1) of the border-padded map, bilinear weights
//   vertex maps: 3 taps = the containing triangle's vertices, barycentric weights (w[3] unused)
struct DirTaps {
    int off[4];
    float w[4];
    int ci, cj, up;     // the index decision (debug output): texel (i0, j0, 0); vertex (ci, cj, upper)
};

template <bool VERTEX>
__device__ __forceinline__ DirTaps dir_taps(const LevelParams& lv, int TB, OctaUV uv) {
    DirTaps d;
    if constexpr (!VERTEX) {
        const Tap t = level_tap(uv, lv.half_r, lv.off);
        const int base = (t.j0 * (int)lv.Rp + t.i0) * TB;
        d.off[0] = base;
        d.off[1] = base + TB;
        d.off[2] = base + (int)lv.row_bytes;
        d.off[3] = base + (int)lv.row_bytes + TB;
        const float wx0 = 1.0f - t.fx, wy0 = 1.0f - t.fy;
        d.w[0] = wx0 * wy0; d.w[1] = t.fx * wy0; d.w[2] = wx0 * t.fy; d.w[3] = t.fx * t.fy;
        d.ci = t.i0; d.cj = t.j0; d.up = 0;
    } else {
        // g = u*(R/2) + R/2 (one rounding: the product is exact), cell = min(floor(g), R-1) (g lies in [0, R]: |u| <= 1), (a, b) = g - cell
        const float gx = __fmaf_rn(uv.ux, lv.half_r, lv.half_r), gy = __fmaf_rn(uv.uy, lv.half_r, lv.half_r);
        const int Rm1 = (int)lv.R - 1;
        const int ci = min(__float2int_rd(gx), Rm1), cj = min(__float2int_rd(gy), Rm1);
        const float a = __fsub_rn(gx, (float)ci), b = __fsub_rn(gy, (float)cj);
        const int half = (int)(lv.R >> 1);
        const bool same = (ci >= half) == (cj >= half);
        const bool up = same ? (__fadd_rn(a, b) >= 1.0f) : (b > a);          // the index decisions, in the contract's form
        // Weights and taps: a cell split along its anti-diagonal (same-sign quadrant) is a cell split along its main diagonal mirrored in
        // x -- a' = 1 - a, columns swapped -- so one rule serves both: vertices (0,0)' and (1,1)' always, (0,1)' above the diagonal
        // and (1,0)' below it, with weights 1 - max(a', b), min(a', b), |b - a'|.
        const float am = same ? 1.0f - a : a;
        const int x0 = same ? TB : 0, x1 = TB - x0;
        const int row = (int)lv.row_bytes;
        const int c00 = (cj * (int)lv.Rp + ci) * TB;
        d.off[0] = c00 + x0;
        d.off[1] = c00 + row + x1;
        d.off[2] = up ? c00 + row + x0 : c00 + x1;
        d.off[3] = d.off[2];
        d.w[0] = 1.0f - (up ? b : am);
        d.w[1] = up ? am : b;
        d.w[2] = fabsf(b - am);
        d.w[3] = 0.0f;
        d.ci = ci; d.cj = cj; d.up = up ? 1 : 0;
    }
    return d;
}

// The neighbour block of the previous station: local node indices (-1 = absent or outside the grid) and base cell.
template <int NJ>
struct Station {
    int node[NJ];
    int k0[3];
};

__device__ __forceinline__ int sel8(const int (&n)[8], int px, int py, int pz) {
    const int a0 = px ? n[1] : n[0], a1 = px ? n[3] : n[2], a2 = px ? n[5] : n[4], a3 = px ? n[7] : n[6];
    const int b0 = py ? a1 : a0, b1 = py ? a3 : a2;
    return pz ? b1 : b0;
}

// base cell (and trilinear fractions) of the neighbour block at `depth`.  TRI8: p = clamp(x,0,1)*2^d - 1/2 (A16), k0 =
// floor(p), t = p - k0 (the product is exact; the subtraction rounds only below 1/2, where floor is -1 either way).
// Nearest: the cell containing x (a2), t unused.
template <bool TRI8>
__device__ __forceinline__ void block_base(const float (&x)[3], uint32_t depth, int (&k0)[3], float (&t)[3]) {
    const float scale = (float)(1u << depth);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if constexpr (TRI8) {
            const float xc = fminf(fmaxf(x[a], 0.0f), 1.0f);
            const float p = __fsub_rn(__fmul_rn(xc, scale), 0.5f);
            const float f = floorf(p);
            k0[a] = (int)f;
            t[a] = __fsub_rn(p, f);
        } else {
            k0[a] = quantise(x[a], scale, (int)(1u << depth) - 1);
            t[a] = 0.0f;
        }
    }
}

template <int NJ>
__device__ __forceinline__ void dense_block(const int32_t* s_dense, uint32_t table_off, uint32_t d, const int (&k0)[3],
                                            int (&out)[NJ]) {
    const int n = 1 << d;
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
        const int cx = k0[0] + (j & 1), cy = k0[1] + ((j >> 1) & 1), cz = k0[2] + ((j >> 2) & 1);
        const bool in = (unsigned)cx < (unsigned)n && (unsigned)cy < (unsigned)n && (unsigned)cz < (unsigned)n;
        out[j] = in ? s_dense[table_off + (((uint32_t)cz << (2 * d)) | ((uint32_t)cy << d) | (uint32_t)cx)] : -1;
    }
}

template <int NJ>
__device__ __forceinline__ void station_init(const TreeParams& T, const int32_t* s_dense, const float (&x)[3],
                                             Station<NJ>& st) {
    float t[3];
    block_base<(NJ == 8)>(x, T.t_depth, st.k0, t);
    dense_block<NJ>(s_dense, T.t_dense_off, T.t_depth, st.k0, st.node);
}

// a3 for the whole block at one used level: slot[j] of neighbour j (-1 = empty / outside); advances the station.
template <int NJ>
__device__ __forceinline__ void block_slots(const LevelParams& lv, const int32_t* s_dense, const int (&k0)[3],
                                            Station<NJ>& st, int (&slot)[NJ]) {
    if (lv.dense) {
        dense_block<NJ>(s_dense, lv.dense_off, lv.depth, k0, slot);
        return;
    }
    const uint32_t g = lv.gap, m = (1u << g) - 1u;
    int pl[3][2];
    uint32_t ix[3][2];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int o = 0; o < (NJ == 8 ? 2 : 1); ++o) {
            const int c = k0[a] + o;
            pl[a][o] = (c >> g) - st.k0[a];            // arithmetic shift: -1 stays -1 (outside the grid)
            ix[a][o] = ((uint32_t)c & m) << (a * g);
        }
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
        const int ox = j & 1, oy = (j >> 1) & 1, oz = (j >> 2) & 1;
        int prev;
        if constexpr (NJ == 8) prev = sel8(st.node, pl[0][ox], pl[1][oy], pl[2][oz]);
        else prev = st.node[0];
        const uint32_t idx = ix[0][ox] | ix[1][oy] | ix[2][oz];
        int v = -1;
        if (prev >= 0) v = __ldg(lv.hop + (((uint32_t)prev << (3 * g)) + idx));
        slot[j] = v;
    }
#pragma unroll
    for (int j = 0; j < NJ; ++j) st.node[j] = slot[j];
#pragma unroll
    for (int a = 0; a < 3; ++a) st.k0[a] = k0[a];
}

// Eq. 10 weights: w_j = 1(c_j) prod(t or 1-t) / sum_p 1(c_p) w_p ; all empty => 0.  Nearest: 1(c).
template <int NJ>
__device__ __forceinline__ void blend_weights(const float (&t)[3], const int (&slot)[NJ], float (&w)[NJ]) {
    if constexpr (NJ == 1) {
        w[0] = slot[0] >= 0 ? 1.0f : 0.0f;
    } else {
        float den = 0.0f;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const float wx = (j & 1) ? t[0] : 1.0f - t[0], wy = (j & 2) ? t[1] : 1.0f - t[1], wz = (j & 4) ? t[2] : 1.0f - t[2];
            w[j] = slot[j] >= 0 ? wx * wy * wz : 0.0f;
            den += w[j];
        }
        const float inv = den > 0.0f ? __fdividef(1.0f, den) : 0.0f;
#pragma unroll
        for (int j = 0; j < 8; ++j) w[j] *= inv;
    }
}

// Eq. 9 numerator for the cell with integer coordinates k at `depth`: w~ = (x - c)*d^ + w_r, c = (k + 1/2) / 2^d (exact)
__device__ __forceinline__ OctaUV shifted_uv(const float (&x)[3], const int (&k)[3], float inv_scale, float disp,
                                             const float (&wr)[3]) {
    float v[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float c = ((float)k[a] + 0.5f) * inv_scale;
        v[a] = __fadd_rn(__fmul_rn(__fsub_rn(x[a], c), disp), wr[a]);
    }
    return octa_project(v[0], v[1], v[2]);
}

struct FullDebug {
    int32_t* slot;     // this query's [L][NJ] or nullptr
    int16_t* cell;     // this query's [L][NJ][3] or nullptr
};

// One used level of the full query for one query: h[0..F) = sum_j w_j * dir_interp(map of neighbour j, direction_j).
// `gather` = false only advances the station (threads that split the levels between them still share the descent).
template <int F, bool F32, bool VERTEX, bool TRI8, bool SHIFTED>
__device__ __forceinline__ void full_level(const LevelParams& lv, const int32_t* s_dense, const float (&x)[3],
                                           const float (&wl)[3], const OctaUV& uv_q, float disp,
                                           Station<(TRI8 ? 8 : 1)>& st, bool gather, float (&h)[F], int level,
                                           const FullDebug& dbg) {
    constexpr int NJ = TRI8 ? 8 : 1;
    constexpr int TB = F * (F32 ? 4 : 2);
    constexpr int NV = TB / 16;
    constexpr int PER = F32 ? 4 : 8;
    constexpr int NT = VERTEX ? 3 : 4;
    constexpr int NB = NJ == 1 ? 1 : (TB == 16 ? 4 : (TB == 32 ? 2 : 1));     // neighbours per load batch
    if (!gather && lv.dense) return;
    int k0[3];
    float t[3];
    block_base<TRI8>(x, lv.depth, k0, t);
    int slot[NJ];
    block_slots<NJ>(lv, s_dense, k0, st, slot);
    if (!gather) return;
    float wj[NJ];
    blend_weights<NJ>(t, slot, wj);
#pragma unroll
    for (int k = 0; k < F; ++k) h[k] = 0.0f;
    DirTaps dq;
    if constexpr (!SHIFTED) dq = dir_taps<VERTEX>(lv, TB, uv_q);
    const float inv_scale = 1.0f / (float)(1u << lv.depth);
#pragma unroll
    for (int j0 = 0; j0 < NJ; j0 += NB) {
        uint4 v[NB][NT][NV];
        TapWeights tw[NB];
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const int j = j0 + b;
            DirTaps d;
            if constexpr (SHIFTED) {
                const int k[3] = {k0[0] + (j & 1), k0[1] + ((j >> 1) & 1), k0[2] + ((j >> 2) & 1)};
                d = dir_taps<VERTEX>(lv, TB, shifted_uv(x, k, inv_scale, disp, wl));
            } else {
                d = dq;
            }
            // an absent neighbour (slot -1) reads the all-zero map in front of slot 0 (and carries weight 0): no test, no predicate
            const uint8_t* p = lv.atlas + (int64_t)slot[j] * (int64_t)lv.map_bytes;
#pragma unroll
            for (int k = 0; k < NT; ++k)
#pragma unroll
                for (int q = 0; q < NV; ++q) v[b][k][q] = ldg16(p + d.off[k] + 16 * q);
            tw[b].w00 = wj[j] * d.w[0]; tw[b].w10 = wj[j] * d.w[1]; tw[b].w01 = wj[j] * d.w[2]; tw[b].w11 = wj[j] * d.w[3];
            if constexpr (!F32) {
                tw[b].p0 = pack_half2(tw[b].w00, tw[b].w10);
                tw[b].p1 = pack_half2(tw[b].w01, tw[b].w11);
            }
            if (dbg.slot) dbg.slot[level * NJ + j] = slot[j];
            if (dbg.cell) {
                int16_t* c = dbg.cell + (level * NJ + j) * 3;
                c[0] = (int16_t)d.ci; c[1] = (int16_t)d.cj; c[2] = (int16_t)d.up;
            }
        }
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int q = 0; q < NV; ++q) {
                accumulate16<F32, 0>(h + PER * q, v[b][0][q], tw[b]);
                accumulate16<F32, 1>(h + PER * q, v[b][1][q], tw[b]);
                accumulate16<F32, 2>(h + PER * q, v[b][2][q], tw[b]);
                if constexpr (!VERTEX) accumulate16<F32, 3>(h + PER * q, v[b][3][q], tw[b]);
            }
    }
}

}  // namespace oo
