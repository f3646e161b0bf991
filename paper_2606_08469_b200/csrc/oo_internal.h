// oo_internal.h — structures shared by the host side of liboo (oo_api.cu) and its kernels (oo_kernels.cu).
// Not part of the ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <string>

#include "oo.h"

namespace oo {

// ---------------------------------------------------------------------------------------------------------------
// Device-side view of one used level.  The library's atlas layout is level-major and BORDER-PADDED: every map is
// (R+2) x (R+2) texels, the one-texel border pre-filled by the octahedral wrap, so the four bilinear taps of any
// base texel (i0, j0) in [-1, R-1]^2 are plain neighbours and the hot loop has no wrap logic.  `atlas` is pre-offset by
// one row and one texel, so tap (i0, j0) is at  atlas + slot*map_bytes + (j0*Rp + i0)*texel_bytes  for i0, j0 >= -1.
// In front of slot 0 lies one all-zero map, "slot -1": a query whose cell is absent at this level (A17) gathers from it with
// the ordinary weights and gets exact zeros, so the specialised gather has no `slot >= 0` test, no clamp and no weight masks.
// `atlas_z` is the start of that zero map and addresses are formed in 16-byte units from it (32 bits reach 64 GB per level):
//   unit index = (slot + 1) * map16 + ((j0*Rp + i0) * texel16 + tap16),   address = atlas_z + 16 * unit index
// with tap16 = (Rp + 1) * texel16 the unit of tap (0, 0) inside a map; the second tap row is rb16 = Rp * texel16 units further.
struct LevelParams {
    const uint8_t* atlas;
    const uint8_t* atlas_z; // texel maps: start of the zero map in front of slot 0 (see above); vertex maps: nullptr
    const int32_t* hop;     // hop table from the previous station: [n_prev][8^gap] -> slot at this depth (-1 = absent)
    float half_r;           // R/2
    float off;              // R/2 - 1/2
    uint32_t R;
    uint32_t Rp;            // R + 2
    uint32_t map_bytes;     // Rp*Rp*texel_bytes
    uint32_t row_bytes;     // Rp*texel_bytes
    uint32_t depth;
    uint32_t shift;         // depth_eff - depth
    uint32_t dense;         // 1: slot = dense table lookup (depth <= 4); 0: hop from the previous station
    uint32_t dense_off;     // offset (ints) of this level's dense table inside the dense block
    uint32_t gap;           // depth - previous station depth (1..3) when !dense
    uint32_t map16;         // map_bytes / 16
    uint32_t tap16;         // (Rp + 1) * texel_bytes / 16
    float rp_f;             // Rp as fp32: (j0*Rp + i0) is formed in fp32 (exact: |value| < 2^24) and converted once
};

struct TreeParams {
    LevelParams lv[OO_MAX_LEVELS];
    uint32_t n_levels;
    uint32_t F;
    uint32_t f32;            // texel dtype is fp32
    uint32_t texel_bytes;
    uint32_t vertex;         // OO_DIRMAP_VERTEX: maps are (R+1)^2 vertices, unpadded (Rp = R+1, atlas not pre-offset)
    uint32_t depth_eff;      // deepest used depth: positions are quantised to 2^depth_eff cells per axis
    float scale_eff;         // 2^depth_eff
    // top station: dense table at depth T = min(4, depth_eff) giving the local node index at that depth
    uint32_t t_depth, t_shift, t_dense_off;
    uint32_t dense_ints;     // total ints of the dense block (staged into shared memory by the fast kernels)
    const int32_t* dense;    // global copy of the dense block
    // plain representation for the generic kernels
    const int32_t* child;    // [n_nodes][8]
    const int32_t* map_slot; // [n_nodes]
};

struct QueryParams {
    uint64_t n;
    const float* x;
    const float* nrm;
    const float* wo;
    const float* extra;
    uint32_t n_extra;
    const uint32_t* perm;
    const float* disparity;  // [n] or nullptr (OO_LOOKUP_SHIFTED)
    const uint32_t* out_idx; // encode kernels and the debug instances (OO_PRESORT_BIN): thread t reads query t and stores its
                             // feature / index rows at out_idx[t] (the query's index in the caller's order)
    // OO_PRESORT_AUTO: where the kernel that sees the queries in the CALLER's order leaves its coherence samples (slots of a
    // small device array) and the call's sequence number; null = no sampling
    unsigned long long* stat;
    uint32_t stat_seq;
    int32_t* dbg_slot;       // oo_query_debug only (read by the DBG instances of the fused kernels): [n][L] (full query [n][L][J])
    int16_t* dbg_texel;      // ... and [n][L][2] (full query [n][L][J][3]); either may be null
};

// Decoder image: the padded, shared-memory-ready copy of the weights (built by oo_upload_mlp).
//   layer 0:        [64][K1 + 8] halves, K1 = in_dim rounded up to 16 (extra columns zero)
//   layers 1..H-1:  [64][72]
//   output layer:   [16][72] (rows >= out_dim zero)      -- 16 rows so that the same image also serves a N=16 UMMA
struct MlpParams {
    const uint16_t* image;   // global
    uint32_t image_bytes;
    uint32_t in_dim, k1, n_hidden, out_dim, out_act;
    uint32_t feat_dim;       // L*F
    // the same weights in the UMMA K-major canonical layout for the tcgen05 kernel: per layer [K/8][N][8] halves
    // (layer 0: K = k1, N = 64; hidden: K = N = 64; output: K = 64, N = 16 with rows >= out_dim zero)
    // (width-W decoders: N = W for the hidden layers, K = W after the first)
    const uint16_t* image_tc;
    uint32_t image_tc_bytes;
    uint32_t width;          // 64 or 128; `image` (the mma.sync copy) exists only for 64
};

// Disparity predictor g_psi (Eq. 7): multi-resolution hash grid over position.  All tables live in one device buffer.
struct GridLevel {
    const uint32_t* table;   // [T_g] entries of two fp16 features (one 32-bit word)
    float scale;             // N_g as fp32
    uint32_t n_max;          // N_g - 1: the last cell
    uint32_t stride;         // N_g + 1 vertices per axis (dense levels)
    uint32_t mask;           // T_max - 1 (hashed levels); 0 = dense
};
struct GridParams {
    GridLevel lv[OO_MAX_GRID_LEVELS];
    uint32_t n_levels;
    uint32_t n_dense;        // dense levels come first and number n_dense; n_levels + 1 if dense and hashed levels interleave
};

struct EncodeOut {
    void* features;          // [n][L*F] tree dtype, or nullptr
    int32_t* slot;           // [n][L] or nullptr
    int16_t* texel;          // [n][L][2] or nullptr
};

// ---------------------------------------------------------------------------------------------------------------
// Coherence statistics (OO_PRESORT_AUTO).  A warp holds 32 consecutive queries of the caller's order; the number of distinct
// depth-4 cells (16^3) among them is ~1-3 for screen-order primary hits and ~30 for random surface samples.  Sampled warps add
// write (sequence number of the call, 1, distinct) into a slot of a small device array; a side stream copies the array to pinned
// host memory after the call's kernels, and the host reads whatever is there when the next call is made: nothing but an event
// record is added to the caller's stream and nobody waits (every slot is always a whole sample of some recent call).
constexpr uint32_t kStatSlots = 256;
constexpr uint32_t kStatSeqBits = 20, kStatCntBits = 12;
inline unsigned long long stat_pack(uint32_t seq, uint32_t cnt, uint32_t sum) {
    return ((unsigned long long)(seq & ((1u << kStatSeqBits) - 1u)) << 44) | ((unsigned long long)(cnt & ((1u << kStatCntBits) - 1u)) << 32) | sum;
}

// cudaFuncAttributeMaxDynamicSharedMemorySize is a PER-DEVICE attribute of a kernel: a context on device 1 created after one
// on device 0 in the same process needs the opt-in again.  Every launch site therefore owns one bit per device ordinal
// (`mask`, a function-local static of that site, one per kernel instance) and opts in the first time it launches on the
// current device.  Returns false when the CUDA call fails (the launcher then returns kLaunchCudaError).
constexpr int kLaunchCudaError = -2;
inline bool opt_in_smem(std::atomic<uint64_t>& mask, const void* kernel, int bytes) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return false;
    const uint64_t bit = (unsigned)dev < 64u ? 1ull << dev : 0ull;       // ordinals >= 64: opt in on every launch
    if (bit && (mask.load(std::memory_order_acquire) & bit)) return true;
    if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) != cudaSuccess) return false;
    if (bit) mask.fetch_or(bit, std::memory_order_release);
    return true;
}

// Launchers (oo_kernels.cu / oo_sort.cu).  Each returns the number of kernels it launched, -1 if the requested
// specialisation does not exist, or kLaunchCudaError if a CUDA call made on the way failed.  All launches go to `stream`.
int launch_pad_atlas(const void* src, void* dst, uint64_t slots, uint32_t R, uint32_t texel_bytes, cudaStream_t stream);
int launch_tie_vertex_borders(void* maps, uint64_t slots, uint32_t R, uint32_t texel_bytes, unsigned long long* changed, cudaStream_t stream);
int launch_encode_generic(const TreeParams& T, const QueryParams& Q, const EncodeOut& O, uint32_t tree_max_depth,
                          cudaStream_t stream);
// cache_cold: binned or measured-incoherent batch -> the pipelined-descent variant where the tree has one (oo_kernels.cu)
int launch_encode_fast(const TreeParams& T, const QueryParams& Q, const EncodeOut& O, int n_sms, cudaStream_t stream, bool cache_cold = false,
                       bool* pipelined = nullptr);
int launch_mlp_rows(const TreeParams& T, const MlpParams& M, const QueryParams& Q, const void* features, float* rgb,
                    int n_sms, cudaStream_t stream);
// dbg = true selects the instances with the index sink compiled in (oo_query_debug; QueryParams::dbg_slot / dbg_texel)
int launch_fused_mma(const TreeParams& T, const MlpParams& M, const QueryParams& Q, float* rgb, int n_sms,
                     cudaStream_t stream, bool dbg = false);
int launch_fused_tc(const TreeParams& T, const MlpParams& M, const QueryParams& Q, float* rgb, int n_sms,
                    cudaStream_t stream, bool dbg = false);
// The pipelined descent (gather_pipelined, oo_device.cuh) exists for fp16 trees whose first two used levels are dense and every
// later one a hop, i.e. the BASELINE.json configs.
inline bool pipe_applies(const TreeParams& T) {
    if (T.n_levels < 3 || T.f32 || !T.lv[0].dense || !T.lv[1].dense) return false;
    for (uint32_t l = 2; l < T.n_levels; ++l)
        if (T.lv[l].dense) return false;
    return true;
}
bool fast_shape_supported(uint32_t L, uint32_t F, bool f32);
bool tc_shape_supported(uint32_t L, uint32_t F, bool f32);
int launch_fused_tm(const TreeParams& T, const MlpParams& M, const QueryParams& Q, float* rgb, int n_sms,
                    cudaStream_t stream);
int launch_fused_tm_dbg(const TreeParams& T, const MlpParams& M, const QueryParams& Q, float* rgb, int n_sms,
                        cudaStream_t stream);
bool tm_shape_supported(uint32_t L, uint32_t F, bool f32);
// full query (oo_full_*.cu)
struct FullModeH { uint32_t tri8, lookup, attrs_paper; };
int launch_encode_full(const TreeParams& T, const QueryParams& Q, const FullModeH& mode, float* features, int32_t* slot,
                       int16_t* cell, int n_sms, cudaStream_t stream);
int launch_fused_full_w64(const TreeParams& T, const MlpParams& M, const QueryParams& Q, const FullModeH& mode, float* rgb,
                          int n_sms, cudaStream_t stream);
int launch_fused_full_w128(const TreeParams& T, const MlpParams& M, const QueryParams& Q, const FullModeH& mode, float* rgb,
                           int n_sms, cudaStream_t stream);
int launch_fused_full_w64_dbg(const TreeParams& T, const MlpParams& M, const QueryParams& Q, const FullModeH& mode, float* rgb,
                              int n_sms, cudaStream_t stream);
int launch_fused_full_w128_dbg(const TreeParams& T, const MlpParams& M, const QueryParams& Q, const FullModeH& mode, float* rgb,
                               int n_sms, cudaStream_t stream);
// g_psi: d^ [n] (and optionally the hash-grid features [n][2G] fp32); M is the predictor's own decoder image (out_dim 1)
int launch_disparity(const GridParams& G, const MlpParams& M, const QueryParams& Q, float* disparity, float* features, int n_sms,
                     cudaStream_t stream);
int launch_raycast(const double* d_spheres, uint32_t n_spheres, double lo, double hi, const double eye[3], const double look[3],
                   const double up[3], double vfov_deg, uint32_t width, uint32_t height, float* x, float* nrm, float* wo,
                   int32_t* surf, cudaStream_t stream);
int launch_morton_sort(const float* x, uint64_t n, uint32_t* keys_a, uint32_t* keys_b, uint32_t* idx_a, uint32_t* perm_out,
                       uint32_t* hist, cudaStream_t stream);
size_t morton_sort_hist_ints(uint64_t n);
int launch_bin_queries(const QueryParams& Q, uint32_t* keys, uint32_t* hist, uint32_t* bin_tot, float* sx, float* sn, float* sw, float* se,
                       uint32_t* inv, uint32_t* idx, float* sdisp, cudaStream_t stream);
int launch_unbin(const float* binned, const uint32_t* inv, uint64_t n, uint32_t out_dim, float* out, int n_sms, cudaStream_t stream);

}  // namespace oo
