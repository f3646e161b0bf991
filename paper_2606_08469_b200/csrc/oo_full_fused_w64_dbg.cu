// oo_full_fused_w64_dbg.cu — the debug (oo_query_debug: index sink compiled in) instances of the fused full-query kernel (oo_full_fused.cuh) for decoders of width 64:
// teams of 1 x 128 threads, 4 teams (tiles in flight) per SM.
// A translation unit of its own so that the product instances are neither recompiled nor perturbed.
#include "oo_full_fused.cuh"

namespace oo {

int launch_fused_full_w64_dbg(const TreeParams& T, const MlpParams& M, const QueryParams& Q, const FullModeH& mode, float* rgb,
           int n_sms, cudaStream_t stream) {
    if (Q.n == 0) return 0;
    if (M.out_dim > 4 || !M.image_tc || M.k1 > 128 || M.width != 64) return -1;
    const uint32_t team_cols = 64 + (M.k1 / 2 > 64 / 2 ? M.k1 / 2 : 64 / 2);
    if (4 * team_cols > 512) return -1;
    return launch_full_w<64, 1, 4, true>(T, M, Q, mode, rgb, n_sms, team_cols, stream);
}

}  // namespace oo
