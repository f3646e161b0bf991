// oo_full_fused_w128.cu — the product instances of the fused full-query kernel (oo_full_fused.cuh) for decoders of width 128:
// four teams of 128 threads (tiles in flight) per SM sharing two accumulator slots.  First layers wider than 128 inputs have no instance.
#include "oo_full_fused.cuh"

namespace oo {

int launch_fused_full_w128(const TreeParams& T, const MlpParams& M, const QueryParams& Q, const FullModeH& mode, float* rgb,
        int n_sms, cudaStream_t stream) {
    if (Q.n == 0) return 0;
    if (M.out_dim > 4 || !M.image_tc || M.k1 > 128 || M.width != 128) return -1;
    // four one-part teams over two accumulator slots (oo_full_fused.cuh, NSLOT): 4 x 64 A columns + 2 x 128 D columns.  Measured on B200 at the
    // paper's shapes against two teams of two parts with a slot each: 0.552 -> 0.456 ms (no shift 0.373 -> 0.283, nearest cell 0.250 -> 0.193).
    return launch_full_w<128, 1, 4, false, 2>(T, M, Q, mode, rgb, n_sms, 64, stream);
}

}  // namespace oo
