// oo_fused_tm.cu — the product instances of the TMEM-resident fused kernel (OO_PATH_FUSED_TC_TMEM); kernel in oo_fused_tm.cuh.
#include "oo_fused_tm.cuh"

namespace oo {

bool tm_shape_supported(uint32_t L, uint32_t F, bool f32) {
#define X(l, f, t) if (L == l && F == f && f32 == t) return true;
    OO_TM_SHAPES(X)
#undef X
    return false;
}

int launch_fused_tm(const TreeParams& T, const MlpParams& M, const QueryParams& Q, float* rgb, int n_sms, cudaStream_t stream) {
    return launch_fused_tm_impl<false>(T, M, Q, rgb, n_sms, stream);
}

}  // namespace oo
