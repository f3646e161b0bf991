// oo_fused_tc.cu — fused encode + MLP on tcgen05.mma with TMEM accumulators (OO_PATH_FUSED_TC).
#include "oo_device.cuh"

namespace oo {

int launch_fused_tc(const TreeParams&, const MlpParams&, const QueryParams&, float*, int, cudaStream_t) {
    return -1;   // not built yet: oo_query reports OO_ERR_UNSUPPORTED for OO_PATH_FUSED_TC
}

}  // namespace oo
