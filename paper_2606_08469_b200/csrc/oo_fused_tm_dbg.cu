// oo_fused_tm_dbg.cu — the debug instances of the TMEM-resident fused kernel (oo_query_debug): the same kernels as
// oo_fused_tm.cu with the index sink compiled in, so that the slot and base texel every query gathers from can be compared
// bit for bit with the CPU side (BASELINE.json north_star: "node indices and texel indices bit-exact").  A separate
// translation unit so that the product instances are not recompiled or perturbed.
#include "oo_fused_tm.cuh"

namespace oo {

int launch_fused_tm_dbg(const TreeParams& T, const MlpParams& M, const QueryParams& Q, float* rgb, int n_sms, cudaStream_t stream) {
    return launch_fused_tm_impl<true>(T, M, Q, rgb, n_sms, stream);
}

}  // namespace oo
