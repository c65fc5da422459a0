// attention_tc.cu -- tensor-core flash attention (bf16).  Placeholder until the kernels land: reports
// "unsupported" so that the dispatcher uses the fp32-FMA kernels.
#include "common.cuh"
namespace orbit {
bool attention_tc_supported(const AttnArgs&) { return false; }
int attention_fwd_tc(const AttnArgs&, cudaStream_t) { set_error("attention_tc not built"); return ORBIT_ERR_UNSUPPORTED; }
int attention_bwd_tc(const AttnArgs&, cudaStream_t) { set_error("attention_tc not built"); return ORBIT_ERR_UNSUPPORTED; }
}  // namespace orbit
