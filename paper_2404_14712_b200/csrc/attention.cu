// attention.cu -- dispatch between the tensor-core (bf16) and the fp32-FMA attention kernels.
#include "common.cuh"

namespace orbit {

bool attention_tc_supported(const AttnArgs& a);
int attention_fwd_tc(const AttnArgs& a, cudaStream_t s);
int attention_bwd_tc(const AttnArgs& a, cudaStream_t s);

int attention_fwd(const AttnArgs& a, cudaStream_t s) {
  if (g_force_simt != 1 && attention_tc_supported(a)) return attention_fwd_tc(a, s);
  return attention_fwd_simt(a, s);
}
int attention_bwd(const AttnArgs& a, cudaStream_t s) {
  if (g_force_simt != 1 && attention_tc_supported(a)) return attention_bwd_tc(a, s);
  return attention_bwd_simt(a, s);
}

}  // namespace orbit
