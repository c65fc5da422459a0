// attention.cu -- dispatch between the attention kernels:
//   tcgen05/TMEM flash kernels (attention_tc5.cu), forward and backward, for bf16, d_h in {64, 128, 192, 256} (192 and
//   256 are the paper's own head widths), N >= 128;
//   mma.sync flash kernels (attention_tc.cu) otherwise for bf16 d_h in {64, 128}; fp32-FMA kernels else (fp32 storage,
//   other head widths, bf16 d_h 192 / 256 with N < 128).
// orbit_set_debug_force_simt: 1 = fp32-FMA kernels everywhere, 3 = skip the tcgen05 attention (A/B comparison),
// 4 = tcgen05 forward only (mma.sync backward).
#include "common.cuh"

namespace orbit {

bool attention_tc_supported(const AttnArgs& a);
int attention_fwd_tc(const AttnArgs& a, cudaStream_t s);
int attention_bwd_tc(const AttnArgs& a, cudaStream_t s);
bool attention_tc5_supported(const AttnArgs& a);
bool attention_bwd_tc5_supported(const AttnArgs& a);
int attention_fwd_tc5(const AttnArgs& a, cudaStream_t s);
int attention_bwd_tc5(const AttnArgs& a, cudaStream_t s);

// algorithmic work: forward 4 B N^2 D FLOP (QK^T and PV), backward twice that (backward = 2x forward)
static double attn_flops(const AttnArgs& a) { return 4.0 * a.B * (double)a.N * a.N * a.heads * a.dh; }

int attention_fwd(const AttnArgs& a, cudaStream_t s) {
  ProfScope prof(PROF_ATTN_FWD, attn_flops(a), s);
  if (g_force_simt != 1 && g_force_simt != 3 && attention_tc5_supported(a)) return attention_fwd_tc5(a, s);
  if (g_force_simt != 1 && attention_tc_supported(a)) return attention_fwd_tc(a, s);
  return attention_fwd_simt(a, s);
}
int attention_bwd(const AttnArgs& a, cudaStream_t s) {
  ProfScope prof(PROF_ATTN_BWD, 2.0 * attn_flops(a), s);
  if (g_force_simt != 1 && g_force_simt != 3 && g_force_simt != 4 && attention_tc5_supported(a) && attention_bwd_tc5_supported(a))
    return attention_bwd_tc5(a, s);
  if (g_force_simt != 1 && attention_tc_supported(a)) return attention_bwd_tc(a, s);
  return attention_bwd_simt(a, s);
}

}  // namespace orbit
