// frontend.cuh -- internal launchers of the front end (tokenise a1/a1', aggregate a2/a2' per-patch kernels).
#pragma once
#include "common.cuh"

namespace orbit {

// a1: tok[b,l,v,:] = sum_r pix(b,v,l,r) Wp[v,r,:] + bp[v,:]     (R1)
int tokenize_fwd(const orbit_embed_desc& d, const float* x, const void* Wp, const void* bp, void* tok, cudaStream_t s);
// a1': accW[v,r,:] += sum pix dtok ; accB[v,:] += sum dtok   (fp32 accumulators, zeroed by the caller)
int tokenize_bwd_acc(const orbit_embed_desc& d, const float* x, const void* dtok, float* accW, float* accB,
                     cudaStream_t s);

// tensor-core versions (bf16; tokenize_tc.cu)
bool tokenize_tc_supported(const orbit_embed_desc& d);
int tokenize_fwd_tc(const orbit_embed_desc& d, const float* x, const void* Wp, const void* bp, void* tok, cudaStream_t s);
int tokenize_bwd_acc_tc(const orbit_embed_desc& d, const float* x, const void* dtok, float* accW, float* accB, cudaStream_t s);

// a2 helpers (collapsed form):
//   Ut[d,a] = sum_{c in head a} Wk[d,c] qt[c] / sqrt(d_a)
//   qt[n] = sum_k q[k] Wq[k,n] + bq[n]
int agg_make_qt(const void* q, const void* Wq, const void* bq, int p_dt, float* qt, int D, cudaStream_t s);
int agg_make_u(const void* Wk, int p_dt, const float* qt, float* Ut, int D, int heads, cudaStream_t s);
//   per patch: s[v,a] = X_v . Ut[:,a]; alpha = softmax_v; Xbar[a,:] = sum_v alpha[v,a] X_v
int agg_patch_fwd(const void* tok, int dt, const float* Ut, float* alpha, void* Xbar, int BL, int V, int D,
                  int heads, cudaStream_t s);
//   per patch backward: dalpha, ds, dtok, dUt accumulation (fp32 atomics into dUt_acc, zeroed by caller)
int agg_patch_bwd(const void* tok, int dt, const float* Ut, const float* alpha, const void* dXbar, void* dtok,
                  float* dUt_acc, int BL, int V, int D, int heads, cudaStream_t s);
//   parameter gradients that hang off dUt:  dWk, dbk(=0), dqt -> dbq, dWq, dq
int agg_param_bwd(const float* dUt, const float* qt, const void* q, const void* Wq, const void* Wk, int p_dt,
                  void* dWk, void* dbk, void* dbq, void* dWq, void* dq, float* dqt_ws, int D, int heads,
                  cudaStream_t s);
//   dpos[l,:] = sum_b dagg[b,l,:]
int agg_dpos(const void* dagg, int dt, void* dpos, int B, int L, int D, cudaStream_t s);
size_t agg_patch_bwd_smem(int V, int D, int heads);
// tensor-core (mma.sync) per-patch kernels, bf16 only (aggregate_tc.cu)
bool agg_tc_supported(int dt, int V, int D, int heads);
size_t agg_tc_utb_bytes(int D);
int agg_patch_fwd_tc(const void* tok, const float* Ut, void* Utb, float* alpha, void* Xbar, int BL, int V, int D, int heads,
                     cudaStream_t s);
int agg_patch_bwd_tc(const void* tok, const void* Utb, const float* alpha, const void* dXbar, void* dtok, float* dUt_acc,
                     int BL, int V, int D, int heads, cudaStream_t s);

}  // namespace orbit
