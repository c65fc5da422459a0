// api_agg.cu -- orbit_var_aggregate / orbit_var_aggregate_bwd (a2 / a2'; R3, R4).
// Collapsed formulation (aggregate.cu header): per-patch kernels over tok + [B*L]-row GEMMs.
#include <math.h>
#include "api_util.cuh"
#include "frontend.cuh"

namespace orbit {
namespace {

struct AggSaved {
  float *alpha, *qt, *Ut;
  void *o, *Xbar, *Utb;
  size_t bytes;
};
AggSaved carve_agg_saved(const orbit_agg_desc& d, void* base) {
  const size_t BL = (size_t)d.B * d.L, D = d.D, h = d.heads;
  Carver c(base);
  AggSaved s;
  s.alpha = c.take_n<float>(BL * h * d.V);      // softmax weights [B*L, heads, V]
  s.qt = c.take_n<float>(D);                    // q Wq + bq
  s.Ut = c.take_n<float>(D * h);                // collapsed key projection [D, heads]
  s.o = c.take(BL * D * dsize(d.dtype));        // concat_a o_a  [B*L, D]
  s.Xbar = c.take(BL * h * D * dsize(d.dtype)); // sum_v alpha[v,a] X_v  [B*L, heads, D]
  s.Utb = c.take(agg_tc_utb_bytes((int)D));     // bf16 copy of Ut^T for the tensor-core kernels
  s.bytes = c.off;
  return s;
}
struct AggBwdWs {
  void *dob, *dXbar, *daggb;
  float *acc;        // [bo D | bv D | dUt D*h | dqt D]
  size_t acc_floats;
  size_t bytes;
};
AggBwdWs carve_agg_bwd(const orbit_agg_desc& d, void* base) {
  const size_t BL = (size_t)d.B * d.L, D = d.D, h = d.heads;
  Carver c(base);
  AggBwdWs w;
  w.acc_floats = 3 * D + D * h;
  w.acc = c.take_n<float>(w.acc_floats);
  w.daggb = c.take(BL * D * dsize(d.dtype));
  w.dob = c.take(BL * D * dsize(d.dtype));
  w.dXbar = c.take(BL * h * D * dsize(d.dtype));
  w.bytes = c.off;
  return w;
}

int check_agg(const orbit_agg_desc* d, bool bwd) {
  if (!d) { set_error("agg desc is NULL"); return ORBIT_ERR_NULL; }
  if (!valid_dtype(d->dtype) || !valid_dtype(d->resid_dtype)) { set_error("agg: bad dtype"); return ORBIT_ERR_DTYPE; }
  if (d->dtype == ORBIT_F32 && d->resid_dtype != ORBIT_F32) { set_error("agg: resid_dtype must be F32 when dtype is F32"); return ORBIT_ERR_DTYPE; }
  if (d->B <= 0 || d->L <= 0 || d->V <= 0 || d->D <= 0 || d->heads <= 0 || d->D % d->heads || d->D % 8 || d->heads > 32 ||
      (d->D / d->heads) % 8) {
    set_error("agg: bad shape B=%d L=%d V=%d D=%d heads=%d (need D%%heads==0, D%%8==0, (D/heads)%%8==0, heads<=32)", d->B, d->L, d->V, d->D, d->heads);
    return ORBIT_ERR_SHAPE;
  }
  // shared-memory bounds of the per-patch kernel that will actually run: the bf16 TMA kernels carry their own bound
  // (agg_tc_supported); the SIMT forward keeps only the [V, heads] scores, the SIMT backward a [heads, D] fp32 accumulator
  const bool tc = g_force_simt != 1 && agg_tc_supported(d->dtype, d->V, d->D, d->heads);
  if (!tc && (size_t)d->V * d->heads * sizeof(float) > 220 * 1024) { set_error("agg: V*heads too large for the per-patch forward kernel"); return ORBIT_ERR_SHAPE; }
  if (bwd && !tc && agg_patch_bwd_smem(d->V, d->D, d->heads) > 220 * 1024) {
    set_error("agg_bwd: (2 V heads + heads D) * 4 bytes = %zu exceeds 220 KB of shared memory for the per-patch backward kernel",
              agg_patch_bwd_smem(d->V, d->D, d->heads));
    return ORBIT_ERR_SHAPE;
  }
  return ORBIT_OK;
}
int check_agg_params(const orbit_agg_params* P) {
  if (!P) { set_error("agg: params NULL"); return ORBIT_ERR_NULL; }
  const void* ps[9] = {P->q, P->Wq, P->bq, P->Wk, P->bk, P->Wv, P->bv, P->Wo, P->bo};
  for (int i = 0; i < 9; i++) {
    if (!ps[i]) { set_error("agg: NULL parameter %d", i); return ORBIT_ERR_NULL; }
    if (!aligned16(ps[i])) { set_error("agg: parameter %d not 16B aligned", i); return ORBIT_ERR_ALIGN; }
  }
  return ORBIT_OK;
}
}  // namespace
}  // namespace orbit

using namespace orbit;

extern "C" {

size_t orbit_var_aggregate_saved_bytes(const orbit_agg_desc* d) { return d ? carve_agg_saved(*d, nullptr).bytes : 0; }
size_t orbit_var_aggregate_workspace_bytes(const orbit_agg_desc* d) { return d ? 256 : 0; }
size_t orbit_var_aggregate_bwd_workspace_bytes(const orbit_agg_desc* d) { return d ? carve_agg_bwd(*d, nullptr).bytes : 0; }

int orbit_var_aggregate(const orbit_agg_desc* d, const void* tok, const orbit_agg_params* P, const void* pos, void* agg,
                        void* saved, void* ws, size_t ws_bytes, void* stream) {
  ORBIT_TRY(check_agg(d, false));
  ORBIT_TRY(check_agg_params(P));
  if (!tok || !agg || !saved || !ws) { set_error("var_aggregate: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!aligned16(tok) || !aligned16(agg) || !aligned16(saved) || !aligned16(ws) || (pos && !aligned16(pos))) { set_error("var_aggregate: pointer not 16B aligned"); return ORBIT_ERR_ALIGN; }
  if (ws_bytes < orbit_var_aggregate_workspace_bytes(d)) { set_error("var_aggregate: workspace too small"); return ORBIT_ERR_WORKSPACE; }
  ORBIT_TRY(check_device());
  cudaStream_t s = (cudaStream_t)stream;
  const int BL = d->B * d->L, D = d->D, h = d->heads, da = D / h, dt = d->dtype, rt = d->resid_dtype;
  AggSaved sv = carve_agg_saved(*d, saved);
  ORBIT_TRY(agg_make_qt(P->q, P->Wq, P->bq, dt, sv.qt, D, s));   // qt = q Wq + bq (data independent; R3, R4)
  ORBIT_TRY(agg_make_u(P->Wk, dt, sv.qt, sv.Ut, D, h, s));
  const bool tc = g_force_simt != 1 && agg_tc_supported(dt, d->V, D, h);
  {
    ProfScope prof(PROF_FRONT, (double)BL * d->V * D * dsize(dt), s);                            // a2 reads tok once (algorithmic)
    if (tc) ORBIT_TRY(agg_patch_fwd_tc(tok, sv.Ut, sv.Utb, sv.alpha, sv.Xbar, BL, d->V, D, h, s));
    else ORBIT_TRY(agg_patch_fwd(tok, dt, sv.Ut, sv.alpha, sv.Xbar, BL, d->V, D, h, s));
  }
  {  // o_a = Xbar_a Wv[:, a] + bv[a], the `heads` products as one strided-batch launch
    GemmArgs g;
    g.A = sv.Xbar; g.a_rs = (long long)h * D; g.a_cs = 1; g.B = P->Wv; g.b_rs = D; g.b_cs = 1;
    g.C = sv.o; g.ldc = D; g.M = BL; g.N = da; g.K = D;
    g.in_dtype = dt; g.out_dtype = dt; g.bias = P->bv; g.bias_dtype = dt;
    g.batch = h; g.a_bs = D; g.b_bs = da; g.c_bs = da; g.bias_bs = da;
    ORBIT_TRY(gemm(g, s));
  }
  {  // agg = o Wo + bo (+ pos[l])
    GemmArgs g;
    g.A = sv.o; g.a_rs = D; g.a_cs = 1; g.B = P->Wo; g.b_rs = D; g.b_cs = 1; g.C = agg; g.ldc = D;
    g.M = BL; g.N = D; g.K = D; g.in_dtype = dt; g.out_dtype = rt; g.bias = P->bo; g.bias_dtype = dt;
    if (pos) { g.resid = pos; g.resid_dtype = rt; g.ldr = D; g.resid_row_mod = d->L; }
    ORBIT_TRY(gemm(g, s));
  }
  return ORBIT_OK;
}

int orbit_var_aggregate_bwd(const orbit_agg_desc* d, const void* tok, const orbit_agg_params* P, const void* dagg,
                            const void* saved, void* dtok, orbit_agg_grads* G, void* dpos, void* ws, size_t ws_bytes,
                            void* stream) {
  ORBIT_TRY(check_agg(d, true));
  ORBIT_TRY(check_agg_params(P));
  if (!tok || !dagg || !saved || !dtok || !G || !ws) { set_error("var_aggregate_bwd: NULL pointer"); return ORBIT_ERR_NULL; }
  {
    void* gs[9] = {G->q, G->Wq, G->bq, G->Wk, G->bk, G->Wv, G->bv, G->Wo, G->bo};
    for (int i = 0; i < 9; i++) {
      if (!gs[i]) { set_error("var_aggregate_bwd: NULL gradient pointer %d", i); return ORBIT_ERR_NULL; }
      if (!aligned16(gs[i])) { set_error("var_aggregate_bwd: gradient %d not 16B aligned", i); return ORBIT_ERR_ALIGN; }
    }
  }
  if (!aligned16(tok) || !aligned16(dagg) || !aligned16(saved) || !aligned16(dtok) || !aligned16(ws) || (dpos && !aligned16(dpos))) { set_error("var_aggregate_bwd: pointer not 16B aligned"); return ORBIT_ERR_ALIGN; }
  if (ws_bytes < orbit_var_aggregate_bwd_workspace_bytes(d)) { set_error("var_aggregate_bwd: workspace too small"); return ORBIT_ERR_WORKSPACE; }
  ORBIT_TRY(check_device());
  cudaStream_t s = (cudaStream_t)stream;
  const int BL = d->B * d->L, D = d->D, h = d->heads, da = D / h, dt = d->dtype, rt = d->resid_dtype;
  AggSaved sv = carve_agg_saved(*d, const_cast<void*>(saved));
  AggBwdWs w = carve_agg_bwd(*d, ws);
  float* acc_bo = w.acc;
  float* acc_bv = acc_bo + D;
  float* acc_dUt = acc_bv + D;
  float* dqt = acc_dUt + (size_t)D * h;
  ORBIT_TRY(fill_zero(w.acc, w.acc_floats * sizeof(float), s));
  // dbo = colsum(g); g in the compute dtype; dpos
  const void* gb = dagg;
  if (rt != dt) { ORBIT_TRY(colsum(dagg, rt, D, BL, D, acc_bo, w.daggb, dt, D, s)); gb = w.daggb; }
  else ORBIT_TRY(colsum(dagg, rt, D, BL, D, acc_bo, nullptr, dt, D, s));
  if (dpos) ORBIT_TRY(agg_dpos(dagg, rt, dpos, d->B, d->L, D, s));
  {  // dWo = o^T g
    GemmArgs g;
    g.A = sv.o; g.a_rs = 1; g.a_cs = D; g.B = gb; g.b_rs = D; g.b_cs = 1; g.C = G->Wo; g.ldc = D;
    g.M = D; g.N = D; g.K = BL; g.in_dtype = dt; g.out_dtype = dt;
    ORBIT_TRY(gemm(g, s));
  }
  {  // do = g Wo^T
    GemmArgs g;
    g.A = gb; g.a_rs = D; g.a_cs = 1; g.B = P->Wo; g.b_rs = 1; g.b_cs = D; g.C = w.dob; g.ldc = D;
    g.M = BL; g.N = D; g.K = D; g.in_dtype = dt; g.out_dtype = dt;
    ORBIT_TRY(gemm(g, s));
  }
  ORBIT_TRY(colsum(w.dob, dt, D, BL, D, acc_bv, nullptr, dt, D, s));   // dbv = sum do   (sum_v alpha = 1)
  {
    GemmArgs gw;   // dWv[:, a] = Xbar_a^T do_a   (strided batch over the heads)
    gw.A = sv.Xbar; gw.a_rs = 1; gw.a_cs = (long long)h * D; gw.B = w.dob; gw.b_rs = D; gw.b_cs = 1;
    gw.C = G->Wv; gw.ldc = D; gw.M = D; gw.N = da; gw.K = BL; gw.in_dtype = dt; gw.out_dtype = dt;
    gw.batch = h; gw.a_bs = D; gw.b_bs = da; gw.c_bs = da;
    ORBIT_TRY(gemm(gw, s));
    GemmArgs gx;   // dXbar_a = do_a Wv[:, a]^T
    gx.A = w.dob; gx.a_rs = D; gx.a_cs = 1; gx.B = P->Wv; gx.b_rs = 1; gx.b_cs = D;
    gx.C = w.dXbar; gx.ldc = (long long)h * D; gx.M = BL; gx.N = D; gx.K = da; gx.in_dtype = dt; gx.out_dtype = dt;
    gx.batch = h; gx.a_bs = da; gx.b_bs = da; gx.c_bs = D;
    ORBIT_TRY(gemm(gx, s));
  }
  const bool tc = g_force_simt != 1 && agg_tc_supported(dt, d->V, D, h);
  {
    ProfScope prof(PROF_FRONT, 2.0 * BL * d->V * D * dsize(dt), s);                              // a2' reads tok and writes dtok
    if (tc) ORBIT_TRY(agg_patch_bwd_tc(tok, sv.Utb, sv.alpha, w.dXbar, dtok, acc_dUt, BL, d->V, D, h, s));
    else ORBIT_TRY(agg_patch_bwd(tok, dt, sv.Ut, sv.alpha, w.dXbar, dtok, acc_dUt, BL, d->V, D, h, s));
  }
  ORBIT_TRY(agg_param_bwd(acc_dUt, sv.qt, P->q, P->Wq, P->Wk, dt, G->Wk, G->bk, G->bq, G->Wq, G->q, dqt, D, h, s));
  ORBIT_TRY(cast_copy(acc_bo, ORBIT_F32, G->bo, dt, D, s));
  ORBIT_TRY(cast_copy(acc_bv, ORBIT_F32, G->bv, dt, D, s));
  return ORBIT_OK;
}

}  // extern "C"
