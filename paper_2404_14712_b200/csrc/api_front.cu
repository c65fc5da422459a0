// api_front.cu -- orbit_embed_fused / orbit_embed_fused_bwd: tokenisation + variable aggregation fused in pixel
// space.  Host code only sequences kernels and GEMMs.
#include "api_util.cuh"
#include "front_fused.cuh"
#include "frontend.cuh"

namespace orbit {
namespace {

struct FeDims {
  int L, BL, P2, R, Vp, KVp, da;
};
FeDims fe_dims(const orbit_front_desc& d) {
  FeDims f;
  f.L = (d.Hg / d.p) * (d.Wg / d.p); f.BL = d.B * f.L; f.P2 = d.p * d.p; f.R = f.P2 + 1;
  f.Vp = (d.V + 7) & ~7; f.KVp = f.R * f.Vp; f.da = d.D / d.heads;
  return f;
}

struct FeSaved {
  float *alpha, *qt, *Ut, *G;
  void *A, *o, *Wpb, *H;
  size_t bytes;
};
FeSaved carve_fe_saved(const orbit_front_desc& d, void* base) {
  const FeDims f = fe_dims(d);
  const size_t es = dsize(d.dtype), D = d.D, h = d.heads;
  Carver c(base);
  FeSaved s;
  s.alpha = c.take_n<float>((size_t)f.BL * h * f.Vp);       // softmax weights [BL, heads, Vp]
  s.qt = c.take_n<float>(D);
  s.Ut = c.take_n<float>(D * h);
  s.G = c.take_n<float>((size_t)f.KVp * FE_HP);
  s.A = c.take((size_t)f.BL * h * f.KVp * es);              // alpha * pixext  [BL, heads, R*Vp]
  s.o = c.take((size_t)f.BL * D * es);
  s.Wpb = c.take((size_t)f.KVp * D * es);
  s.H = c.take((size_t)f.KVp * D * es);                     // Wpb Wv
  s.bytes = c.off;
  return s;
}
struct FeBwdWs {
  float *acc, *dsT, *dG, *accW;   // acc = [bo D | bv D | dUt D*h | dqt D]
  size_t acc_floats;
  void *daggb, *dob, *dH, *dA;
  size_t bytes;
};
FeBwdWs carve_fe_bwd(const orbit_front_desc& d, void* base) {
  const FeDims f = fe_dims(d);
  const size_t es = dsize(d.dtype), D = d.D, h = d.heads;
  Carver c(base);
  FeBwdWs w;
  w.acc_floats = 3 * D + D * h;
  w.acc = c.take_n<float>(w.acc_floats);
  w.dG = c.take_n<float>((size_t)f.KVp * FE_HP);
  w.dsT = c.take_n<float>((size_t)f.Vp * f.BL * FE_HP);
  w.accW = c.take_n<float>((size_t)f.KVp * D);
  w.daggb = c.take((size_t)f.BL * D * es);
  w.dob = c.take((size_t)f.BL * D * es);
  w.dH = c.take((size_t)f.KVp * D * es);
  w.dA = c.take((size_t)f.BL * h * f.KVp * es);
  w.bytes = c.off;
  return w;
}

int check_front(const orbit_front_desc* d) {
  if (!d) { set_error("front desc is NULL"); return ORBIT_ERR_NULL; }
  if (!valid_dtype(d->dtype) || !valid_dtype(d->resid_dtype)) { set_error("embed_fused: bad dtype"); return ORBIT_ERR_DTYPE; }
  if (d->dtype == ORBIT_F32 && d->resid_dtype != ORBIT_F32) { set_error("embed_fused: resid_dtype must be F32 when dtype is F32"); return ORBIT_ERR_DTYPE; }
  if (d->B <= 0 || d->V <= 0 || d->Hg <= 0 || d->Wg <= 0 || d->p <= 0 || d->D <= 0 || d->heads <= 0 || d->Hg % d->p ||
      d->Wg % d->p || d->D % d->heads || d->D % 8 || (d->D / d->heads) % 8 || !fe_supported(d->V, d->p, d->heads)) {
    set_error("embed_fused: bad shape B=%d V=%d grid=%dx%d p=%d D=%d heads=%d (need Hg%%p==0, Wg%%p==0, D%%heads==0, D%%8==0, "
              "(D/heads)%%8==0, V<=128, p in {1,2,4}, heads<=16)", d->B, d->V, d->Hg, d->Wg, d->p, d->D, d->heads);
    return ORBIT_ERR_SHAPE;
  }
  return ORBIT_OK;
}
int check_front_params(const orbit_agg_params* P) {
  if (!P) { set_error("embed_fused: params NULL"); return ORBIT_ERR_NULL; }
  const void* ps[9] = {P->q, P->Wq, P->bq, P->Wk, P->bk, P->Wv, P->bv, P->Wo, P->bo};
  for (int i = 0; i < 9; i++) {
    if (!ps[i]) { set_error("embed_fused: NULL parameter %d", i); return ORBIT_ERR_NULL; }
    if (!aligned16(ps[i])) { set_error("embed_fused: parameter %d not 16B aligned", i); return ORBIT_ERR_ALIGN; }
  }
  return ORBIT_OK;
}
}  // namespace
}  // namespace orbit

using namespace orbit;

extern "C" {

size_t orbit_embed_fused_saved_bytes(const orbit_front_desc* d) { return d ? carve_fe_saved(*d, nullptr).bytes : 0; }
size_t orbit_embed_fused_workspace_bytes(const orbit_front_desc* d) { return d ? 256 : 0; }
size_t orbit_embed_fused_bwd_workspace_bytes(const orbit_front_desc* d) { return d ? carve_fe_bwd(*d, nullptr).bytes : 0; }

int orbit_embed_fused(const orbit_front_desc* d, const float* x, const void* Wp, const void* bp, const orbit_agg_params* P,
                      const void* pos, void* agg, void* saved, void* ws, size_t ws_bytes, void* stream) {
  ORBIT_TRY(check_front(d));
  ORBIT_TRY(check_front_params(P));
  if (!x || !Wp || !bp || !agg || !saved || !ws) { set_error("embed_fused: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!aligned16(x) || !aligned16(Wp) || !aligned16(bp) || !aligned16(agg) || !aligned16(saved) || !aligned16(ws) ||
      (pos && !aligned16(pos))) { set_error("embed_fused: pointer not 16B aligned"); return ORBIT_ERR_ALIGN; }
  if (ws_bytes < orbit_embed_fused_workspace_bytes(d)) { set_error("embed_fused: workspace too small"); return ORBIT_ERR_WORKSPACE; }
  ORBIT_TRY(check_device());
  cudaStream_t s = (cudaStream_t)stream;
  const FeDims f = fe_dims(*d);
  const int D = d->D, h = d->heads, dt = d->dtype, rt = d->resid_dtype;
  FeSaved sv = carve_fe_saved(*d, saved);
  // parameter-only operands: qt, Ut (collapsed key projection), Wpb, G = Wpb Ut, H = Wpb Wv
  ORBIT_TRY(agg_make_qt(P->q, P->Wq, P->bq, dt, sv.qt, D, s));
  ORBIT_TRY(agg_make_u(P->Wk, dt, sv.qt, sv.Ut, D, h, s));
  ORBIT_TRY(fe_pack_wpb(Wp, bp, dt, sv.Wpb, d->V, f.Vp, f.P2, D, s));
  ORBIT_TRY(fe_make_g(sv.Wpb, dt, sv.Ut, sv.G, f.KVp, f.Vp, D, h, s));
  {
    GemmArgs g;
    g.A = sv.Wpb; g.a_rs = D; g.a_cs = 1; g.B = P->Wv; g.b_rs = D; g.b_cs = 1; g.C = sv.H; g.ldc = D;
    g.M = f.KVp; g.N = D; g.K = D; g.in_dtype = dt; g.out_dtype = dt;
    ORBIT_TRY(gemm(g, s));
  }
  // per patch: scores, softmax over the variables, A = alpha * pixext
  {   // writes the A operand [BL, heads, R Vp] once (the algorithmic bytes of the pixel-space front end)
    ProfScope prof(PROF_FRONT, (double)f.BL * h * (d->p * d->p + 1) * f.Vp * dsize(dt), s);
    ORBIT_TRY(fe_patch_fwd(x, sv.G, sv.alpha, sv.A, dt, d->V, f.Vp, d->Hg, d->Wg, d->p, h, f.BL, s));
  }
  {  // o_a = A_a H[:, a] + bv[a]   (strided batch over the heads; K = R*Vp)
    GemmArgs g;
    g.A = sv.A; g.a_rs = (long long)h * f.KVp; g.a_cs = 1; g.B = sv.H; g.b_rs = D; g.b_cs = 1;
    g.C = sv.o; g.ldc = D; g.M = f.BL; g.N = f.da; g.K = f.KVp; g.in_dtype = dt; g.out_dtype = dt;
    g.bias = P->bv; g.bias_dtype = dt;
    g.batch = h; g.a_bs = f.KVp; g.b_bs = f.da; g.c_bs = f.da; g.bias_bs = f.da;
    ORBIT_TRY(gemm(g, s));
  }
  {  // agg = o Wo + bo (+ pos[l])
    GemmArgs g;
    g.A = sv.o; g.a_rs = D; g.a_cs = 1; g.B = P->Wo; g.b_rs = D; g.b_cs = 1; g.C = agg; g.ldc = D;
    g.M = f.BL; g.N = D; g.K = D; g.in_dtype = dt; g.out_dtype = rt; g.bias = P->bo; g.bias_dtype = dt;
    if (pos) { g.resid = pos; g.resid_dtype = rt; g.ldr = D; g.resid_row_mod = f.L; }
    ORBIT_TRY(gemm(g, s));
  }
  return ORBIT_OK;
}

int orbit_embed_fused_bwd(const orbit_front_desc* d, const float* x, const void* Wp, const void* bp, const orbit_agg_params* P,
                          const void* dagg, const void* saved, void* dWp, void* dbp, orbit_agg_grads* G, void* dpos, void* ws,
                          size_t ws_bytes, void* stream) {
  ORBIT_TRY(check_front(d));
  ORBIT_TRY(check_front_params(P));
  if (!x || !Wp || !bp || !dagg || !saved || !dWp || !dbp || !G || !ws) { set_error("embed_fused_bwd: NULL pointer"); return ORBIT_ERR_NULL; }
  {
    void* gs[9] = {G->q, G->Wq, G->bq, G->Wk, G->bk, G->Wv, G->bv, G->Wo, G->bo};
    for (int i = 0; i < 9; i++) {
      if (!gs[i]) { set_error("embed_fused_bwd: NULL gradient pointer %d", i); return ORBIT_ERR_NULL; }
      if (!aligned16(gs[i])) { set_error("embed_fused_bwd: gradient %d not 16B aligned", i); return ORBIT_ERR_ALIGN; }
    }
  }
  if (!aligned16(x) || !aligned16(dagg) || !aligned16(saved) || !aligned16(dWp) || !aligned16(dbp) || !aligned16(ws) ||
      (dpos && !aligned16(dpos))) { set_error("embed_fused_bwd: pointer not 16B aligned"); return ORBIT_ERR_ALIGN; }
  if (ws_bytes < orbit_embed_fused_bwd_workspace_bytes(d)) { set_error("embed_fused_bwd: workspace too small"); return ORBIT_ERR_WORKSPACE; }
  ORBIT_TRY(check_device());
  cudaStream_t s = (cudaStream_t)stream;
  const FeDims f = fe_dims(*d);
  const int D = d->D, h = d->heads, dt = d->dtype, rt = d->resid_dtype, BL = f.BL;
  FeSaved sv = carve_fe_saved(*d, const_cast<void*>(saved));
  FeBwdWs w = carve_fe_bwd(*d, ws);
  float* acc_bo = w.acc;
  float* acc_bv = acc_bo + D;
  float* acc_dUt = acc_bv + D;
  float* dqt = acc_dUt + (size_t)D * h;
  ORBIT_TRY(fill_zero(w.acc, w.acc_floats * sizeof(float), s));
  ORBIT_TRY(fill_zero(w.dG, (size_t)f.KVp * FE_HP * sizeof(float), s));
  // dbo = colsum(dagg); dagg in the compute dtype; dpos
  const void* gb = dagg;
  if (rt != dt) { ORBIT_TRY(colsum(dagg, rt, D, BL, D, acc_bo, w.daggb, dt, D, s)); gb = w.daggb; }
  else ORBIT_TRY(colsum(dagg, rt, D, BL, D, acc_bo, nullptr, dt, D, s));
  if (dpos) ORBIT_TRY(agg_dpos(dagg, rt, dpos, d->B, f.L, D, s));
  {  // dWo = o^T dagg
    GemmArgs g;
    g.A = sv.o; g.a_rs = 1; g.a_cs = D; g.B = gb; g.b_rs = D; g.b_cs = 1; g.C = G->Wo; g.ldc = D;
    g.M = D; g.N = D; g.K = BL; g.in_dtype = dt; g.out_dtype = dt;
    ORBIT_TRY(gemm(g, s));
  }
  {  // do = dagg Wo^T
    GemmArgs g;
    g.A = gb; g.a_rs = D; g.a_cs = 1; g.B = P->Wo; g.b_rs = 1; g.b_cs = D; g.C = w.dob; g.ldc = D;
    g.M = BL; g.N = D; g.K = D; g.in_dtype = dt; g.out_dtype = dt;
    ORBIT_TRY(gemm(g, s));
  }
  ORBIT_TRY(colsum(w.dob, dt, D, BL, D, acc_bv, nullptr, dt, D, s));   // dbv = sum do   (sum_v alpha = 1)
  {  // dH[:, a] = A_a^T do_a
    GemmArgs g;
    g.A = sv.A; g.a_rs = 1; g.a_cs = (long long)h * f.KVp; g.B = w.dob; g.b_rs = D; g.b_cs = 1;
    g.C = w.dH; g.ldc = D; g.M = f.KVp; g.N = f.da; g.K = BL; g.in_dtype = dt; g.out_dtype = dt;
    g.batch = h; g.a_bs = f.KVp; g.b_bs = f.da; g.c_bs = f.da;
    ORBIT_TRY(gemm(g, s));
  }
  {  // dA_a = do_a H[:, a]^T
    GemmArgs g;
    g.A = w.dob; g.a_rs = D; g.a_cs = 1; g.B = sv.H; g.b_rs = 1; g.b_cs = D;
    g.C = w.dA; g.ldc = (long long)h * f.KVp; g.M = BL; g.N = f.KVp; g.K = f.da; g.in_dtype = dt; g.out_dtype = dt;
    g.batch = h; g.a_bs = f.da; g.b_bs = f.da; g.c_bs = f.KVp;
    ORBIT_TRY(gemm(g, s));
  }
  {  // dWv = Wpb^T dH
    GemmArgs g;
    g.A = sv.Wpb; g.a_rs = 1; g.a_cs = D; g.B = w.dH; g.b_rs = D; g.b_cs = 1; g.C = G->Wv; g.ldc = D;
    g.M = D; g.N = D; g.K = f.KVp; g.in_dtype = dt; g.out_dtype = dt;
    ORBIT_TRY(gemm(g, s));
  }
  {  // accW = dH Wv^T   (value path of dWpb, fp32)
    GemmArgs g;
    g.A = w.dH; g.a_rs = D; g.a_cs = 1; g.B = P->Wv; g.b_rs = 1; g.b_cs = D; g.C = w.accW; g.ldc = D;
    g.M = f.KVp; g.N = D; g.K = D; g.in_dtype = dt; g.out_dtype = ORBIT_F32;
    ORBIT_TRY(gemm(g, s));
  }
  // score path: ds per patch, dG = sum_bl pixext ds, dUt = Wpb^T dG
  {   // reads dA once
    ProfScope prof(PROF_FRONT, (double)BL * h * (d->p * d->p + 1) * f.Vp * dsize(dt), s);
    ORBIT_TRY(fe_patch_bwd(x, sv.alpha, w.dA, dt, w.dsT, d->V, f.Vp, d->Hg, d->Wg, d->p, h, BL, s));
  }
  ORBIT_TRY(fe_dg(x, w.dsT, w.dG, d->B, d->V, f.Vp, d->Hg, d->Wg, d->p, s));
  ORBIT_TRY(fe_dut(sv.Wpb, dt, w.dG, acc_dUt, f.KVp, D, h, s));
  ORBIT_TRY(fe_finish_dwp(w.accW, w.dG, sv.Ut, dWp, dbp, dt, d->V, f.Vp, f.P2, D, h, s));
  ORBIT_TRY(agg_param_bwd(acc_dUt, sv.qt, P->q, P->Wq, P->Wk, dt, G->Wk, G->bk, G->bq, G->Wq, G->q, dqt, D, h, s));
  ORBIT_TRY(cast_copy(acc_bo, ORBIT_F32, G->bo, dt, D, s));
  ORBIT_TRY(cast_copy(acc_bv, ORBIT_F32, G->bv, dt, D, s));
  return ORBIT_OK;
}

int orbit_debug_gemm_batched(int M, int N, int K, int batch, orbit_dtype dtype, const void* A, long long a_rs, long long a_cs,
                             long long a_bs, const void* B, long long b_rs, long long b_cs, long long b_bs, float* C,
                             long long ldc, long long c_bs, void* stream) {
  if (!A || !B || !C) { set_error("debug_gemm_batched: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!valid_dtype(dtype)) { set_error("debug_gemm_batched: bad dtype"); return ORBIT_ERR_DTYPE; }
  if (M <= 0 || N <= 0 || K <= 0 || batch <= 0) { set_error("debug_gemm_batched: bad shape"); return ORBIT_ERR_SHAPE; }
  ORBIT_TRY(check_device());
  GemmArgs g;
  g.A = A; g.a_rs = a_rs; g.a_cs = a_cs; g.B = B; g.b_rs = b_rs; g.b_cs = b_cs; g.C = C; g.ldc = ldc;
  g.M = M; g.N = N; g.K = K; g.in_dtype = dtype; g.out_dtype = ORBIT_F32;
  g.batch = batch; g.a_bs = a_bs; g.b_bs = b_bs; g.c_bs = c_bs;
  return gemm(g, (cudaStream_t)stream);
}

}  // extern "C"
