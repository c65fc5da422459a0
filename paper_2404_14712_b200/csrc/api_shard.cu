// api_shard.cu -- orbit_rank_*: the rank-local Hybrid-STOP program (Fig. 3): what ONE rank of a
// tensor-parallel group computes between the collectives.  Rank k holds the column shards Wqkv^k, Wfc1^k and the row
// shards Wproj^k, Wfc2^k; "GPUs in each tensor-parallel group add their individual activations together"
// after the row-sharded products and "add their activation gradients together through all-reduce" after
// the transposed column-sharded products.  One block = six calls; between them the CALLER all-reduces (sum) the fp32
// [B, N, D] partial `part` over the group (NCCL over NVLink in production, gloo in the tests): the library itself holds no
// communicator.  Host code only sequences kernels on the caller's stream; same kernels as api_block.cu.
#include "api_util.cuh"

namespace orbit {
namespace {

inline bool qk_norm(const orbit_block_desc& d) { return (d.flags & ORBIT_QK_NORM) != 0; }
inline int qkv_cols(const orbit_block_desc& d) { return qk_norm(d) ? 5 : 3; }   // [Q | K | V] (+ [Q' | K'])

// forward state of this rank's shard (layout private to this file)
struct RankSaved {
  float *mean1, *rstd1, *mean2, *rstd2, *lse;
  void *x, *a, *qkv, *O, *x1, *m, *u, *g;
  size_t bytes;
};
RankSaved carve_rank_saved(const orbit_block_desc& d, void* base) {
  const size_t M = (size_t)d.B * d.N, D = d.D, dc = D / d.T, fc = (size_t)d.F / d.T;
  const size_t es = dsize(d.dtype), rs = dsize(d.resid_dtype);
  Carver c(base);
  RankSaved s;
  s.mean1 = c.take_n<float>(M); s.rstd1 = c.take_n<float>(M);
  s.mean2 = c.take_n<float>(M); s.rstd2 = c.take_n<float>(M);
  s.lse = c.take_n<float>((size_t)d.B * (d.heads / d.T) * d.N);
  s.x = c.take(M * D * rs);
  s.a = c.take(M * D * es);
  s.qkv = c.take(M * qkv_cols(d) * dc * es);
  s.O = c.take(M * dc * es);
  s.x1 = c.take(M * D * rs);
  s.m = c.take(M * D * es);
  s.u = c.take(M * fc * es);
  s.g = c.take(M * fc * es);
  s.bytes = c.off;
  return s;
}

// backward workspace: carried UNCHANGED through orbit_rank_bwd_mlp -> _attn -> _out (fp32 accumulators, dx1)
struct RankBwdWs {
  float *acc;                 // [bfc2 D | bfc1 F/T | bproj D | bqkv 3D/T | ln2_g D | ln2_b D | ln1_g D | ln1_b D | qk-norm 4 d_h]
  size_t acc_floats;
  void *dyb, *du, *dx1b, *dO, *dqkv;
  float *dx1f, *delta, *dq_acc;
  size_t bytes;
};
RankBwdWs carve_rank_bwd(const orbit_block_desc& d, void* base) {
  const size_t M = (size_t)d.B * d.N, D = d.D, dc = D / d.T, fc = (size_t)d.F / d.T;
  const size_t es = dsize(d.dtype);
  Carver c(base);
  RankBwdWs w;
  w.acc_floats = 6 * D + fc + 3 * dc + 4 * (D / d.heads);
  w.acc = c.take_n<float>(w.acc_floats);
  w.dyb = c.take(M * D * es);
  w.du = c.take(M * fc * es);
  w.dx1f = c.take_n<float>(M * D);
  w.dx1b = c.take(M * D * es);
  w.dO = c.take(M * dc * es);
  w.dqkv = c.take(M * qkv_cols(d) * dc * es);
  w.delta = c.take_n<float>((size_t)d.B * (d.heads / d.T) * d.N);
  w.dq_acc = c.take_n<float>(M * dc);
  w.bytes = c.off;
  return w;
}
struct Acc { float *bfc2, *bfc1, *bproj, *bqkv, *ln2g, *ln2b, *ln1g, *ln1b, *qkn; };
Acc acc_of(const orbit_block_desc& d, const RankBwdWs& w) {
  const size_t D = d.D, dc = D / d.T, fc = (size_t)d.F / d.T;
  Acc a;
  a.bfc2 = w.acc; a.bfc1 = a.bfc2 + D; a.bproj = a.bfc1 + fc; a.bqkv = a.bproj + D;
  a.ln2g = a.bqkv + 3 * dc; a.ln2b = a.ln2g + D; a.ln1g = a.ln2b + D; a.ln1b = a.ln1g + D; a.qkn = a.ln1b + D;
  return a;
}

int check_rank(const orbit_block_desc* d) {
  ORBIT_TRY(check_block(d));
  if (d->flags & ORBIT_RECOMPUTE) { set_error("rank-local mode: ORBIT_RECOMPUTE is not supported"); return ORBIT_ERR_UNSUPPORTED; }
  return ORBIT_OK;
}
int check_rank_grads(const orbit_block_desc* d, const orbit_block_grads* G) {
  if (!G || !G->shards || !G->ln1_g || !G->ln1_b || !G->ln2_g || !G->ln2_b || !G->bproj || !G->bfc2) { set_error("rank_bwd: NULL gradient pointer"); return ORBIT_ERR_NULL; }
  const orbit_block_shard_grads& S = G->shards[0];
  if (!S.Wqkv || !S.bqkv || !S.Wproj || !S.Wfc1 || !S.bfc1 || !S.Wfc2) { set_error("rank_bwd: NULL shard gradient pointer"); return ORBIT_ERR_NULL; }
  if (!aligned16(S.Wqkv) || !aligned16(S.bqkv) || !aligned16(S.Wproj) || !aligned16(S.Wfc1) || !aligned16(S.bfc1) || !aligned16(S.Wfc2) ||
      !aligned16(G->ln1_g) || !aligned16(G->ln1_b) || !aligned16(G->ln2_g) || !aligned16(G->ln2_b) || !aligned16(G->bproj) || !aligned16(G->bfc2)) {
    set_error("rank_bwd: gradient not 16B aligned"); return ORBIT_ERR_ALIGN;
  }
  if (d->flags & ORBIT_QK_NORM) {
    if (!G->qn_g || !G->qn_b || !G->kn_g || !G->kn_b) { set_error("rank_bwd: NULL QK-LayerNorm gradient pointer"); return ORBIT_ERR_NULL; }
    if (!aligned16(G->qn_g) || !aligned16(G->qn_b) || !aligned16(G->kn_g) || !aligned16(G->kn_b)) { set_error("rank_bwd: QK-LayerNorm gradient not 16B aligned"); return ORBIT_ERR_ALIGN; }
  }
  return ORBIT_OK;
}

AttnArgs rank_attn_args(const orbit_block_desc& d, const RankSaved& sv) {
  const int dc = d.D / d.T;
  AttnArgs a;
  const int nc = qkv_cols(d);
  a.qkv = sv.qkv; a.ld = (long long)nc * dc; a.v_off = 2 * dc;
  if (qk_norm(d)) { a.q_off = 3 * dc; a.k_off = 4 * dc; } else { a.q_off = 0; a.k_off = dc; }
  a.B = d.B; a.N = d.N; a.heads = d.heads / d.T; a.dh = d.D / d.heads; a.dtype = d.dtype;
  a.O = sv.O; a.ldo = dc; a.lse = sv.lse;
  return a;
}
}  // namespace
}  // namespace orbit

using namespace orbit;

extern "C" {

size_t orbit_rank_saved_bytes(const orbit_block_desc* d) { return d ? carve_rank_saved(*d, nullptr).bytes : 0; }
size_t orbit_rank_bwd_workspace_bytes(const orbit_block_desc* d) { return d ? carve_rank_bwd(*d, nullptr).bytes : 0; }

int orbit_rank_fwd_attn(const orbit_block_desc* d, const void* x, const orbit_block_params* P, float* part, void* saved,
                        void* stream) {
  ORBIT_TRY(check_rank(d));
  ORBIT_TRY(check_shard_params(d, P));
  if (!x || !part || !saved) { set_error("rank_fwd_attn: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!aligned16(x) || !aligned16(part) || !aligned16(saved)) { set_error("rank_fwd_attn: pointer not 16B aligned"); return ORBIT_ERR_ALIGN; }
  ORBIT_TRY(check_device());
  cudaStream_t s = (cudaStream_t)stream;
  const int M = d->B * d->N, D = d->D, dc = D / d->T, dt = d->dtype, rt = d->resid_dtype, nc = qkv_cols(*d);
  RankSaved sv = carve_rank_saved(*d, saved);
  const orbit_block_shard& S = P->shards[0];
  ORBIT_TRY(layernorm_fwd(x, rt, P->ln1_g, P->ln1_b, dt, sv.a, dt, sv.mean1, sv.rstd1, M, D, d->ln_eps, sv.x, s));
  GemmArgs g;                      // qkv^k = a Wqkv^k + bqkv^k   (column shard)
  g.A = sv.a; g.a_rs = D; g.a_cs = 1; g.B = S.Wqkv; g.b_rs = 3 * dc; g.b_cs = 1;
  g.C = sv.qkv; g.ldc = (long long)nc * dc; g.M = M; g.N = 3 * dc; g.K = D;
  g.in_dtype = dt; g.out_dtype = dt; g.bias = S.bqkv; g.bias_dtype = dt;
  ORBIT_TRY(gemm(g, s));
  if (qk_norm(*d))
    ORBIT_TRY(qknorm_fwd(sv.qkv, g.ldc, M, d->heads / d->T, D / d->heads, dc, P->qn_g, P->qn_b, P->kn_g, P->kn_b, dt, dt, d->ln_eps, s));
  ORBIT_TRY(attention_fwd(rank_attn_args(*d, sv), s));
  GemmArgs p;                      // part = O^k Wproj^k   (row shard: a partial of the full product, Eq. 2)
  p.A = sv.O; p.a_rs = dc; p.a_cs = 1; p.B = S.Wproj; p.b_rs = D; p.b_cs = 1;
  p.C = part; p.ldc = D; p.M = M; p.N = D; p.K = dc; p.in_dtype = dt; p.out_dtype = ORBIT_F32;
  ORBIT_TRY(gemm(p, s));
  return ORBIT_OK;
}

int orbit_rank_fwd_mlp(const orbit_block_desc* d, const orbit_block_params* P, float* part, void* saved, void* stream) {
  ORBIT_TRY(check_rank(d));
  ORBIT_TRY(check_shard_params(d, P));
  if (!part || !saved) { set_error("rank_fwd_mlp: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!aligned16(part) || !aligned16(saved)) { set_error("rank_fwd_mlp: pointer not 16B aligned"); return ORBIT_ERR_ALIGN; }
  ORBIT_TRY(check_device());
  cudaStream_t s = (cudaStream_t)stream;
  const int M = d->B * d->N, D = d->D, fc = d->F / d->T, dt = d->dtype, rt = d->resid_dtype;
  RankSaved sv = carve_rank_saved(*d, saved);
  const orbit_block_shard& S = P->shards[0];
  // x1 = x + sum_k part^k + bproj: bias and residual enter once, after the combine (R14)
  ORBIT_TRY(add_partial(sv.x, rt, part, P->bproj, dt, sv.x1, rt, M, D, s));
  ORBIT_TRY(layernorm_fwd(sv.x1, rt, P->ln2_g, P->ln2_b, dt, sv.m, dt, sv.mean2, sv.rstd2, M, D, d->ln_eps, nullptr, s));
  GemmArgs g;                      // u^k = m Wfc1^k + bfc1^k; g^k = GELU(u^k)
  g.A = sv.m; g.a_rs = D; g.a_cs = 1; g.B = S.Wfc1; g.b_rs = fc; g.b_cs = 1;
  g.C = sv.g; g.ldc = fc; g.M = M; g.N = fc; g.K = D; g.in_dtype = dt; g.out_dtype = dt; g.bias = S.bfc1; g.bias_dtype = dt;
  g.act = ACT_GELU; g.aux_out = sv.u; g.ld_aux = fc; g.aux_dtype = dt;
  ORBIT_TRY(gemm(g, s));
  GemmArgs p;                      // part = g^k Wfc2^k
  p.A = sv.g; p.a_rs = fc; p.a_cs = 1; p.B = S.Wfc2; p.b_rs = D; p.b_cs = 1;
  p.C = part; p.ldc = D; p.M = M; p.N = D; p.K = fc; p.in_dtype = dt; p.out_dtype = ORBIT_F32;
  ORBIT_TRY(gemm(p, s));
  return ORBIT_OK;
}

int orbit_rank_fwd_out(const orbit_block_desc* d, const orbit_block_params* P, const float* part, void* y, const void* saved,
                       void* stream) {
  ORBIT_TRY(check_rank(d));
  ORBIT_TRY(check_shard_params(d, P));
  if (!part || !y || !saved) { set_error("rank_fwd_out: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!aligned16(part) || !aligned16(y) || !aligned16(saved)) { set_error("rank_fwd_out: pointer not 16B aligned"); return ORBIT_ERR_ALIGN; }
  ORBIT_TRY(check_device());
  RankSaved sv = carve_rank_saved(*d, const_cast<void*>(saved));
  return add_partial(sv.x1, d->resid_dtype, part, P->bfc2, d->dtype, y, d->resid_dtype, d->B * d->N, d->D, (cudaStream_t)stream);
}

int orbit_rank_bwd_mlp(const orbit_block_desc* d, const void* dy, const orbit_block_params* P, const void* saved,
                       orbit_block_grads* G, float* part, void* ws, size_t ws_bytes, void* stream) {
  ORBIT_TRY(check_rank(d));
  ORBIT_TRY(check_shard_params(d, P));
  ORBIT_TRY(check_rank_grads(d, G));
  if (!dy || !saved || !part || !ws) { set_error("rank_bwd_mlp: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!aligned16(dy) || !aligned16(saved) || !aligned16(part) || !aligned16(ws)) { set_error("rank_bwd_mlp: pointer not 16B aligned"); return ORBIT_ERR_ALIGN; }
  if (ws_bytes < orbit_rank_bwd_workspace_bytes(d)) { set_error("rank_bwd_mlp: workspace too small"); return ORBIT_ERR_WORKSPACE; }
  ORBIT_TRY(check_device());
  cudaStream_t s = (cudaStream_t)stream;
  const int M = d->B * d->N, D = d->D, fc = d->F / d->T, dt = d->dtype, rt = d->resid_dtype;
  RankSaved sv = carve_rank_saved(*d, const_cast<void*>(saved));
  RankBwdWs w = carve_rank_bwd(*d, ws);
  const Acc a = acc_of(*d, w);
  const orbit_block_shard& S = P->shards[0];
  ORBIT_TRY(fill_zero(w.acc, w.acc_floats * sizeof(float), s));
  const void* dyb = dy;            // dbfc2 = colsum(dy) (replicated: every rank computes the same sum)
  if (rt != dt) { ORBIT_TRY(colsum(dy, rt, D, M, D, a.bfc2, w.dyb, dt, D, s)); dyb = w.dyb; }
  else ORBIT_TRY(colsum(dy, rt, D, M, D, a.bfc2, nullptr, dt, D, s));
  GemmArgs gw;                     // dWfc2^k = g^k^T dy
  gw.A = sv.g; gw.a_rs = 1; gw.a_cs = fc; gw.B = dyb; gw.b_rs = D; gw.b_cs = 1;
  gw.C = G->shards[0].Wfc2; gw.ldc = D; gw.M = fc; gw.N = D; gw.K = M; gw.in_dtype = dt; gw.out_dtype = dt;
  ORBIT_TRY(gemm(gw, s));
  GemmArgs gu;                     // du^k = (dy Wfc2^k^T) o GELU'(u^k)
  gu.A = dyb; gu.a_rs = D; gu.a_cs = 1; gu.B = S.Wfc2; gu.b_rs = 1; gu.b_cs = D;
  gu.C = w.du; gu.ldc = fc; gu.M = M; gu.N = fc; gu.K = D; gu.in_dtype = dt; gu.out_dtype = dt;
  gu.act = ACT_GELU_GRAD; gu.aux_in = sv.u; gu.ld_aux = fc; gu.aux_dtype = dt;
  ORBIT_TRY(gemm(gu, s));
  ORBIT_TRY(colsum(w.du, dt, fc, M, fc, a.bfc1, nullptr, dt, fc, s));
  GemmArgs g1;                     // dWfc1^k = m^T du^k
  g1.A = sv.m; g1.a_rs = 1; g1.a_cs = D; g1.B = w.du; g1.b_rs = fc; g1.b_cs = 1;
  g1.C = G->shards[0].Wfc1; g1.ldc = fc; g1.M = D; g1.N = fc; g1.K = M; g1.in_dtype = dt; g1.out_dtype = dt;
  ORBIT_TRY(gemm(g1, s));
  GemmArgs gm;                     // part = du^k Wfc1^k^T   (Eq. 3: this rank's partial of dm)
  gm.A = w.du; gm.a_rs = fc; gm.a_cs = 1; gm.B = S.Wfc1; gm.b_rs = 1; gm.b_cs = fc;
  gm.C = part; gm.ldc = D; gm.M = M; gm.N = D; gm.K = fc; gm.in_dtype = dt; gm.out_dtype = ORBIT_F32;
  ORBIT_TRY(gemm(gm, s));
  return ORBIT_OK;
}

int orbit_rank_bwd_attn(const orbit_block_desc* d, const void* dy, const orbit_block_params* P, const void* saved,
                        orbit_block_grads* G, float* part, void* ws, size_t ws_bytes, void* stream) {
  ORBIT_TRY(check_rank(d));
  ORBIT_TRY(check_shard_params(d, P));
  ORBIT_TRY(check_rank_grads(d, G));
  if (!dy || !saved || !part || !ws) { set_error("rank_bwd_attn: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!aligned16(dy) || !aligned16(saved) || !aligned16(part) || !aligned16(ws)) { set_error("rank_bwd_attn: pointer not 16B aligned"); return ORBIT_ERR_ALIGN; }
  if (ws_bytes < orbit_rank_bwd_workspace_bytes(d)) { set_error("rank_bwd_attn: workspace too small"); return ORBIT_ERR_WORKSPACE; }
  ORBIT_TRY(check_device());
  cudaStream_t s = (cudaStream_t)stream;
  const int M = d->B * d->N, D = d->D, dc = D / d->T, dt = d->dtype, rt = d->resid_dtype, nc = qkv_cols(*d), dh = D / d->heads;
  RankSaved sv = carve_rank_saved(*d, const_cast<void*>(saved));
  RankBwdWs w = carve_rank_bwd(*d, ws);
  const Acc a = acc_of(*d, w);
  const orbit_block_shard& S = P->shards[0];
  // dx1 = dy + LN2'(dm), dm = the all-reduced `part`
  ORBIT_TRY(layernorm_bwd(part, ORBIT_F32, sv.x1, rt, sv.mean2, sv.rstd2, P->ln2_g, dt, dy, rt, w.dx1f, w.dx1b, dt, a.ln2g, a.ln2b, M, D, s));
  ORBIT_TRY(colsum(w.dx1f, ORBIT_F32, D, M, D, a.bproj, nullptr, dt, D, s));
  GemmArgs gw;                     // dWproj^k = O^k^T dx1
  gw.A = sv.O; gw.a_rs = 1; gw.a_cs = dc; gw.B = w.dx1b; gw.b_rs = D; gw.b_cs = 1;
  gw.C = G->shards[0].Wproj; gw.ldc = D; gw.M = dc; gw.N = D; gw.K = M; gw.in_dtype = dt; gw.out_dtype = dt;
  ORBIT_TRY(gemm(gw, s));
  GemmArgs go;                     // dO^k = dx1 Wproj^k^T
  go.A = w.dx1b; go.a_rs = D; go.a_cs = 1; go.B = S.Wproj; go.b_rs = 1; go.b_cs = D;
  go.C = w.dO; go.ldc = dc; go.M = M; go.N = dc; go.K = D; go.in_dtype = dt; go.out_dtype = dt;
  ORBIT_TRY(gemm(go, s));
  AttnArgs at = rank_attn_args(*d, sv);
  at.dO = w.dO; at.lddo = dc; at.dqkv = w.dqkv; at.delta = w.delta; at.dq_acc = w.dq_acc;
  ORBIT_TRY(attention_bwd(at, s));
  const long long ldq = (long long)nc * dc;
  if (qk_norm(*d))
    ORBIT_TRY(qknorm_bwd(at.qkv, at.dqkv, ldq, M, d->heads / d->T, dh, dc, P->qn_g, P->kn_g, dt, dt, d->ln_eps, a.qkn, s));
  ORBIT_TRY(colsum(at.dqkv, dt, ldq, M, 3 * dc, a.bqkv, nullptr, dt, 3 * dc, s));
  GemmArgs gq;                     // dWqkv^k = a^T dqkv^k
  gq.A = sv.a; gq.a_rs = 1; gq.a_cs = D; gq.B = at.dqkv; gq.b_rs = ldq; gq.b_cs = 1;
  gq.C = G->shards[0].Wqkv; gq.ldc = 3 * dc; gq.M = D; gq.N = 3 * dc; gq.K = M; gq.in_dtype = dt; gq.out_dtype = dt;
  ORBIT_TRY(gemm(gq, s));
  GemmArgs ga;                     // part = dqkv^k Wqkv^k^T   (this rank's partial of da)
  ga.A = at.dqkv; ga.a_rs = ldq; ga.a_cs = 1; ga.B = S.Wqkv; ga.b_rs = 1; ga.b_cs = 3 * dc;
  ga.C = part; ga.ldc = D; ga.M = M; ga.N = D; ga.K = 3 * dc; ga.in_dtype = dt; ga.out_dtype = ORBIT_F32;
  ORBIT_TRY(gemm(ga, s));
  return ORBIT_OK;
}

int orbit_rank_bwd_out(const orbit_block_desc* d, const orbit_block_params* P, const void* saved, orbit_block_grads* G,
                       const float* part, void* dx, void* ws, size_t ws_bytes, void* stream) {
  ORBIT_TRY(check_rank(d));
  ORBIT_TRY(check_shard_params(d, P));
  ORBIT_TRY(check_rank_grads(d, G));
  if (!saved || !part || !dx || !ws) { set_error("rank_bwd_out: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!aligned16(saved) || !aligned16(part) || !aligned16(dx) || !aligned16(ws)) { set_error("rank_bwd_out: pointer not 16B aligned"); return ORBIT_ERR_ALIGN; }
  if (ws_bytes < orbit_rank_bwd_workspace_bytes(d)) { set_error("rank_bwd_out: workspace too small"); return ORBIT_ERR_WORKSPACE; }
  ORBIT_TRY(check_device());
  cudaStream_t s = (cudaStream_t)stream;
  const int M = d->B * d->N, D = d->D, dc = D / d->T, fc = d->F / d->T, dt = d->dtype, rt = d->resid_dtype, dh = D / d->heads;
  RankSaved sv = carve_rank_saved(*d, const_cast<void*>(saved));
  RankBwdWs w = carve_rank_bwd(*d, ws);
  const Acc a = acc_of(*d, w);
  // dx = dx1 + LN1'(da), da = the all-reduced `part`
  ORBIT_TRY(layernorm_bwd(part, ORBIT_F32, sv.x, rt, sv.mean1, sv.rstd1, P->ln1_g, dt, w.dx1f, ORBIT_F32, nullptr, dx, rt, a.ln1g, a.ln1b, M, D, s));
  CastSegs cs;
  cs.add(a.bfc2, G->bfc2, D); cs.add(a.bproj, G->bproj, D);
  cs.add(a.ln2g, G->ln2_g, D); cs.add(a.ln2b, G->ln2_b, D);
  cs.add(a.ln1g, G->ln1_g, D); cs.add(a.ln1b, G->ln1_b, D);
  cs.add(a.bfc1, G->shards[0].bfc1, fc); cs.add(a.bqkv, G->shards[0].bqkv, 3 * dc);
  if (qk_norm(*d)) {
    cs.add(a.qkn, G->qn_g, dh); cs.add(a.qkn + dh, G->qn_b, dh);
    cs.add(a.qkn + 2 * dh, G->kn_g, dh); cs.add(a.qkn + 3 * dh, G->kn_b, dh);
  }
  ORBIT_TRY(cast_multi(cs, dt, s));
  return ORBIT_OK;
}

}  // extern "C"
