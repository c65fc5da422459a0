// api_block.cu -- orbit_block_fwd / orbit_block_bwd: one pre-LN ViT block with optional
// Hybrid-STOP shard-local mode (Eq. 1-3): T column/row shard pairs run one after another,
// fp32 partials combined on the device.  Host code only sequences kernels on the caller's stream.
#include "api_util.cuh"

namespace orbit {
namespace {

struct BlockSaved {
  float *mean1, *rstd1, *mean2, *rstd2, *lse;
  void *x, *a, *qkv, *O, *x1, *m, *u, *g;
  size_t bytes;
};
inline bool qk_norm(const orbit_block_desc& d) { return (d.flags & ORBIT_QK_NORM) != 0; }
inline bool recompute(const orbit_block_desc& d) { return (d.flags & ORBIT_RECOMPUTE) != 0; }
// columns of the per-shard qkv / dqkv buffers in units of dc = D/T: [Q | K | V] or, with QK-LayerNorm, [Q | K | V | Q' | K']
inline int qkv_cols(const orbit_block_desc& d) { return qk_norm(d) ? 5 : 3; }

// full forward state of a block (what backward reads)
BlockSaved carve_saved(const orbit_block_desc& d, void* base) {
  const size_t M = (size_t)d.B * d.N, D = d.D, F = d.F;
  const size_t es = dsize(d.dtype), rs = dsize(d.resid_dtype);
  Carver c(base);
  BlockSaved s;
  s.mean1 = c.take_n<float>(M); s.rstd1 = c.take_n<float>(M);
  s.mean2 = c.take_n<float>(M); s.rstd2 = c.take_n<float>(M);
  s.lse = c.take_n<float>((size_t)d.B * d.heads * d.N);
  s.x = c.take(M * D * rs);           // copy of the block input (LN1 backward needs it)
  s.a = c.take(M * D * es);
  s.qkv = c.take(M * qkv_cols(d) * D * es);   // T blocks of [M, 3D/T] ([M, 5D/T] with QK-LayerNorm)
  s.O = c.take(M * D * es);           // [M, D]; shard k owns columns k*D/T ..
  s.x1 = c.take(M * D * rs);
  s.m = c.take(M * D * es);
  s.u = c.take(M * F * es);           // [M, F]; shard k owns columns k*F/T ..
  s.g = c.take(M * F * es);
  s.bytes = c.off;
  return s;
}

struct BlockBwdWs {
  void *dyb, *du, *dx1b, *dO, *dqkv;
  float *dm, *dx1f, *da, *delta, *dq_acc;
  float *acc;                      // [bfc2 D | bfc1 F | bproj D | bqkv 3D | ln2_g D | ln2_b D | ln1_g D | ln1_b D | qk-norm 4 d_h]
  size_t acc_floats;
  // ORBIT_RECOMPUTE: the forward state is rebuilt here by orbit_block_bwd
  void *re_saved, *re_y, *re_part;
  size_t bytes;
};
BlockBwdWs carve_bwd(const orbit_block_desc& d, void* base) {
  const size_t M = (size_t)d.B * d.N, D = d.D, F = d.F;
  const size_t es = dsize(d.dtype);
  Carver c(base);
  BlockBwdWs w;
  w.acc_floats = 9 * D + F + 4 * (D / d.heads) + block_tail_tickets(F + 4 * D, 2 * d.T + 1);   // + the ticket words of block_tail()
  w.acc = c.take_n<float>(w.acc_floats);
  w.dyb = c.take(M * D * es);
  w.du = c.take(M * F * es);
  w.dm = c.take_n<float>(M * D);
  w.dx1f = c.take_n<float>(M * D);
  w.dx1b = c.take(M * D * es);
  w.dO = c.take(M * D * es);
  w.dqkv = c.take(M * qkv_cols(d) * D * es);
  w.da = c.take_n<float>(M * D);
  w.delta = c.take_n<float>((size_t)d.B * d.heads * d.N);
  w.dq_acc = c.take_n<float>(M * D);
  w.re_saved = w.re_y = w.re_part = nullptr;
  if (recompute(d)) {
    w.re_saved = c.take(carve_saved(d, nullptr).bytes);
    w.re_y = c.take(M * D * dsize(d.resid_dtype));
    w.re_part = c.take(M * D * sizeof(float));
  }
  w.bytes = c.off;
  return w;
}

}  // namespace

int check_block(const orbit_block_desc* d) {
  if (!d) { set_error("block desc is NULL"); return ORBIT_ERR_NULL; }
  if (!valid_dtype(d->dtype) || !valid_dtype(d->resid_dtype)) { set_error("block: bad dtype"); return ORBIT_ERR_DTYPE; }
  if (d->dtype == ORBIT_F32 && d->resid_dtype != ORBIT_F32) { set_error("block: resid_dtype must be F32 when dtype is F32"); return ORBIT_ERR_DTYPE; }
  if (d->flags & ~(ORBIT_QK_NORM | ORBIT_RECOMPUTE)) { set_error("block: unknown flag bits 0x%x", d->flags); return ORBIT_ERR_UNSUPPORTED; }
  if (d->B <= 0 || d->N <= 0 || d->D <= 0 || d->heads <= 0 || d->F <= 0 || d->T <= 0 || d->D % d->heads || d->heads % d->T ||
      d->F % d->T || d->D % 8 || (d->F / d->T) % 8 || (d->D / d->T) % 8 || (d->D / d->heads) > 256 || d->D > ORBIT_LN_MAX_D) {
    set_error("block: bad shape B=%d N=%d D=%d heads=%d F=%d T=%d (need D%%heads==0, heads%%T==0, F%%T==0, D%%8==0, "
              "(F/T)%%8==0, (D/T)%%8==0, d_h<=256, D<=16384)", d->B, d->N, d->D, d->heads, d->F, d->T);
    return ORBIT_ERR_SHAPE;
  }
  if ((d->flags & ORBIT_QK_NORM) && !qknorm_supported(d->D / d->heads)) {
    set_error("block: QK-LayerNorm needs d_h in {32, 64, 128, 192, 256} (d_h = %d)", d->D / d->heads);
    return ORBIT_ERR_SHAPE;
  }
  return ORBIT_OK;
}
static int check_params_n(const orbit_block_desc* d, const orbit_block_params* P, int nshards) {
  if (!P || !P->ln1_g || !P->ln1_b || !P->ln2_g || !P->ln2_b || !P->bproj || !P->bfc2 || !P->shards) { set_error("block: NULL parameter"); return ORBIT_ERR_NULL; }
  for (int k = 0; k < nshards; k++) {
    const orbit_block_shard& S = P->shards[k];
    if (!S.Wqkv || !S.bqkv || !S.Wproj || !S.Wfc1 || !S.bfc1 || !S.Wfc2) { set_error("block: NULL shard parameter (shard %d)", k); return ORBIT_ERR_NULL; }
    if (!aligned16(S.Wqkv) || !aligned16(S.bqkv) || !aligned16(S.Wproj) || !aligned16(S.Wfc1) || !aligned16(S.bfc1) || !aligned16(S.Wfc2)) { set_error("block: shard parameter not 16B aligned"); return ORBIT_ERR_ALIGN; }
  }
  if (!aligned16(P->ln1_g) || !aligned16(P->ln1_b) || !aligned16(P->ln2_g) || !aligned16(P->ln2_b) || !aligned16(P->bproj) || !aligned16(P->bfc2)) { set_error("block: parameter not 16B aligned"); return ORBIT_ERR_ALIGN; }
  if (d->flags & ORBIT_QK_NORM) {
    if (!P->qn_g || !P->qn_b || !P->kn_g || !P->kn_b) { set_error("block: NULL QK-LayerNorm parameter"); return ORBIT_ERR_NULL; }
    if (!aligned16(P->qn_g) || !aligned16(P->qn_b) || !aligned16(P->kn_g) || !aligned16(P->kn_b)) { set_error("block: QK-LayerNorm parameter not 16B aligned"); return ORBIT_ERR_ALIGN; }
  }
  return ORBIT_OK;
}

int check_block_params(const orbit_block_desc* d, const orbit_block_params* P) { return check_params_n(d, P, d->T); }
int check_shard_params(const orbit_block_desc* d, const orbit_block_params* P) { return check_params_n(d, P, 1); }

namespace {
AttnArgs attn_args(const orbit_block_desc& d, const BlockSaved& sv, int k) {
  const int dc = d.D / d.T, hk = d.heads / d.T, dh = d.D / d.heads;
  const size_t M = (size_t)d.B * d.N;
  AttnArgs a;
  const int nc = qkv_cols(d);
  a.qkv = offs(sv.qkv, (size_t)k * M * nc * dc, d.dtype);
  a.ld = (long long)nc * dc; a.v_off = 2 * dc;
  if (qk_norm(d)) { a.q_off = 3 * dc; a.k_off = 4 * dc; }     // attention reads the normalised Q', K'
  else { a.q_off = 0; a.k_off = dc; }
  a.B = d.B; a.N = d.N; a.heads = hk; a.dh = dh; a.dtype = d.dtype;
  a.O = offs(sv.O, (size_t)k * dc, d.dtype); a.ldo = d.D;
  a.lse = sv.lse + (size_t)k * d.B * hk * d.N;
  return a;
}
}  // namespace
}  // namespace orbit

using namespace orbit;

extern "C" {

size_t orbit_block_saved_bytes(const orbit_block_desc* d) {
  if (!d) return 0;
  if (recompute(*d)) return align_up((size_t)d->B * d->N * d->D * dsize(d->resid_dtype), 256);   // the block input only
  return carve_saved(*d, nullptr).bytes;
}
size_t orbit_block_fwd_workspace_bytes(const orbit_block_desc* d) {
  if (!d) return 0;
  size_t b = align_up((size_t)d->B * d->N * d->D * sizeof(float), 256) + 256;   // fp32 Hybrid-STOP partial sum
  if (recompute(*d)) b += carve_saved(*d, nullptr).bytes;                        // transient forward state
  return b;
}
size_t orbit_block_bwd_workspace_bytes(const orbit_block_desc* d) { return d ? carve_bwd(*d, nullptr).bytes : 0; }

// forward arithmetic of one block into the state `sv` (checks done by the callers); `copy_x`: keep a copy of x in sv.x
static int block_fwd_impl(const orbit_block_desc* d, const void* x, const orbit_block_params* P, void* y, BlockSaved& sv,
                          float* part, bool copy_x, cudaStream_t s) {
  const int M = d->B * d->N, D = d->D, F = d->F, T = d->T, dc = D / T, fc = F / T;
  const int dt = d->dtype, rt = d->resid_dtype;
  const int nc = qkv_cols(*d);
  // a3: a = LN1(x); qkv^k = a Wqkv^k + bqkv^k ; a4: attention on shard k's heads
  ORBIT_TRY(layernorm_fwd(x, rt, P->ln1_g, P->ln1_b, dt, sv.a, dt, sv.mean1, sv.rstd1, M, D, d->ln_eps, copy_x ? sv.x : nullptr, s));
  for (int k = 0; k < T; k++) {
    const orbit_block_shard& S = P->shards[k];
    GemmArgs g;
    g.A = sv.a; g.a_rs = D; g.a_cs = 1; g.B = S.Wqkv; g.b_rs = 3 * dc; g.b_cs = 1;
    g.C = offs(sv.qkv, (size_t)k * M * nc * dc, dt); g.ldc = (long long)nc * dc; g.M = M; g.N = 3 * dc; g.K = D;
    g.in_dtype = dt; g.out_dtype = dt; g.bias = S.bqkv; g.bias_dtype = dt;
    ORBIT_TRY(gemm(g, s));
    if (qk_norm(*d))   // Q', K' = LayerNorm over d_h of every head's q, k
      ORBIT_TRY(qknorm_fwd(g.C, g.ldc, M, d->heads / T, D / d->heads, dc, P->qn_g, P->qn_b, P->kn_g, P->kn_b, dt, dt, d->ln_eps, s));
    ORBIT_TRY(attention_fwd(attn_args(*d, sv, k), s));
  }
  // a5: x1 = x + sum_k O^k Wproj^k + bproj
  for (int k = 0; k < T; k++) {
    const orbit_block_shard& S = P->shards[k];
    GemmArgs g;
    g.A = offs(sv.O, (size_t)k * dc, dt); g.a_rs = D; g.a_cs = 1; g.B = S.Wproj; g.b_rs = D; g.b_cs = 1;
    g.M = M; g.N = D; g.K = dc; g.in_dtype = dt;
    if (T == 1) {
      g.C = sv.x1; g.ldc = D; g.out_dtype = rt; g.bias = P->bproj; g.bias_dtype = dt;
      g.resid = x; g.resid_dtype = rt; g.ldr = D;
    } else {
      g.C = part; g.ldc = D; g.out_dtype = ORBIT_F32; g.accumulate = k > 0;
    }
    ORBIT_TRY(gemm(g, s));
  }
  if (T > 1) ORBIT_TRY(add_partial(x, rt, part, P->bproj, dt, sv.x1, rt, M, D, s));
  // a6: m = LN2(x1); u^k = m Wfc1^k + bfc1^k; g^k = GELU(u^k); y = x1 + sum_k g^k Wfc2^k + bfc2
  ORBIT_TRY(layernorm_fwd(sv.x1, rt, P->ln2_g, P->ln2_b, dt, sv.m, dt, sv.mean2, sv.rstd2, M, D, d->ln_eps, nullptr, s));
  for (int k = 0; k < T; k++) {
    const orbit_block_shard& S = P->shards[k];
    GemmArgs g;
    g.A = sv.m; g.a_rs = D; g.a_cs = 1; g.B = S.Wfc1; g.b_rs = fc; g.b_cs = 1;
    g.C = offs(sv.g, (size_t)k * fc, dt); g.ldc = F; g.M = M; g.N = fc; g.K = D;
    g.in_dtype = dt; g.out_dtype = dt; g.bias = S.bfc1; g.bias_dtype = dt;
    g.act = ACT_GELU; g.aux_out = offs(sv.u, (size_t)k * fc, dt); g.ld_aux = F; g.aux_dtype = dt;
    ORBIT_TRY(gemm(g, s));
  }
  for (int k = 0; k < T; k++) {
    const orbit_block_shard& S = P->shards[k];
    GemmArgs g;
    g.A = offs(sv.g, (size_t)k * fc, dt); g.a_rs = F; g.a_cs = 1; g.B = S.Wfc2; g.b_rs = D; g.b_cs = 1;
    g.M = M; g.N = D; g.K = fc; g.in_dtype = dt;
    if (T == 1) {
      g.C = y; g.ldc = D; g.out_dtype = rt; g.bias = P->bfc2; g.bias_dtype = dt;
      g.resid = sv.x1; g.resid_dtype = rt; g.ldr = D;
    } else {
      g.C = part; g.ldc = D; g.out_dtype = ORBIT_F32; g.accumulate = k > 0;
    }
    ORBIT_TRY(gemm(g, s));
  }
  if (T > 1) ORBIT_TRY(add_partial(sv.x1, rt, part, P->bfc2, dt, y, rt, M, D, s));
  return ORBIT_OK;
}

int orbit_block_fwd(const orbit_block_desc* d, const void* x, const orbit_block_params* P, void* y, void* saved,
                    void* ws, size_t ws_bytes, void* stream) {
  ORBIT_TRY(check_block(d));
  ORBIT_TRY(check_block_params(d, P));
  if (!x || !y || !saved || !ws) { set_error("block_fwd: NULL pointer"); return ORBIT_ERR_NULL; }
  if (x == y) { set_error("block_fwd: in-place (y == x) not allowed"); return ORBIT_ERR_UNSUPPORTED; }
  if (!aligned16(x) || !aligned16(y) || !aligned16(saved) || !aligned16(ws)) { set_error("block_fwd: pointer not 16B aligned"); return ORBIT_ERR_ALIGN; }
  if (ws_bytes < orbit_block_fwd_workspace_bytes(d)) { set_error("block_fwd: workspace too small"); return ORBIT_ERR_WORKSPACE; }
  ORBIT_TRY(check_device());
  cudaStream_t s = (cudaStream_t)stream;
  const size_t part_bytes = align_up((size_t)d->B * d->N * d->D * sizeof(float), 256);
  if (recompute(*d)) {   // activation checkpointing: the state lives in ws, only the input copy persists
    BlockSaved sv = carve_saved(*d, (char*)ws + part_bytes);
    sv.x = saved;
    return block_fwd_impl(d, x, P, y, sv, (float*)ws, true, s);
  }
  BlockSaved sv = carve_saved(*d, saved);
  return block_fwd_impl(d, x, P, y, sv, (float*)ws, true, s);
}

int orbit_block_bwd(const orbit_block_desc* d, const void* dy, const orbit_block_params* P, const void* saved,
                    void* dx, orbit_block_grads* G, void* ws, size_t ws_bytes, void* stream) {
  ORBIT_TRY(check_block(d));
  ORBIT_TRY(check_block_params(d, P));
  if (!dy || !dx || !saved || !ws || !G || !G->shards || !G->ln1_g || !G->ln1_b || !G->ln2_g || !G->ln2_b || !G->bproj || !G->bfc2) { set_error("block_bwd: NULL pointer"); return ORBIT_ERR_NULL; }
  for (int k = 0; k < d->T; k++) {
    const orbit_block_shard_grads& S = G->shards[k];
    if (!S.Wqkv || !S.bqkv || !S.Wproj || !S.Wfc1 || !S.bfc1 || !S.Wfc2) { set_error("block_bwd: NULL shard gradient pointer"); return ORBIT_ERR_NULL; }
    if (!aligned16(S.Wqkv) || !aligned16(S.bqkv) || !aligned16(S.Wproj) || !aligned16(S.Wfc1) || !aligned16(S.bfc1) || !aligned16(S.Wfc2)) { set_error("block_bwd: shard gradient not 16B aligned"); return ORBIT_ERR_ALIGN; }
  }
  if (qk_norm(*d)) {   // checked before the first launch (the ORBIT_RECOMPUTE forward below already enqueues kernels)
    if (!G->qn_g || !G->qn_b || !G->kn_g || !G->kn_b) { set_error("block_bwd: NULL QK-LayerNorm gradient pointer"); return ORBIT_ERR_NULL; }
    if (!aligned16(G->qn_g) || !aligned16(G->qn_b) || !aligned16(G->kn_g) || !aligned16(G->kn_b)) { set_error("block_bwd: QK-LayerNorm gradient not 16B aligned"); return ORBIT_ERR_ALIGN; }
  }
  if (!aligned16(G->ln1_g) || !aligned16(G->ln1_b) || !aligned16(G->ln2_g) || !aligned16(G->ln2_b) || !aligned16(G->bproj) || !aligned16(G->bfc2)) { set_error("block_bwd: gradient not 16B aligned"); return ORBIT_ERR_ALIGN; }
  if (dx == dy) { set_error("block_bwd: in-place (dx == dy) not allowed"); return ORBIT_ERR_UNSUPPORTED; }
  if (!aligned16(dy) || !aligned16(dx) || !aligned16(saved) || !aligned16(ws)) { set_error("block_bwd: pointer not 16B aligned"); return ORBIT_ERR_ALIGN; }
  if (ws_bytes < orbit_block_bwd_workspace_bytes(d)) { set_error("block_bwd: workspace too small"); return ORBIT_ERR_WORKSPACE; }
  ORBIT_TRY(check_device());
  cudaStream_t s = (cudaStream_t)stream;
  const int M = d->B * d->N, D = d->D, F = d->F, T = d->T, dc = D / T, fc = F / T;
  const int dt = d->dtype, rt = d->resid_dtype;
  BlockBwdWs w = carve_bwd(*d, ws);
  BlockSaved sv = carve_saved(*d, recompute(*d) ? w.re_saved : const_cast<void*>(saved));
  if (recompute(*d)) {   // "the needed activation outputs are recomputed by rerunning the forward pass segment"
    sv.x = const_cast<void*>(saved);
    ORBIT_TRY(block_fwd_impl(d, saved, P, w.re_y, sv, (float*)w.re_part, false, s));
  }
  const int nc = qkv_cols(*d), dh = D / d->heads;
  float* acc_bfc2 = w.acc;
  float* acc_bfc1 = acc_bfc2 + D;
  float* acc_bproj = acc_bfc1 + F;
  float* acc_bqkv = acc_bproj + D;
  float* acc_ln2g = acc_bqkv + 3 * D;
  float* acc_ln2b = acc_ln2g + D;
  float* acc_ln1g = acc_ln2b + D;
  float* acc_ln1b = acc_ln1g + D;
  float* acc_qkn = acc_ln1b + D;          // [q gamma | q beta | k gamma | k beta], d_h each
  unsigned int* tickets = reinterpret_cast<unsigned int*>(acc_qkn + 4 * dh);
  // The column sums of du, dx1 and dqkv (bias gradients) are taken at the END of the call, in one launch together with the
  // fp32 -> dtype casts of all accumulators (block_tail): 4 launches fewer per block (C2: 226 -> 202 per step).
  const bool tail = 2 * T + 1 <= 12;
  TailSegs ts;
  ORBIT_TRY(fill_zero(w.acc, w.acc_floats * sizeof(float), s));

  // dbfc2 = colsum(dy); dy in the compute dtype for the contractions
  const void* dyb = dy;
  if (rt != dt) { ORBIT_TRY(colsum(dy, rt, D, M, D, acc_bfc2, w.dyb, dt, D, s)); dyb = w.dyb; }
  else ORBIT_TRY(colsum(dy, rt, D, M, D, acc_bfc2, nullptr, dt, D, s));
  // MLP backward
  for (int k = 0; k < T; k++) {
    const orbit_block_shard& S = P->shards[k];
    GemmArgs gw;   // dWfc2^k = g^k^T dy
    gw.A = offs(sv.g, (size_t)k * fc, dt); gw.a_rs = 1; gw.a_cs = F; gw.B = dyb; gw.b_rs = D; gw.b_cs = 1;
    gw.C = G->shards[k].Wfc2; gw.ldc = D; gw.M = fc; gw.N = D; gw.K = M; gw.in_dtype = dt; gw.out_dtype = dt;
    ORBIT_TRY(gemm(gw, s));
    GemmArgs gu;   // du^k = (dy Wfc2^k^T) o GELU'(u^k)
    gu.A = dyb; gu.a_rs = D; gu.a_cs = 1; gu.B = S.Wfc2; gu.b_rs = 1; gu.b_cs = D;
    gu.C = offs(w.du, (size_t)k * fc, dt); gu.ldc = F; gu.M = M; gu.N = fc; gu.K = D; gu.in_dtype = dt; gu.out_dtype = dt;
    gu.act = ACT_GELU_GRAD; gu.aux_in = offs(sv.u, (size_t)k * fc, dt); gu.ld_aux = F; gu.aux_dtype = dt;
    ORBIT_TRY(gemm(gu, s));
  }
  if (tail) for (int k = 0; k < T; k++) ts.add(offs(w.du, (size_t)k * fc, dt), dt, F, M, fc, acc_bfc1 + (size_t)k * fc, G->shards[k].bfc1);
  else ORBIT_TRY(colsum(w.du, dt, F, M, F, acc_bfc1, nullptr, dt, F, s));
  for (int k = 0; k < T; k++) {
    const orbit_block_shard& S = P->shards[k];
    GemmArgs gw;   // dWfc1^k = m^T du^k
    gw.A = sv.m; gw.a_rs = 1; gw.a_cs = D; gw.B = offs(w.du, (size_t)k * fc, dt); gw.b_rs = F; gw.b_cs = 1;
    gw.C = G->shards[k].Wfc1; gw.ldc = fc; gw.M = D; gw.N = fc; gw.K = M; gw.in_dtype = dt; gw.out_dtype = dt;
    ORBIT_TRY(gemm(gw, s));
    GemmArgs gm;   // dm += du^k Wfc1^k^T   (Eq. 3: partial activation gradients summed in fp32)
    gm.A = offs(w.du, (size_t)k * fc, dt); gm.a_rs = F; gm.a_cs = 1; gm.B = S.Wfc1; gm.b_rs = 1; gm.b_cs = fc;
    gm.C = w.dm; gm.ldc = D; gm.M = M; gm.N = D; gm.K = fc; gm.in_dtype = dt; gm.out_dtype = ORBIT_F32; gm.accumulate = k > 0;
    ORBIT_TRY(gemm(gm, s));
  }
  // dx1 = dy + LN2'(dm)
  ORBIT_TRY(layernorm_bwd(w.dm, ORBIT_F32, sv.x1, rt, sv.mean2, sv.rstd2, P->ln2_g, dt, dy, rt, w.dx1f, w.dx1b, dt,
                          acc_ln2g, acc_ln2b, M, D, s));
  if (tail) ts.add(w.dx1f, ORBIT_F32, D, M, D, acc_bproj, G->bproj);
  else ORBIT_TRY(colsum(w.dx1f, ORBIT_F32, D, M, D, acc_bproj, nullptr, dt, D, s));
  // attention sub-layer backward
  for (int k = 0; k < T; k++) {
    const orbit_block_shard& S = P->shards[k];
    GemmArgs gw;   // dWproj^k = O^k^T dx1
    gw.A = offs(sv.O, (size_t)k * dc, dt); gw.a_rs = 1; gw.a_cs = D; gw.B = w.dx1b; gw.b_rs = D; gw.b_cs = 1;
    gw.C = G->shards[k].Wproj; gw.ldc = D; gw.M = dc; gw.N = D; gw.K = M; gw.in_dtype = dt; gw.out_dtype = dt;
    ORBIT_TRY(gemm(gw, s));
    GemmArgs go;   // dO^k = dx1 Wproj^k^T
    go.A = w.dx1b; go.a_rs = D; go.a_cs = 1; go.B = S.Wproj; go.b_rs = 1; go.b_cs = D;
    go.C = offs(w.dO, (size_t)k * dc, dt); go.ldc = D; go.M = M; go.N = dc; go.K = D; go.in_dtype = dt; go.out_dtype = dt;
    ORBIT_TRY(gemm(go, s));
    AttnArgs a = attn_args(*d, sv, k);
    a.dO = offs(w.dO, (size_t)k * dc, dt); a.lddo = D;
    a.dqkv = offs(w.dqkv, (size_t)k * M * nc * dc, dt);
    a.delta = w.delta; a.dq_acc = w.dq_acc;
    ORBIT_TRY(attention_bwd(a, s));
    const long long ldq = (long long)nc * dc;
    if (qk_norm(*d))   // (dQ', dK') -> (dQ, dK) in columns [0, 2 dc) of dqkv; d gamma / d beta summed over tokens, heads, shards
      ORBIT_TRY(qknorm_bwd(a.qkv, a.dqkv, ldq, M, d->heads / T, dh, dc, P->qn_g, P->kn_g, dt, dt, d->ln_eps, acc_qkn, s));
    if (tail) ts.add(a.dqkv, dt, ldq, M, 3 * dc, acc_bqkv + (size_t)k * 3 * dc, G->shards[k].bqkv);
    else ORBIT_TRY(colsum(a.dqkv, dt, ldq, M, 3 * dc, acc_bqkv + (size_t)k * 3 * dc, nullptr, dt, 3 * dc, s));
    GemmArgs gq;   // dWqkv^k = a^T dqkv^k
    gq.A = sv.a; gq.a_rs = 1; gq.a_cs = D; gq.B = a.dqkv; gq.b_rs = ldq; gq.b_cs = 1;
    gq.C = G->shards[k].Wqkv; gq.ldc = 3 * dc; gq.M = D; gq.N = 3 * dc; gq.K = M; gq.in_dtype = dt; gq.out_dtype = dt;
    ORBIT_TRY(gemm(gq, s));
    GemmArgs ga;   // da += dqkv^k Wqkv^k^T
    ga.A = a.dqkv; ga.a_rs = ldq; ga.a_cs = 1; ga.B = S.Wqkv; ga.b_rs = 1; ga.b_cs = 3 * dc;
    ga.C = w.da; ga.ldc = D; ga.M = M; ga.N = D; ga.K = 3 * dc; ga.in_dtype = dt; ga.out_dtype = ORBIT_F32; ga.accumulate = k > 0;
    ORBIT_TRY(gemm(ga, s));
  }
  // dx = dx1 + LN1'(da)
  ORBIT_TRY(layernorm_bwd(w.da, ORBIT_F32, sv.x, rt, sv.mean1, sv.rstd1, P->ln1_g, dt, w.dx1f, ORBIT_F32,
                          nullptr, dx, rt, acc_ln1g, acc_ln1b, M, D, s));
  // fp32 accumulators -> gradient dtype
  CastSegs cs;
  cs.add(acc_bfc2, G->bfc2, D);
  if (!tail) cs.add(acc_bproj, G->bproj, D);
  cs.add(acc_ln2g, G->ln2_g, D); cs.add(acc_ln2b, G->ln2_b, D);
  cs.add(acc_ln1g, G->ln1_g, D); cs.add(acc_ln1b, G->ln1_b, D);
  if (qk_norm(*d)) {
    cs.add(acc_qkn, G->qn_g, dh); cs.add(acc_qkn + dh, G->qn_b, dh);
    cs.add(acc_qkn + 2 * dh, G->kn_g, dh); cs.add(acc_qkn + 3 * dh, G->kn_b, dh);
  }
  if (tail) {                             // the bias gradients of the sums above are cast by block_tail itself
    ORBIT_TRY(block_tail(ts, cs, dt, tickets, s));
    return ORBIT_OK;
  }
  for (int k = 0; k < T; k++) {
    if (cs.count > 13) { ORBIT_TRY(cast_multi(cs, dt, s)); cs.count = 0; }
    cs.add(acc_bfc1 + (size_t)k * fc, G->shards[k].bfc1, fc);
    cs.add(acc_bqkv + (size_t)k * 3 * dc, G->shards[k].bqkv, 3 * dc);
  }
  ORBIT_TRY(cast_multi(cs, dt, s));
  return ORBIT_OK;
}

}  // extern "C"
