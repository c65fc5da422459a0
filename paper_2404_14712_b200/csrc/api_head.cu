// api_head.cu -- orbit_head_loss / orbit_head_loss_bwd: final LayerNorm, projection to the image space and
// latitude-weighted MSE, readings R26-R28.  The un-patchify is index arithmetic
// inside the loss kernel: pred / target are addressed in image layout, P / dP in token layout.
#include <math.h>
#include "api_util.cuh"

namespace orbit {
namespace {

// w_y = cos(lat_y) / mean cos, lat_y = -90 + (y + 1/2) 180 / Hg  (one block; double precision: Hg values)
__global__ void latw_kernel(float* __restrict__ w, int Hg) {
  __shared__ double sh[32];
  __shared__ double tot;
  double acc = 0.0;
  for (int y = threadIdx.x; y < Hg; y += blockDim.x) acc += cos((-90.0 + (y + 0.5) * 180.0 / Hg) * 0.017453292519943295);
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int i = 0; i < (int)(blockDim.x + 31) / 32; i++) t += sh[i];
    tot = t;
  }
  __syncthreads();
  const double mean = tot / Hg;
  for (int y = threadIdx.x; y < Hg; y += blockDim.x)
    w[y] = (float)(cos((-90.0 + (y + 0.5) * 180.0 / Hg) * 0.017453292519943295) / mean);
}

// one thread per element of P [B*L, C]: diff against the target pixel, weighted square into the loss, dP = 2 w diff / n
template <typename T>
__global__ void __launch_bounds__(256) wmse_kernel(const float* __restrict__ P, const float* __restrict__ target,
    const float* __restrict__ w, float* __restrict__ pred, T* __restrict__ dP, float* __restrict__ loss, int B, int V, int Hg,
    int Wg, int p) {
  __shared__ float sh[32];
  const int gw = Wg / p, L = (Hg / p) * gw, P2 = p * p, C = V * P2;
  const size_t n = (size_t)B * L * C;
  const float inv = 1.0f / (float)n;
  float acc = 0.f;
  for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += (size_t)gridDim.x * blockDim.x) {
    const int c = (int)(idx % C);
    const size_t bl = idx / C;
    const int b = (int)(bl / L), l = (int)(bl - (size_t)b * L), i = l / gw, j = l - i * gw;
    const int v = c / P2, r = c - v * P2, di = r / p, dj = r - di * p;
    const int y = i * p + di;
    const size_t img = (((size_t)b * V + v) * Hg + y) * Wg + (size_t)j * p + dj;
    const float pv = P[idx];
    const float diff = pv - target[img], wy = w[y];
    if (pred) pred[img] = pv;
    acc = fmaf(wy * diff, diff, acc);
    dP[idx] = from_f<T>(2.f * wy * diff * inv);
  }
  acc = block_sum(acc, sh);
  if (threadIdx.x == 0) atomicAdd(loss, acc * inv);
}

struct HeadDims { int L, BL, C; };
HeadDims head_dims(const orbit_head_desc& d) {
  HeadDims h;
  h.L = (d.Hg / d.p) * (d.Wg / d.p); h.BL = d.B * h.L; h.C = d.V * d.p * d.p;
  return h;
}
struct HeadSaved { float *mean, *rstd; void *zn, *dP; size_t bytes; };
HeadSaved carve_head_saved(const orbit_head_desc& d, void* base) {
  const HeadDims h = head_dims(d);
  Carver c(base);
  HeadSaved s;
  s.mean = c.take_n<float>(h.BL); s.rstd = c.take_n<float>(h.BL);
  s.zn = c.take((size_t)h.BL * d.D * dsize(d.dtype));
  s.dP = c.take((size_t)h.BL * h.C * dsize(d.dtype));
  s.bytes = c.off;
  return s;
}
struct HeadFwdWs { float *P, *latw; size_t bytes; };
HeadFwdWs carve_head_fwd(const orbit_head_desc& d, void* base) {
  const HeadDims h = head_dims(d);
  Carver c(base);
  HeadFwdWs w;
  w.P = c.take_n<float>((size_t)h.BL * h.C);
  w.latw = c.take_n<float>(d.Hg);
  w.bytes = c.off;
  return w;
}
struct HeadBwdWs { float *acc, *dzn; size_t acc_floats; size_t bytes; };   // acc = [bh C | lnf_g D | lnf_b D]
HeadBwdWs carve_head_bwd(const orbit_head_desc& d, void* base) {
  const HeadDims h = head_dims(d);
  Carver c(base);
  HeadBwdWs w;
  w.acc_floats = (size_t)h.C + 2 * d.D;
  w.acc = c.take_n<float>(w.acc_floats);
  w.dzn = c.take_n<float>((size_t)h.BL * d.D);
  w.bytes = c.off;
  return w;
}
int check_head(const orbit_head_desc* d) {
  if (!d) { set_error("head desc is NULL"); return ORBIT_ERR_NULL; }
  if (!valid_dtype(d->dtype) || !valid_dtype(d->resid_dtype)) { set_error("head: bad dtype"); return ORBIT_ERR_DTYPE; }
  if (d->dtype == ORBIT_F32 && d->resid_dtype != ORBIT_F32) { set_error("head: resid_dtype must be F32 when dtype is F32"); return ORBIT_ERR_DTYPE; }
  if (d->B <= 0 || d->V <= 0 || d->Hg <= 0 || d->Wg <= 0 || d->p <= 0 || d->D <= 0 || d->Hg % d->p || d->Wg % d->p || d->D % 8 ||
      (d->V * d->p * d->p) % 8 || d->D > ORBIT_LN_MAX_D) {
    set_error("head: bad shape B=%d V=%d grid=%dx%d p=%d D=%d (need Hg%%p==0, Wg%%p==0, D%%8==0, (V p^2)%%8==0, D<=16384)", d->B, d->V,
              d->Hg, d->Wg, d->p, d->D);
    return ORBIT_ERR_SHAPE;
  }
  return ORBIT_OK;
}
}  // namespace
}  // namespace orbit

using namespace orbit;

extern "C" {

size_t orbit_head_loss_saved_bytes(const orbit_head_desc* d) { return d ? carve_head_saved(*d, nullptr).bytes : 0; }
size_t orbit_head_loss_workspace_bytes(const orbit_head_desc* d) { return d ? carve_head_fwd(*d, nullptr).bytes : 0; }
size_t orbit_head_loss_bwd_workspace_bytes(const orbit_head_desc* d) { return d ? carve_head_bwd(*d, nullptr).bytes : 0; }

int orbit_head_loss(const orbit_head_desc* d, const void* z, const void* lnf_g, const void* lnf_b, const void* Wh, const void* bh,
                    const float* target, const float* latw, float* pred, float* loss, void* saved, void* ws, size_t ws_bytes,
                    void* stream) {
  ORBIT_TRY(check_head(d));
  if (!z || !lnf_g || !lnf_b || !Wh || !bh || !target || !loss || !saved || !ws) { set_error("head_loss: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!aligned16(z) || !aligned16(lnf_g) || !aligned16(lnf_b) || !aligned16(Wh) || !aligned16(bh) || !aligned16(target) ||
      !aligned16(saved) || !aligned16(ws) || (pred && !aligned16(pred))) { set_error("head_loss: pointer not 16B aligned"); return ORBIT_ERR_ALIGN; }
  if (ws_bytes < orbit_head_loss_workspace_bytes(d)) { set_error("head_loss: workspace too small"); return ORBIT_ERR_WORKSPACE; }
  ORBIT_TRY(check_device());
  cudaStream_t s = (cudaStream_t)stream;
  const HeadDims h = head_dims(*d);
  const int D = d->D, dt = d->dtype, rt = d->resid_dtype;
  HeadSaved sv = carve_head_saved(*d, saved);
  HeadFwdWs w = carve_head_fwd(*d, ws);
  ORBIT_TRY(layernorm_fwd(z, rt, lnf_g, lnf_b, dt, sv.zn, dt, sv.mean, sv.rstd, h.BL, D, d->ln_eps, nullptr, s));
  {  // P = zn Wh + bh (fp32: the loss and its gradient are formed from the unrounded prediction)
    GemmArgs g;
    g.A = sv.zn; g.a_rs = D; g.a_cs = 1; g.B = Wh; g.b_rs = h.C; g.b_cs = 1; g.C = w.P; g.ldc = h.C;
    g.M = h.BL; g.N = h.C; g.K = D; g.in_dtype = dt; g.out_dtype = ORBIT_F32; g.bias = bh; g.bias_dtype = dt;
    ORBIT_TRY(gemm(g, s));
  }
  const float* wl = latw;
  if (!wl) {
    latw_kernel<<<1, 256, 0, s>>>(w.latw, d->Hg);
    ORBIT_LAUNCH_CHECK();
    wl = w.latw;
  }
  ORBIT_CUDA_CHECK(cudaMemsetAsync(loss, 0, sizeof(float), s));
  const size_t n = (size_t)h.BL * h.C;
  int grid = (int)((n + 255) / 256 < 148 * 8 ? (n + 255) / 256 : 148 * 8);
  if (dt == ORBIT_BF16) wmse_kernel<bf16><<<grid, 256, 0, s>>>(w.P, target, wl, pred, (bf16*)sv.dP, loss, d->B, d->V, d->Hg, d->Wg, d->p);
  else wmse_kernel<float><<<grid, 256, 0, s>>>(w.P, target, wl, pred, (float*)sv.dP, loss, d->B, d->V, d->Hg, d->Wg, d->p);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int orbit_head_loss_bwd(const orbit_head_desc* d, const void* z, const void* lnf_g, const void* Wh, const void* saved, void* dz,
                        void* dlnf_g, void* dlnf_b, void* dWh, void* dbh, void* ws, size_t ws_bytes, void* stream) {
  ORBIT_TRY(check_head(d));
  if (!z || !lnf_g || !Wh || !saved || !dz || !dlnf_g || !dlnf_b || !dWh || !dbh || !ws) { set_error("head_loss_bwd: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!aligned16(z) || !aligned16(lnf_g) || !aligned16(Wh) || !aligned16(saved) || !aligned16(dz) || !aligned16(dlnf_g) ||
      !aligned16(dlnf_b) || !aligned16(dWh) || !aligned16(dbh) || !aligned16(ws)) { set_error("head_loss_bwd: pointer not 16B aligned"); return ORBIT_ERR_ALIGN; }
  if (ws_bytes < orbit_head_loss_bwd_workspace_bytes(d)) { set_error("head_loss_bwd: workspace too small"); return ORBIT_ERR_WORKSPACE; }
  ORBIT_TRY(check_device());
  cudaStream_t s = (cudaStream_t)stream;
  const HeadDims h = head_dims(*d);
  const int D = d->D, dt = d->dtype, rt = d->resid_dtype;
  HeadSaved sv = carve_head_saved(*d, const_cast<void*>(saved));
  HeadBwdWs w = carve_head_bwd(*d, ws);
  float* acc_bh = w.acc;
  float* acc_g = acc_bh + h.C;
  float* acc_b = acc_g + D;
  ORBIT_TRY(fill_zero(w.acc, w.acc_floats * sizeof(float), s));
  ORBIT_TRY(colsum(sv.dP, dt, h.C, h.BL, h.C, acc_bh, nullptr, dt, h.C, s));        // dbh = sum dP
  {  // dWh = zn^T dP
    GemmArgs g;
    g.A = sv.zn; g.a_rs = 1; g.a_cs = D; g.B = sv.dP; g.b_rs = h.C; g.b_cs = 1; g.C = dWh; g.ldc = h.C;
    g.M = D; g.N = h.C; g.K = h.BL; g.in_dtype = dt; g.out_dtype = dt;
    ORBIT_TRY(gemm(g, s));
  }
  {  // dzn = dP Wh^T
    GemmArgs g;
    g.A = sv.dP; g.a_rs = h.C; g.a_cs = 1; g.B = Wh; g.b_rs = 1; g.b_cs = h.C; g.C = w.dzn; g.ldc = D;
    g.M = h.BL; g.N = D; g.K = h.C; g.in_dtype = dt; g.out_dtype = ORBIT_F32;
    ORBIT_TRY(gemm(g, s));
  }
  ORBIT_TRY(layernorm_bwd(w.dzn, ORBIT_F32, z, rt, sv.mean, sv.rstd, lnf_g, dt, nullptr, rt, nullptr, dz, rt, acc_g, acc_b,
                          h.BL, D, s));
  CastSegs cs;
  cs.add(acc_bh, dbh, h.C); cs.add(acc_g, dlnf_g, D); cs.add(acc_b, dlnf_b, D);
  ORBIT_TRY(cast_multi(cs, dt, s));
  return ORBIT_OK;
}

}  // extern "C"
