// aggregate.cu -- a2 / a2': per-patch kernels of the variable-aggregation cross-attention (PAPER.md:46
// "aggregated together across different channels using cross-attention"; readings R3, R4).
//
// Collapsed form (exact in real arithmetic): with qt = q Wq + bq and
//   Ut[d,a] = sum_{c in head a} Wk[d,c] qt[c] / sqrt(d_a)
// the logits are s[v,a] = X_v . Ut[:,a] + const_a (bk and the constant cancel in the softmax over v) and,
// because sum_v alpha_v = 1,  o_a = (sum_v alpha[v,a] X_v) Wv[:, a] + bv[a] = Xbar[a,:] Wv[:,a] + bv[a].
// So the V x (K,V projection) GEMMs disappear: one pass over tok per direction plus [B*L]-row GEMMs.
#include "frontend.cuh"

namespace orbit {
namespace {

__device__ __forceinline__ void ld2(const void* p, size_t i, int dt, float& a, float& b) {
  if (dt == ORBIT_BF16) {
    float2 f = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>((const bf16*)p + i));
    a = f.x; b = f.y;
  } else {
    float2 f = *reinterpret_cast<const float2*>((const float*)p + i);
    a = f.x; b = f.y;
  }
}
__device__ __forceinline__ void st2(void* p, size_t i, int dt, float a, float b) {
  if (dt == ORBIT_BF16) *reinterpret_cast<__nv_bfloat162*>((bf16*)p + i) = __floats2bfloat162_rn(a, b);
  else *reinterpret_cast<float2*>((float*)p + i) = make_float2(a, b);
}

__global__ void agg_make_u_kernel(const void* __restrict__ Wk, int p_dt, const float* __restrict__ qt,
                                  float* __restrict__ Ut, int D, int heads) {
  const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (w >= D * heads) return;
  const int d = w / heads, a = w - d * heads, da = D / heads;
  float s = 0.f;
  for (int c = lane; c < da; c += 32) s += ldf(Wk, (size_t)d * D + a * da + c, p_dt) * qt[a * da + c];
  s = warp_sum(s);
  if (lane == 0) Ut[(size_t)d * heads + a] = s * rsqrtf((float)da);
}

// ---- forward: scores, softmax over V, weighted token mean per head -----------------------------------
template <int MAXH>
__global__ void __launch_bounds__(256) agg_patch_fwd_kernel(const void* __restrict__ tok, int dt,
    const float* __restrict__ Ut, float* __restrict__ alpha, void* __restrict__ Xbar, int BL, int V, int D, int h) {
  extern __shared__ float sm[];
  float* s_al = sm;                       // [V][h]
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
  for (int bl = blockIdx.x; bl < BL; bl += gridDim.x) {
    const size_t xbase = (size_t)bl * V * D;
    // phase 1: s[v,a] = X_v . Ut[:,a]
    for (int v = w; v < V; v += nw) {
      float acc[MAXH];
#pragma unroll
      for (int a = 0; a < MAXH; a++) acc[a] = 0.f;
      for (int d = lane * 2; d < D; d += 64) {
        float x0, x1;
        ld2(tok, xbase + (size_t)v * D + d, dt, x0, x1);
        const float* u0 = Ut + (size_t)d * h;
#pragma unroll
        for (int a = 0; a < MAXH; a++)
          if (a < h) acc[a] = fmaf(x0, u0[a], fmaf(x1, u0[h + a], acc[a]));
      }
#pragma unroll
      for (int a = 0; a < MAXH; a++)
        if (a < h) {
          float t = warp_sum(acc[a]);
          if (lane == 0) s_al[v * h + a] = t;
        }
    }
    __syncthreads();
    // phase 2: softmax over v for each head (warp-level: lanes stride over v)
    for (int a = w; a < h; a += nw) {
      float m = -INFINITY;
      for (int v = lane; v < V; v += 32) m = fmaxf(m, s_al[v * h + a]);
      m = warp_max(m);
      float l = 0.f;
      for (int v = lane; v < V; v += 32) l += __expf(s_al[v * h + a] - m);
      l = warp_sum(l);
      float inv = 1.f / l;
      for (int v = lane; v < V; v += 32) {
        float p = __expf(s_al[v * h + a] - m) * inv;
        s_al[v * h + a] = p;
        alpha[((size_t)bl * h + a) * V + v] = p;
      }
    }
    __syncthreads();
    // phase 3: Xbar[a,:] = sum_v alpha[v,a] X_v
    for (int d = threadIdx.x * 2; d < D; d += blockDim.x * 2) {
      float a0[MAXH], a1[MAXH];
#pragma unroll
      for (int a = 0; a < MAXH; a++) { a0[a] = 0.f; a1[a] = 0.f; }
      for (int v = 0; v < V; v++) {
        float x0, x1;
        ld2(tok, xbase + (size_t)v * D + d, dt, x0, x1);
        const float* al = s_al + v * h;
#pragma unroll
        for (int a = 0; a < MAXH; a++)
          if (a < h) { a0[a] = fmaf(al[a], x0, a0[a]); a1[a] = fmaf(al[a], x1, a1[a]); }
      }
#pragma unroll
      for (int a = 0; a < MAXH; a++)
        if (a < h) st2(Xbar, ((size_t)bl * h + a) * D + d, dt, a0[a], a1[a]);
    }
    __syncthreads();
  }
}

// ---- backward ---------------------------------------------------------------------------------------
template <int MAXH>
__global__ void __launch_bounds__(256) agg_patch_bwd_kernel(const void* __restrict__ tok, int dt,
    const float* __restrict__ Ut, const float* __restrict__ alpha, const void* __restrict__ dXbar,
    void* __restrict__ dtok, float* __restrict__ dUt_acc, int BL, int V, int D, int h) {
  extern __shared__ float sm[];
  float* s_al = sm;                       // [V][h]
  float* s_ds = s_al + V * h;             // [V][h]
  float* s_accU = s_ds + V * h;           // [h][D]  block-private accumulator of dUt^T
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
  for (int i = threadIdx.x; i < h * D; i += blockDim.x) s_accU[i] = 0.f;
  __syncthreads();
  for (int bl = blockIdx.x; bl < BL; bl += gridDim.x) {
    const size_t xbase = (size_t)bl * V * D;
    for (int i = threadIdx.x; i < V * h; i += blockDim.x) {
      int v = i / h, a = i - v * h;
      s_al[i] = alpha[((size_t)bl * h + a) * V + v];
    }
    // phase 1: dalpha[v,a] = X_v . dXbar[a,:]
    for (int v = w; v < V; v += nw) {
      float acc[MAXH];
#pragma unroll
      for (int a = 0; a < MAXH; a++) acc[a] = 0.f;
      for (int d = lane * 2; d < D; d += 64) {
        float x0, x1;
        ld2(tok, xbase + (size_t)v * D + d, dt, x0, x1);
#pragma unroll
        for (int a = 0; a < MAXH; a++)
          if (a < h) {
            float g0, g1;
            ld2(dXbar, ((size_t)bl * h + a) * D + d, dt, g0, g1);
            acc[a] = fmaf(x0, g0, fmaf(x1, g1, acc[a]));
          }
      }
#pragma unroll
      for (int a = 0; a < MAXH; a++)
        if (a < h) {
          float t = warp_sum(acc[a]);
          if (lane == 0) s_ds[v * h + a] = t;
        }
    }
    __syncthreads();
    // phase 2: ds[v,a] = alpha (dalpha - sum_w alpha_w dalpha_w)
    for (int a = w; a < h; a += nw) {
      float dot = 0.f;
      for (int v = lane; v < V; v += 32) dot += s_al[v * h + a] * s_ds[v * h + a];
      dot = warp_sum(dot);
      for (int v = lane; v < V; v += 32) s_ds[v * h + a] = s_al[v * h + a] * (s_ds[v * h + a] - dot);
    }
    __syncthreads();
    // phase 3: dX[v,:] = sum_a alpha[v,a] dXbar[a,:] + ds[v,a] Ut[:,a]^T ;  dUt^T[a,:] += sum_v ds[v,a] X_v
    for (int d = threadIdx.x * 2; d < D; d += blockDim.x * 2) {
      float g0[MAXH], g1[MAXH], u0[MAXH], u1[MAXH], c0[MAXH], c1[MAXH];
#pragma unroll
      for (int a = 0; a < MAXH; a++) {
        g0[a] = g1[a] = u0[a] = u1[a] = c0[a] = c1[a] = 0.f;
        if (a < h) {
          ld2(dXbar, ((size_t)bl * h + a) * D + d, dt, g0[a], g1[a]);
          u0[a] = Ut[(size_t)d * h + a];
          u1[a] = Ut[(size_t)(d + 1) * h + a];
        }
      }
      for (int v = 0; v < V; v++) {
        float x0, x1, o0 = 0.f, o1 = 0.f;
        ld2(tok, xbase + (size_t)v * D + d, dt, x0, x1);
        const float* al = s_al + v * h;
        const float* ds = s_ds + v * h;
#pragma unroll
        for (int a = 0; a < MAXH; a++)
          if (a < h) {
            float av = al[a], dv = ds[a];
            o0 = fmaf(av, g0[a], fmaf(dv, u0[a], o0));
            o1 = fmaf(av, g1[a], fmaf(dv, u1[a], o1));
            c0[a] = fmaf(dv, x0, c0[a]);
            c1[a] = fmaf(dv, x1, c1[a]);
          }
        st2(dtok, xbase + (size_t)v * D + d, dt, o0, o1);
      }
#pragma unroll
      for (int a = 0; a < MAXH; a++)
        if (a < h) { s_accU[a * D + d] += c0[a]; s_accU[a * D + d + 1] += c1[a]; }
    }
    __syncthreads();
  }
  for (int i = threadIdx.x; i < h * D; i += blockDim.x) {
    int a = i / D, d = i - a * D;
    atomicAdd(dUt_acc + (size_t)d * h + a, s_accU[i]);
  }
}

// dqt[c] = sum_d dUt[d,a(c)] Wk[d,c] / sqrt(d_a): 32 columns x 8 row-lanes per block, rows strided over lanes
__global__ void __launch_bounds__(256) agg_dqt_kernel(const float* __restrict__ dUt, const void* __restrict__ Wk, int p_dt,
                                                      float* __restrict__ dqt, int D, int h) {
  __shared__ float sh[8][33];
  const int cx = threadIdx.x & 31, ry = threadIdx.x >> 5;
  const int c = blockIdx.x * 32 + cx;
  const int da = D / h, a = c < D ? c / da : 0;
  float s = 0.f;
  if (c < D) {
    int d = ry;
    if (p_dt == ORBIT_BF16) {               // eight rows requested before the first FMA (one 2-byte load per thread in flight: 42 us at D = 2048)
      const bf16* W = (const bf16*)Wk + c;
      for (; d + 56 < D; d += 64) {
        float w[8], u[8];
#pragma unroll
        for (int i = 0; i < 8; i++) { w[i] = __bfloat162float(W[(size_t)(d + 8 * i) * D]); u[i] = dUt[(size_t)(d + 8 * i) * h + a]; }
#pragma unroll
        for (int i = 0; i < 8; i++) s = fmaf(u[i], w[i], s);
      }
    }
    for (; d < D; d += 8) s = fmaf(dUt[(size_t)d * h + a], ldf(Wk, (size_t)d * D + c, p_dt), s);
  }
  sh[ry][cx] = s;
  __syncthreads();
  if (ry == 0 && c < D) {
    float t = 0.f;
#pragma unroll
    for (int y = 0; y < 8; y++) t += sh[y][cx];
    dqt[c] = t * rsqrtf((float)da);
  }
}
// qt[n] = sum_k q[k] Wq[k,n] + bq[n]   (one learned query, R4: a GEMV, same column-strided scheme)
__global__ void __launch_bounds__(256) agg_qt_kernel(const void* __restrict__ q, const void* __restrict__ Wq,
                                                     const void* __restrict__ bq, int p_dt, float* __restrict__ qt, int D) {
  __shared__ float sh[8][33];
  const int cx = threadIdx.x & 31, ry = threadIdx.x >> 5;
  const int n = blockIdx.x * 32 + cx;
  float s = 0.f;
  if (n < D) {
    int k = ry;
    if (p_dt == ORBIT_BF16) {               // as in agg_dqt_kernel: eight loads in flight per thread (48 -> ~10 us at D = 2048)
      const bf16* W = (const bf16*)Wq + n;
      const bf16* qv = (const bf16*)q;
      for (; k + 56 < D; k += 64) {
        float w[8], u[8];
#pragma unroll
        for (int i = 0; i < 8; i++) { w[i] = __bfloat162float(W[(size_t)(k + 8 * i) * D]); u[i] = __bfloat162float(qv[k + 8 * i]); }
#pragma unroll
        for (int i = 0; i < 8; i++) s = fmaf(u[i], w[i], s);
      }
    }
    for (; k < D; k += 8) s = fmaf(ldf(q, k, p_dt), ldf(Wq, (size_t)k * D + n, p_dt), s);
  }
  sh[ry][cx] = s;
  __syncthreads();
  if (ry == 0 && n < D) {
    float t = 0.f;
#pragma unroll
    for (int y = 0; y < 8; y++) t += sh[y][cx];
    qt[n] = t + ldf(bq, n, p_dt);
  }
}
// dWk[d,c] = dUt[d,a(c)] qt[c]/sqrt(d_a); dWq[i,c] = q[i] dqt[c]; dbk = 0; dbq = dqt
__global__ void agg_outer_kernel(const float* __restrict__ dUt, const float* __restrict__ qt,
    const float* __restrict__ dqt, const void* __restrict__ q, int p_dt, void* __restrict__ dWk,
    void* __restrict__ dWq, void* __restrict__ dbk, void* __restrict__ dbq, int D, int h) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (size_t)D * D) return;
  int r = (int)(i / D), c = (int)(i - (size_t)r * D), da = D / h, a = c / da;
  stf(dWk, i, dUt[(size_t)r * h + a] * qt[c] * rsqrtf((float)da), p_dt);
  stf(dWq, i, ldf(q, r, p_dt) * dqt[c], p_dt);
  if (r == 0) { stf(dbk, c, 0.f, p_dt); stf(dbq, c, dqt[c], p_dt); }
}
// dq[i] = sum_c dqt[c] Wq[i,c]
__global__ void agg_dq_kernel(const float* __restrict__ dqt, const void* __restrict__ Wq, int p_dt,
                              void* __restrict__ dq, int D) {
  const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (w >= D) return;
  float s = 0.f;
  for (int c = lane; c < D; c += 32) s = fmaf(dqt[c], ldf(Wq, (size_t)w * D + c, p_dt), s);
  s = warp_sum(s);
  if (lane == 0) stf(dq, w, s, p_dt);
}
__global__ void agg_dpos_kernel(const void* __restrict__ dagg, int dt, void* __restrict__ dpos, int B, size_t LD) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= LD) return;
  float s = 0.f;
  for (int b = 0; b < B; b++) s += ldf(dagg, (size_t)b * LD + i, dt);
  stf(dpos, i, s, dt);
}
}  // namespace

int agg_make_qt(const void* q, const void* Wq, const void* bq, int p_dt, float* qt, int D, cudaStream_t s) {
  agg_qt_kernel<<<cdiv(D, 32), 256, 0, s>>>(q, Wq, bq, p_dt, qt, D);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int agg_make_u(const void* Wk, int p_dt, const float* qt, float* Ut, int D, int heads, cudaStream_t s) {
  long long threads = (long long)D * heads * 32;
  agg_make_u_kernel<<<cdiv(threads, 256), 256, 0, s>>>(Wk, p_dt, qt, Ut, D, heads);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int agg_patch_fwd(const void* tok, int dt, const float* Ut, float* alpha, void* Xbar, int BL, int V, int D,
                  int heads, cudaStream_t s) {
  size_t smb = (size_t)V * heads * sizeof(float);
  int grid = BL < 148 * 8 ? BL : 148 * 8;
#define AF(H) do { if (smb > 48 * 1024) ORBIT_CUDA_CHECK(cudaFuncSetAttribute((const void*)agg_patch_fwd_kernel<H>, \
      cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smb));                                                      \
    agg_patch_fwd_kernel<H><<<grid, 256, smb, s>>>(tok, dt, Ut, alpha, Xbar, BL, V, D, heads); } while (0)
  if (heads <= 4) AF(4);
  else if (heads <= 16) AF(16);
  else if (heads <= 32) AF(32);
  else { set_error("var_aggregate: heads=%d > 32 unsupported", heads); return ORBIT_ERR_SHAPE; }
#undef AF
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

size_t agg_patch_bwd_smem(int V, int D, int heads) {
  return ((size_t)2 * V * heads + (size_t)heads * D) * sizeof(float);
}

int agg_patch_bwd(const void* tok, int dt, const float* Ut, const float* alpha, const void* dXbar, void* dtok,
                  float* dUt_acc, int BL, int V, int D, int heads, cudaStream_t s) {
  size_t smb = agg_patch_bwd_smem(V, D, heads);
  if (smb > 220 * 1024) { set_error("var_aggregate_bwd: heads*D=%d too large for shared memory", heads * D); return ORBIT_ERR_SHAPE; }
  int per_sm = (int)((220 * 1024) / smb);
  if (per_sm < 1) per_sm = 1;
  if (per_sm > 4) per_sm = 4;
  int grid = BL < 148 * per_sm ? BL : 148 * per_sm;
#define AB(H) do { if (smb > 48 * 1024) ORBIT_CUDA_CHECK(cudaFuncSetAttribute((const void*)agg_patch_bwd_kernel<H>, \
      cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smb));                                                      \
    agg_patch_bwd_kernel<H><<<grid, 256, smb, s>>>(tok, dt, Ut, alpha, dXbar, dtok, dUt_acc, BL, V, D, heads); } while (0)
  if (heads <= 4) AB(4);
  else if (heads <= 16) AB(16);
  else if (heads <= 32) AB(32);
  else { set_error("var_aggregate_bwd: heads=%d > 32 unsupported", heads); return ORBIT_ERR_SHAPE; }
#undef AB
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int agg_param_bwd(const float* dUt, const float* qt, const void* q, const void* Wq, const void* Wk, int p_dt,
                  void* dWk, void* dbk, void* dbq, void* dWq, void* dq, float* dqt_ws, int D, int heads,
                  cudaStream_t s) {
  agg_dqt_kernel<<<cdiv(D, 32), 256, 0, s>>>(dUt, Wk, p_dt, dqt_ws, D, heads);
  ORBIT_LAUNCH_CHECK();
  agg_outer_kernel<<<cdiv((long long)D * D, 256), 256, 0, s>>>(dUt, qt, dqt_ws, q, p_dt, dWk, dWq, dbk, dbq, D, heads);
  ORBIT_LAUNCH_CHECK();
  agg_dq_kernel<<<cdiv((long long)D * 32, 256), 256, 0, s>>>(dqt_ws, Wq, p_dt, dq, D);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int agg_dpos(const void* dagg, int dt, void* dpos, int B, int L, int D, cudaStream_t s) {
  size_t LD = (size_t)L * D;
  agg_dpos_kernel<<<cdiv((long long)LD, 256), 256, 0, s>>>(dagg, dt, dpos, B, LD);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

}  // namespace orbit
