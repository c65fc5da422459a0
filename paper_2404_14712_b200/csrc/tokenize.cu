// tokenize.cu -- a1 / a1': per-variable patch tokenisation and its parameter gradients.
// PAPER.md:46 "independent patch tokenization for each channel input"; PAPER.md:155 (128x256xC_d samples).
// Output-write bound (tok is [B,L,V,D]); each thread owns 4 consecutive d, keeps Wp[v,:,d..d+3] in
// registers and streams PC patches whose pixels sit in shared memory.
#include "frontend.cuh"

namespace orbit {
namespace {

__device__ __forceinline__ void ld4(const void* p, size_t i, int dt, float* v) {
  if (dt == ORBIT_BF16) {
    uint2 raw = *reinterpret_cast<const uint2*>((const bf16*)p + i);
    const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&raw);
    float2 a = __bfloat1622float2(h[0]), b = __bfloat1622float2(h[1]);
    v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
  } else {
    float4 a = *reinterpret_cast<const float4*>((const float*)p + i);
    v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w;
  }
}
__device__ __forceinline__ void st4(void* p, size_t i, int dt, const float* v) {
  if (dt == ORBIT_BF16) {
    uint2 raw;
    __nv_bfloat162* h = reinterpret_cast<__nv_bfloat162*>(&raw);
    h[0] = __floats2bfloat162_rn(v[0], v[1]);
    h[1] = __floats2bfloat162_rn(v[2], v[3]);
    *reinterpret_cast<uint2*>((bf16*)p + i) = raw;
  } else {
    *reinterpret_cast<float4*>((float*)p + i) = make_float4(v[0], v[1], v[2], v[3]);
  }
}

// pixels of patches [l0, l0+npatch) of (b, v) -> sm[patch][P2]
__device__ __forceinline__ void load_pixels(float* sm, const float* x, int b, int v, int V, int Hg, int Wg, int p,
                                            int l0, int npatch) {
  const int gw = Wg / p, P2 = p * p;
  const float* xv = x + ((size_t)b * V + v) * Hg * Wg;
  for (int idx = threadIdx.x; idx < npatch * P2; idx += blockDim.x) {
    int lp = idx / P2, r = idx - lp * P2;
    int l = l0 + lp, i = l / gw, j = l - i * gw, di = r / p, dj = r - di * p;
    sm[idx] = xv[(size_t)(i * p + di) * Wg + j * p + dj];
  }
}

template <int P2>
__global__ void __launch_bounds__(512) tok_fwd_kernel(orbit_embed_desc d, const float* __restrict__ x,
    const void* __restrict__ Wp, const void* __restrict__ bp, void* __restrict__ tok, int L, int PC) {
  extern __shared__ float spix[];
  const int v = blockIdx.y, b = blockIdx.z;
  const int l0 = blockIdx.x * PC, np = min(PC, L - l0);
  load_pixels(spix, x, b, v, d.V, d.Hg, d.Wg, d.p, l0, np);
  __syncthreads();
  for (int d0 = threadIdx.x * 4; d0 < d.D; d0 += blockDim.x * 4) {
    float w[P2][4], bias[4];
#pragma unroll
    for (int r = 0; r < P2; r++) ld4(Wp, ((size_t)v * P2 + r) * d.D + d0, d.dtype, w[r]);
    ld4(bp, (size_t)v * d.D + d0, d.dtype, bias);
    for (int lp = 0; lp < np; lp++) {
      float o[4] = {bias[0], bias[1], bias[2], bias[3]};
      const float* px = spix + lp * P2;
#pragma unroll
      for (int r = 0; r < P2; r++) {
        float pv = px[r];
#pragma unroll
        for (int j = 0; j < 4; j++) o[j] = fmaf(pv, w[r][j], o[j]);
      }
      st4(tok, (((size_t)b * L + l0 + lp) * d.V + v) * d.D + d0, d.dtype, o);
    }
  }
}

template <int P2>
__global__ void __launch_bounds__(512) tok_bwd_kernel(orbit_embed_desc d, const float* __restrict__ x,
    const void* __restrict__ dtok, float* __restrict__ accW, float* __restrict__ accB, int L, int PC) {
  extern __shared__ float spix[];
  const int v = blockIdx.y, b = blockIdx.z;
  const int l0 = blockIdx.x * PC, np = min(PC, L - l0);
  load_pixels(spix, x, b, v, d.V, d.Hg, d.Wg, d.p, l0, np);
  __syncthreads();
  for (int d0 = threadIdx.x * 4; d0 < d.D; d0 += blockDim.x * 4) {
    float aw[P2][4], ab[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int r = 0; r < P2; r++)
#pragma unroll
      for (int j = 0; j < 4; j++) aw[r][j] = 0.f;
    for (int lp = 0; lp < np; lp++) {
      float g[4];
      ld4(dtok, (((size_t)b * L + l0 + lp) * d.V + v) * d.D + d0, d.dtype, g);
      const float* px = spix + lp * P2;
#pragma unroll
      for (int j = 0; j < 4; j++) ab[j] += g[j];
#pragma unroll
      for (int r = 0; r < P2; r++) {
        float pv = px[r];
#pragma unroll
        for (int j = 0; j < 4; j++) aw[r][j] = fmaf(pv, g[j], aw[r][j]);
      }
    }
#pragma unroll
    for (int j = 0; j < 4; j++) atomicAdd(accB + (size_t)v * d.D + d0 + j, ab[j]);
#pragma unroll
    for (int r = 0; r < P2; r++)
#pragma unroll
      for (int j = 0; j < 4; j++) atomicAdd(accW + ((size_t)v * P2 + r) * d.D + d0 + j, aw[r][j]);
  }
}

int block_threads(int D) {
  int t = ((D / 4 + 31) / 32) * 32;
  return t > 512 ? 512 : (t < 32 ? 32 : t);
}
}  // namespace

int tokenize_fwd(const orbit_embed_desc& d, const float* x, const void* Wp, const void* bp, void* tok, cudaStream_t s) {
  const int L = (d.Hg / d.p) * (d.Wg / d.p), P2 = d.p * d.p;
  const int PC = 64;
  dim3 grid(cdiv(L, PC), d.V, d.B);
  int thr = block_threads(d.D);
  size_t sm = (size_t)PC * P2 * sizeof(float);
  switch (P2) {
    case 1: tok_fwd_kernel<1><<<grid, thr, sm, s>>>(d, x, Wp, bp, tok, L, PC); break;
    case 4: tok_fwd_kernel<4><<<grid, thr, sm, s>>>(d, x, Wp, bp, tok, L, PC); break;
    case 16: tok_fwd_kernel<16><<<grid, thr, sm, s>>>(d, x, Wp, bp, tok, L, PC); break;
    default: set_error("tokenize: patch size %d unsupported (1, 2, 4)", d.p); return ORBIT_ERR_SHAPE;
  }
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int tokenize_bwd_acc(const orbit_embed_desc& d, const float* x, const void* dtok, float* accW, float* accB,
                     cudaStream_t s) {
  const int L = (d.Hg / d.p) * (d.Wg / d.p), P2 = d.p * d.p;
  // enough patches per block to keep the fp32 atomics (D*(P2+1) per block) well below the dtok stream
  int PC = 1024;
  while (PC > 64 && (long long)cdiv(L, PC) * d.V * d.B < 148 * 2) PC >>= 1;
  dim3 grid(cdiv(L, PC), d.V, d.B);
  int thr = block_threads(d.D);
  size_t sm = (size_t)PC * P2 * sizeof(float);
  if (sm > 48 * 1024) {
    ORBIT_CUDA_CHECK(cudaFuncSetAttribute((const void*)tok_bwd_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
  }
  switch (P2) {
    case 1: tok_bwd_kernel<1><<<grid, thr, sm, s>>>(d, x, dtok, accW, accB, L, PC); break;
    case 4: tok_bwd_kernel<4><<<grid, thr, sm, s>>>(d, x, dtok, accW, accB, L, PC); break;
    case 16: tok_bwd_kernel<16><<<grid, thr, sm, s>>>(d, x, dtok, accW, accB, L, PC); break;
    default: set_error("tokenize_bwd: patch size %d unsupported (1, 2, 4)", d.p); return ORBIT_ERR_SHAPE;
  }
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

}  // namespace orbit
