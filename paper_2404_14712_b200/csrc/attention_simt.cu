// attention_simt.cu -- fp32-FMA softmax attention forward/backward (PAPER.md:88 softmax(QK^T)V, :114 scaled
// dot product; reading R8), flash-style: no N x N matrix is ever stored, only logsumexp per row.
// One warp per query row (fwd, dQ) or per key row (dK/dV); the 32 lanes sweep the other index in tiles of 32.
// This is the ORBIT_F32 path and the small-shape / debug path of ORBIT_BF16; the large bf16 shapes use
// attention_tc.cu.
#include "common.cuh"

namespace orbit {
namespace {

constexpr int WPB = 8;          // warps (rows) per block
constexpr int MAXI = 8;         // dh <= 256

struct Smem {
  float* a;   // tile A [32][dh+1]
  float* b;   // tile B [32][dh+1]
  float* r0;  // per-warp row 0 [WPB][dh]
  float* r1;  // per-warp row 1 [WPB][dh]
  float* t0;  // [32]
  float* t1;  // [32]
};
__device__ __forceinline__ Smem carve(float* base, int dh) {
  Smem s;
  s.a = base;
  s.b = s.a + 32 * (dh + 1);
  s.r0 = s.b + 32 * (dh + 1);
  s.r1 = s.r0 + WPB * dh;
  s.t0 = s.r1 + WPB * dh;
  s.t1 = s.t0 + 32;
  return s;
}
size_t smem_bytes(int dh) { return sizeof(float) * (2 * 32 * (dh + 1) + 2 * WPB * dh + 64); }

// load a 32 x dh tile (rows row0.., column offset col) of a [rows, ld] matrix into sm[32][dh+1]; zero past N
__device__ __forceinline__ void load_tile(float* sm, const void* src, int dt, long long ld, size_t base_row,
                                          int row0, int N, int col, int dh) {
  for (int idx = threadIdx.x; idx < 32 * dh; idx += blockDim.x) {
    int r = idx / dh, d = idx - r * dh;
    float v = 0.f;
    if (row0 + r < N) v = ldf(src, (base_row + row0 + r) * ld + col + d, dt);
    sm[r * (dh + 1) + d] = v;
  }
}

__global__ void __launch_bounds__(WPB * 32) attn_fwd_kernel(AttnArgs a, float scale) {
  extern __shared__ float smem[];
  Smem s = carve(smem, a.dh);
  const int dh = a.dh, N = a.N;
  const int bh = blockIdx.y, b = bh / a.heads, h = bh - b * a.heads;
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int qi = blockIdx.x * WPB + w;
  const size_t brow = (size_t)b * N;
  const bool active = qi < N;
  float* qs = s.r0 + w * dh;
  for (int d = lane; d < dh; d += 32) qs[d] = active ? ldf(a.qkv, (brow + qi) * a.ld + a.q_off + h * dh + d, a.dtype) : 0.f;
  float m = -INFINITY, l = 0.f, acc[MAXI];
#pragma unroll
  for (int i = 0; i < MAXI; i++) acc[i] = 0.f;
  for (int k0 = 0; k0 < N; k0 += 32) {
    __syncthreads();
    load_tile(s.a, a.qkv, a.dtype, a.ld, brow, k0, N, a.k_off + h * dh, dh);
    load_tile(s.b, a.qkv, a.dtype, a.ld, brow, k0, N, a.v_off + h * dh, dh);
    __syncthreads();
    float sc = 0.f;
    const float* kr = s.a + lane * (dh + 1);
    for (int d = 0; d < dh; d++) sc = fmaf(qs[d], kr[d], sc);
    sc = (k0 + lane < N) ? sc * scale : -INFINITY;
    float mn = fmaxf(m, warp_max(sc));
    float p = __expf(sc - mn);
    float corr = __expf(m - mn);
    l = l * corr + warp_sum(p);
    m = mn;
#pragma unroll
    for (int i = 0; i < MAXI; i++) acc[i] *= corr;
    for (int jj = 0; jj < 32; jj++) {
      float pj = __shfl_sync(0xffffffffu, p, jj);
      const float* vr = s.b + jj * (dh + 1);
#pragma unroll
      for (int i = 0; i < MAXI; i++) {
        int d = lane + 32 * i;
        if (d < dh) acc[i] = fmaf(pj, vr[d], acc[i]);
      }
    }
  }
  if (active) {
    float inv = 1.f / l;
#pragma unroll
    for (int i = 0; i < MAXI; i++) {
      int d = lane + 32 * i;
      if (d < dh) stf(a.O, (brow + qi) * a.ldo + h * dh + d, acc[i] * inv, a.dtype);
    }
    if (lane == 0) a.lse[(size_t)bh * N + qi] = m + __logf(l);
  }
}

// delta[b,h,i] = sum_d dO[i, h*dh+d] * O[i, h*dh+d]   (= rowsum(dP o P))
__global__ void attn_delta_kernel(AttnArgs a) {
  const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  const int total = a.B * a.heads * a.N;
  if (w >= total) return;
  const int bh = w / a.N, i = w - bh * a.N, b = bh / a.heads, h = bh - b * a.heads;
  const size_t row = (size_t)b * a.N + i;
  float s = 0.f;
  for (int d = lane; d < a.dh; d += 32)
    s += ldf(a.dO, row * a.lddo + h * a.dh + d, a.dtype) * ldf(a.O, row * a.ldo + h * a.dh + d, a.dtype);
  s = warp_sum(s);
  if (lane == 0) a.delta[w] = s;
}

__global__ void __launch_bounds__(WPB * 32) attn_bwd_dq_kernel(AttnArgs a, float scale) {
  extern __shared__ float smem[];
  Smem s = carve(smem, a.dh);
  const int dh = a.dh, N = a.N;
  const int bh = blockIdx.y, b = bh / a.heads, h = bh - b * a.heads;
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int qi = blockIdx.x * WPB + w;
  const size_t brow = (size_t)b * N;
  const bool active = qi < N;
  float* qs = s.r0 + w * dh;
  float* dos = s.r1 + w * dh;
  for (int d = lane; d < dh; d += 32) {
    qs[d] = active ? ldf(a.qkv, (brow + qi) * a.ld + a.q_off + h * dh + d, a.dtype) : 0.f;
    dos[d] = active ? ldf(a.dO, (brow + qi) * a.lddo + h * dh + d, a.dtype) : 0.f;
  }
  const float lse = active ? a.lse[(size_t)bh * N + qi] : 0.f;
  const float dl = active ? a.delta[(size_t)bh * N + qi] : 0.f;
  float acc[MAXI];
#pragma unroll
  for (int i = 0; i < MAXI; i++) acc[i] = 0.f;
  for (int k0 = 0; k0 < N; k0 += 32) {
    __syncthreads();
    load_tile(s.a, a.qkv, a.dtype, a.ld, brow, k0, N, a.k_off + h * dh, dh);
    load_tile(s.b, a.qkv, a.dtype, a.ld, brow, k0, N, a.v_off + h * dh, dh);
    __syncthreads();
    float sc = 0.f, dp = 0.f;
    const float* kr = s.a + lane * (dh + 1);
    const float* vr = s.b + lane * (dh + 1);
    for (int d = 0; d < dh; d++) { sc = fmaf(qs[d], kr[d], sc); dp = fmaf(dos[d], vr[d], dp); }
    float p = (k0 + lane < N) ? __expf(sc * scale - lse) : 0.f;
    float ds = p * (dp - dl) * scale;
    for (int jj = 0; jj < 32; jj++) {
      float dsj = __shfl_sync(0xffffffffu, ds, jj);
      const float* krj = s.a + jj * (dh + 1);
#pragma unroll
      for (int i = 0; i < MAXI; i++) {
        int d = lane + 32 * i;
        if (d < dh) acc[i] = fmaf(dsj, krj[d], acc[i]);
      }
    }
  }
  if (active) {
#pragma unroll
    for (int i = 0; i < MAXI; i++) {
      int d = lane + 32 * i;
      if (d < dh) stf(a.dqkv, (brow + qi) * a.ld + a.q_off + h * dh + d, acc[i], a.dtype);
    }
  }
}

__global__ void __launch_bounds__(WPB * 32) attn_bwd_dkv_kernel(AttnArgs a, float scale) {
  extern __shared__ float smem[];
  Smem s = carve(smem, a.dh);
  const int dh = a.dh, N = a.N;
  const int bh = blockIdx.y, b = bh / a.heads, h = bh - b * a.heads;
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int kj = blockIdx.x * WPB + w;
  const size_t brow = (size_t)b * N;
  const bool active = kj < N;
  float* ks = s.r0 + w * dh;
  float* vs = s.r1 + w * dh;
  for (int d = lane; d < dh; d += 32) {
    ks[d] = active ? ldf(a.qkv, (brow + kj) * a.ld + a.k_off + h * dh + d, a.dtype) : 0.f;
    vs[d] = active ? ldf(a.qkv, (brow + kj) * a.ld + a.v_off + h * dh + d, a.dtype) : 0.f;
  }
  float dk[MAXI], dv[MAXI];
#pragma unroll
  for (int i = 0; i < MAXI; i++) { dk[i] = 0.f; dv[i] = 0.f; }
  for (int q0 = 0; q0 < N; q0 += 32) {
    __syncthreads();
    load_tile(s.a, a.qkv, a.dtype, a.ld, brow, q0, N, a.q_off + h * dh, dh);
    load_tile(s.b, a.dO, a.dtype, a.lddo, brow, q0, N, h * dh, dh);
    if (threadIdx.x < 32) {
      int qi = q0 + threadIdx.x;
      s.t0[threadIdx.x] = qi < N ? a.lse[(size_t)bh * N + qi] : 0.f;
      s.t1[threadIdx.x] = qi < N ? a.delta[(size_t)bh * N + qi] : 0.f;
    }
    __syncthreads();
    float sc = 0.f, dp = 0.f;
    const float* qr = s.a + lane * (dh + 1);
    const float* dor = s.b + lane * (dh + 1);
    for (int d = 0; d < dh; d++) { sc = fmaf(qr[d], ks[d], sc); dp = fmaf(dor[d], vs[d], dp); }
    float p = (q0 + lane < N) ? __expf(sc * scale - s.t0[lane]) : 0.f;
    float ds = p * (dp - s.t1[lane]) * scale;
    for (int ii = 0; ii < 32; ii++) {
      float pi = __shfl_sync(0xffffffffu, p, ii);
      float dsi = __shfl_sync(0xffffffffu, ds, ii);
      const float* qri = s.a + ii * (dh + 1);
      const float* dori = s.b + ii * (dh + 1);
#pragma unroll
      for (int i = 0; i < MAXI; i++) {
        int d = lane + 32 * i;
        if (d < dh) { dv[i] = fmaf(pi, dori[d], dv[i]); dk[i] = fmaf(dsi, qri[d], dk[i]); }
      }
    }
  }
  if (active) {
#pragma unroll
    for (int i = 0; i < MAXI; i++) {
      int d = lane + 32 * i;
      if (d < dh) {
        stf(a.dqkv, (brow + kj) * a.ld + a.k_off + h * dh + d, dk[i], a.dtype);
        stf(a.dqkv, (brow + kj) * a.ld + a.v_off + h * dh + d, dv[i], a.dtype);
      }
    }
  }
}

int set_smem(const void* fn, size_t bytes) {
  if (bytes > 48 * 1024) ORBIT_CUDA_CHECK(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
  return ORBIT_OK;
}
}  // namespace

int attention_fwd_simt(const AttnArgs& a, cudaStream_t st) {
  if (a.dh > 32 * MAXI) { set_error("attention: d_h=%d > %d unsupported", a.dh, 32 * MAXI); return ORBIT_ERR_SHAPE; }
  size_t sb = smem_bytes(a.dh);
  ORBIT_TRY(set_smem((const void*)attn_fwd_kernel, sb));
  dim3 grid(cdiv(a.N, WPB), a.B * a.heads);
  attn_fwd_kernel<<<grid, WPB * 32, sb, st>>>(a, 1.0f / sqrtf((float)a.dh));
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int attention_bwd_simt(const AttnArgs& a, cudaStream_t st) {
  if (a.dh > 32 * MAXI) { set_error("attention: d_h=%d > %d unsupported", a.dh, 32 * MAXI); return ORBIT_ERR_SHAPE; }
  size_t sb = smem_bytes(a.dh);
  ORBIT_TRY(set_smem((const void*)attn_bwd_dq_kernel, sb));
  ORBIT_TRY(set_smem((const void*)attn_bwd_dkv_kernel, sb));
  int total_w = a.B * a.heads * a.N;
  attn_delta_kernel<<<cdiv((long long)total_w * 32, 256), 256, 0, st>>>(a);
  ORBIT_LAUNCH_CHECK();
  dim3 grid(cdiv(a.N, WPB), a.B * a.heads);
  float scale = 1.0f / sqrtf((float)a.dh);
  attn_bwd_dq_kernel<<<grid, WPB * 32, sb, st>>>(a, scale);
  ORBIT_LAUNCH_CHECK();
  attn_bwd_dkv_kernel<<<grid, WPB * 32, sb, st>>>(a, scale);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

}  // namespace orbit
