// qknorm.cu -- QK-LayerNorm ("additional layer normalization to the queries ... and keys ... before
// computing the self-attention scaled dot product", after ref. [8]; reading R9): LayerNorm over the d_h
// entries of every head's query and key vector, gamma / beta in R^{d_h} shared by all heads.
//
// Layout: the block keeps a [M, 5*dc] buffer per shard, columns [Q | K | V | Q' | K'] (dc = D/T): the QKV GEMM writes
// the first 3*dc columns, qknorm_fwd writes Q', K' and attention reads (Q', K', V).  Backward: attention writes
// dQ', dK', dV into the same layout of dqkv; qknorm_bwd turns (dQ', dK') into (dQ, dK) in columns [0, 2*dc) and
// accumulates dgamma / dbeta (fp32, [4][d_h]: q-gamma, q-beta, k-gamma, k-beta).  Statistics are recomputed in the
// backward pass (one warp holds a whole head vector: d_h / 32 elements per lane), nothing extra is saved.
// HBM-bound row kernels: one warp per (token, head), fp32 statistics.
#include "common.cuh"

namespace orbit {
namespace {

template <typename T, int EPL>
__device__ __forceinline__ void ld_vec(const T* p, float* v) {
#pragma unroll
  for (int i = 0; i < EPL; i++) v[i] = to_f<T>(p[i]);
}
template <int EPL>
__device__ __forceinline__ void ld_vec_bf16(const bf16* p, float* v) {
  if (EPL % 2 == 0) {
#pragma unroll
    for (int i = 0; i < EPL / 2; i++) {
      const float2 f = __bfloat1622float2(reinterpret_cast<const __nv_bfloat162*>(p)[i]);
      v[2 * i] = f.x; v[2 * i + 1] = f.y;
    }
  } else {
    v[0] = __bfloat162float(p[0]);
  }
}
template <> __device__ __forceinline__ void ld_vec<bf16, 2>(const bf16* p, float* v) { ld_vec_bf16<2>(p, v); }
template <> __device__ __forceinline__ void ld_vec<bf16, 4>(const bf16* p, float* v) { ld_vec_bf16<4>(p, v); }
template <> __device__ __forceinline__ void ld_vec<bf16, 6>(const bf16* p, float* v) { ld_vec_bf16<6>(p, v); }
template <> __device__ __forceinline__ void ld_vec<bf16, 8>(const bf16* p, float* v) { ld_vec_bf16<8>(p, v); }

template <typename T, int EPL>
__device__ __forceinline__ void st_vec(T* p, const float* v) {
#pragma unroll
  for (int i = 0; i < EPL; i++) p[i] = from_f<T>(v[i]);
}
template <int EPL>
__device__ __forceinline__ void st_vec_bf16(bf16* p, const float* v) {
#pragma unroll
  for (int i = 0; i < EPL / 2; i++) reinterpret_cast<__nv_bfloat162*>(p)[i] = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]);
}
template <> __device__ __forceinline__ void st_vec<bf16, 2>(bf16* p, const float* v) { st_vec_bf16<2>(p, v); }
template <> __device__ __forceinline__ void st_vec<bf16, 4>(bf16* p, const float* v) { st_vec_bf16<4>(p, v); }
template <> __device__ __forceinline__ void st_vec<bf16, 6>(bf16* p, const float* v) { st_vec_bf16<6>(p, v); }
template <> __device__ __forceinline__ void st_vec<bf16, 8>(bf16* p, const float* v) { st_vec_bf16<8>(p, v); }

// mean / rstd of one head vector spread over the warp (EPL elements per lane)
template <int EPL>
__device__ __forceinline__ void warp_stats(const float* z, int dh, float eps, float& mu, float& rs) {
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < EPL; i++) s += z[i];
  mu = warp_sum(s) / dh;
  float q = 0.f;
#pragma unroll
  for (int i = 0; i < EPL; i++) { const float d = z[i] - mu; q += d * d; }
  rs = rsqrtf(warp_sum(q) / dh + eps);
}

template <typename T, int EPL>
__global__ void __launch_bounds__(256) qknorm_fwd_kernel(T* __restrict__ qkv, long long ld, long long items, int hk, int dh,
    int dc, const void* __restrict__ qg, const void* __restrict__ qb, const void* __restrict__ kg,
    const void* __restrict__ kb, int p_dt, float eps) {
  const int lane = threadIdx.x & 31;
  const long long w0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = ((long long)gridDim.x * blockDim.x) >> 5;
  float g[2][EPL], bt[2][EPL];
#pragma unroll
  for (int i = 0; i < EPL; i++) {
    g[0][i] = ldf(qg, lane * EPL + i, p_dt); bt[0][i] = ldf(qb, lane * EPL + i, p_dt);
    g[1][i] = ldf(kg, lane * EPL + i, p_dt); bt[1][i] = ldf(kb, lane * EPL + i, p_dt);
  }
  for (long long it = w0; it < items; it += nw) {
    const long long m = it / hk;
    const int j = (int)(it - m * hk);
    T* row = qkv + m * ld + (size_t)j * dh + lane * EPL;
#pragma unroll
    for (int which = 0; which < 2; which++) {           // 0: queries, 1: keys
      float z[EPL], o[EPL], mu, rs;
      ld_vec<T, EPL>(row + (size_t)which * dc, z);
      warp_stats<EPL>(z, dh, eps, mu, rs);
#pragma unroll
      for (int i = 0; i < EPL; i++) o[i] = (z[i] - mu) * rs * g[which][i] + bt[which][i];
      st_vec<T, EPL>(row + (size_t)(3 + which) * dc, o);
    }
  }
}

template <typename T, int EPL>
__global__ void __launch_bounds__(256) qknorm_bwd_kernel(const T* __restrict__ qkv, T* __restrict__ dqkv, long long ld,
    long long items, int hk, int dh, int dc, const void* __restrict__ qg, const void* __restrict__ kg, int p_dt, float eps,
    float* __restrict__ acc) {
  __shared__ float sacc[4 * 256];
  const int lane = threadIdx.x & 31;
  const long long w0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = ((long long)gridDim.x * blockDim.x) >> 5;
  for (int i = threadIdx.x; i < 4 * dh; i += blockDim.x) sacc[i] = 0.f;
  __syncthreads();
  float g[2][EPL], dg[2][EPL], db[2][EPL];
#pragma unroll
  for (int i = 0; i < EPL; i++) {
    g[0][i] = ldf(qg, lane * EPL + i, p_dt); g[1][i] = ldf(kg, lane * EPL + i, p_dt);
    dg[0][i] = dg[1][i] = db[0][i] = db[1][i] = 0.f;
  }
  for (long long it = w0; it < items; it += nw) {
    const long long m = it / hk;
    const int j = (int)(it - m * hk);
    const size_t off = (size_t)m * ld + (size_t)j * dh + lane * EPL;
#pragma unroll
    for (int which = 0; which < 2; which++) {
      float z[EPL], dv[EPL], o[EPL], mu, rs;
      ld_vec<T, EPL>(qkv + off + (size_t)which * dc, z);
      ld_vec<T, EPL>(dqkv + off + (size_t)(3 + which) * dc, dv);
      warp_stats<EPL>(z, dh, eps, mu, rs);
      float s1 = 0.f, s2 = 0.f;
#pragma unroll
      for (int i = 0; i < EPL; i++) {
        z[i] = (z[i] - mu) * rs;                        // zhat
        dg[which][i] += dv[i] * z[i];
        db[which][i] += dv[i];
        dv[i] *= g[which][i];                           // ghat
        s1 += dv[i]; s2 += dv[i] * z[i];
      }
      const float m1 = warp_sum(s1) / dh, m2 = warp_sum(s2) / dh;
#pragma unroll
      for (int i = 0; i < EPL; i++) o[i] = (dv[i] - m1 - z[i] * m2) * rs;
      st_vec<T, EPL>(dqkv + off + (size_t)which * dc, o);
    }
  }
#pragma unroll
  for (int which = 0; which < 2; which++)
#pragma unroll
    for (int i = 0; i < EPL; i++) {
      atomicAdd(&sacc[(2 * which) * dh + lane * EPL + i], dg[which][i]);
      atomicAdd(&sacc[(2 * which + 1) * dh + lane * EPL + i], db[which][i]);
    }
  __syncthreads();
  for (int i = threadIdx.x; i < 4 * dh; i += blockDim.x) atomicAdd(acc + i, sacc[i]);
}

template <typename T>
int launch_fwd(void* qkv, long long ld, long long items, int hk, int dh, int dc, const void* qg, const void* qb, const void* kg,
               const void* kb, int p_dt, float eps, int grid, cudaStream_t s) {
#define QF(E) qknorm_fwd_kernel<T, E><<<grid, 256, 0, s>>>((T*)qkv, ld, items, hk, dh, dc, qg, qb, kg, kb, p_dt, eps)
  switch (dh / 32) { case 1: QF(1); break; case 2: QF(2); break; case 4: QF(4); break; case 6: QF(6); break; case 8: QF(8); break; default: return ORBIT_ERR_SHAPE; }
#undef QF
  return ORBIT_OK;
}
template <typename T>
int launch_bwd(const void* qkv, void* dqkv, long long ld, long long items, int hk, int dh, int dc, const void* qg, const void* kg,
               int p_dt, float eps, float* acc, int grid, cudaStream_t s) {
#define QB(E) qknorm_bwd_kernel<T, E><<<grid, 256, 0, s>>>((const T*)qkv, (T*)dqkv, ld, items, hk, dh, dc, qg, kg, p_dt, eps, acc)
  switch (dh / 32) { case 1: QB(1); break; case 2: QB(2); break; case 4: QB(4); break; case 6: QB(6); break; case 8: QB(8); break; default: return ORBIT_ERR_SHAPE; }
#undef QB
  return ORBIT_OK;
}
int grid_items(long long items) {
  long long g = (items + 7) / 8;
  return (int)(g < 148 * 8 ? (g ? g : 1) : 148 * 8);
}
}  // namespace

bool qknorm_supported(int dh) { return dh == 32 || dh == 64 || dh == 128 || dh == 192 || dh == 256; }

int qknorm_fwd(void* qkv, long long ld, int M, int hk, int dh, int dc, const void* qg, const void* qb, const void* kg,
               const void* kb, int p_dt, int dt, float eps, cudaStream_t s) {
  const long long items = (long long)M * hk;
  int rc = dt == ORBIT_BF16 ? launch_fwd<bf16>(qkv, ld, items, hk, dh, dc, qg, qb, kg, kb, p_dt, eps, grid_items(items), s)
                            : launch_fwd<float>(qkv, ld, items, hk, dh, dc, qg, qb, kg, kb, p_dt, eps, grid_items(items), s);
  if (rc != ORBIT_OK) { set_error("qk-norm: d_h=%d unsupported (32, 64, 128, 256)", dh); return rc; }
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int qknorm_bwd(const void* qkv, void* dqkv, long long ld, int M, int hk, int dh, int dc, const void* qg, const void* kg,
               int p_dt, int dt, float eps, float* acc, cudaStream_t s) {
  const long long items = (long long)M * hk;
  int rc = dt == ORBIT_BF16 ? launch_bwd<bf16>(qkv, dqkv, ld, items, hk, dh, dc, qg, kg, p_dt, eps, acc, grid_items(items), s)
                            : launch_bwd<float>(qkv, dqkv, ld, items, hk, dh, dc, qg, kg, p_dt, eps, acc, grid_items(items), s);
  if (rc != ORBIT_OK) { set_error("qk-norm: d_h=%d unsupported (32, 64, 128, 256)", dh); return rc; }
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

}  // namespace orbit
