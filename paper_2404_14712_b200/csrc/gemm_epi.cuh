// gemm_epi.cuh -- fused epilogue shared by the tensor-core GEMM kernels: one thread owns one output row and
// processes 32 consecutive accumulator columns (one tcgen05.ld.32x32b.x32) in 8-element / 16-byte groups:
//   v = acc (+ bias[n]) ; GELU (side output of the pre-activation) | * GELU'(aux) ; (+ resid) ; (+ C) ; store.
#pragma once
#include "common.cuh"

namespace orbit {
namespace epi {

struct Args {
  void* C; long long ldc; int out_dt;
  const void* bias; int bias_dt;
  const void* resid; int resid_dt; long long ldr; int resid_row_mod;
  int accumulate; int act;
  void* aux_out; const void* aux_in; long long ld_aux; int aux_dt;
};

inline Args from_gemm(const GemmArgs& g) {
  Args e;
  e.C = g.C; e.ldc = g.ldc; e.out_dt = g.out_dtype; e.bias = g.bias; e.bias_dt = g.bias_dtype;
  e.resid = g.resid; e.resid_dt = g.resid_dtype; e.ldr = g.ldr; e.resid_row_mod = g.resid_row_mod;
  e.accumulate = g.accumulate; e.act = g.act; e.aux_out = g.aux_out; e.aux_in = g.aux_in; e.ld_aux = g.ld_aux;
  e.aux_dt = g.aux_dtype;
  return e;
}

// strided batch (GemmArgs::batch): problem `bi` writes C + bi*c_bs and reads bias + bi*bias_bs (element offsets)
__device__ __forceinline__ void offset_batch(Args& e, int bi, long long c_bs, long long bias_bs) {
  e.C = (char*)e.C + (size_t)bi * c_bs * (e.out_dt == ORBIT_BF16 ? 2 : 4);
  if (e.bias) e.bias = (const char*)e.bias + (size_t)bi * bias_bs * (e.bias_dt == ORBIT_BF16 ? 2 : 4);
}

__device__ __forceinline__ void load8(const void* p, size_t i, int dt, float* v) {
  if (dt == ORBIT_BF16) {
    uint4 raw = *reinterpret_cast<const uint4*>((const bf16*)p + i);
    const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&raw);
#pragma unroll
    for (int j = 0; j < 4; j++) { float2 f = __bfloat1622float2(h[j]); v[2 * j] = f.x; v[2 * j + 1] = f.y; }
  } else {
    const float4* q = reinterpret_cast<const float4*>((const float*)p + i);
    float4 a = q[0], b = q[1];
    v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
  }
}
__device__ __forceinline__ void store8(void* p, size_t i, int dt, const float* v) {
  if (dt == ORBIT_BF16) {
    uint4 raw;
    __nv_bfloat162* h = reinterpret_cast<__nv_bfloat162*>(&raw);
#pragma unroll
    for (int j = 0; j < 4; j++) h[j] = __floats2bfloat162_rn(v[2 * j], v[2 * j + 1]);
    *reinterpret_cast<uint4*>((bf16*)p + i) = raw;
  } else {
    float4* q = reinterpret_cast<float4*>((float*)p + i);
    q[0] = make_float4(v[0], v[1], v[2], v[3]);
    q[1] = make_float4(v[4], v[5], v[6], v[7]);
  }
}

// r[32]: fp32 accumulator bits of row `row`, columns [col0, col0 + 32)
__device__ __forceinline__ void chunk32(const Args& e, const uint32_t* r, int row, int rrow, int col0, int N) {
#pragma unroll
  for (int g8 = 0; g8 < 4; g8++) {
    const int col = col0 + g8 * 8;
    if (col < N) {
      float v[8];
#pragma unroll
      for (int j = 0; j < 8; j++) v[j] = __uint_as_float(r[g8 * 8 + j]);
      if (e.bias) {
        float b[8];
        load8(e.bias, col, e.bias_dt, b);
#pragma unroll
        for (int j = 0; j < 8; j++) v[j] += b[j];
      }
      if (e.act == ACT_GELU) {
        if (e.aux_out) {
          store8(e.aux_out, (size_t)row * e.ld_aux + col, e.aux_dt, v);
          if (e.aux_dt == ORBIT_BF16) {
#pragma unroll
            for (int j = 0; j < 8; j++) v[j] = __bfloat162float(__float2bfloat16_rn(v[j]));
          }
        }
#pragma unroll
        for (int j = 0; j < 8; j++) v[j] = gelu_f(v[j]);
      } else if (e.act == ACT_GELU_GRAD) {
        float u[8];
        load8(e.aux_in, (size_t)row * e.ld_aux + col, e.aux_dt, u);
#pragma unroll
        for (int j = 0; j < 8; j++) v[j] *= gelu_grad_f(u[j]);
      }
      if (e.resid) {
        float q[8];
        load8(e.resid, (size_t)rrow * e.ldr + col, e.resid_dt, q);
#pragma unroll
        for (int j = 0; j < 8; j++) v[j] += q[j];
      }
      const size_t ci = (size_t)row * e.ldc + col;
      if (e.accumulate) {
        float q[8];
        load8(e.C, ci, e.out_dt, q);
#pragma unroll
        for (int j = 0; j < 8; j++) v[j] += q[j];
      }
      store8(e.C, ci, e.out_dt, v);
    }
  }
}

}  // namespace epi
}  // namespace orbit
