// vec8.cuh -- 16/32-byte vector load / store of 8 consecutive elements with a runtime dtype (row-wise kernels).
#pragma once
#include "common.cuh"

namespace orbit {

// 8 consecutive elements starting at element index i (i % 8 == 0, base 16B aligned)
__device__ __forceinline__ void ld8(const void* p, size_t i, int dt, float* v) {
  if (dt == ORBIT_BF16) {
    uint4 raw = *reinterpret_cast<const uint4*>((const bf16*)p + i);
    const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&raw);
#pragma unroll
    for (int j = 0; j < 4; j++) {
      float2 f = __bfloat1622float2(h[j]);
      v[2 * j] = f.x; v[2 * j + 1] = f.y;
    }
  } else {
    const float4* q = reinterpret_cast<const float4*>((const float*)p + i);
    float4 a = q[0], b = q[1];
    v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
  }
}
__device__ __forceinline__ void st8(void* p, size_t i, int dt, const float* v) {
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

}  // namespace orbit
