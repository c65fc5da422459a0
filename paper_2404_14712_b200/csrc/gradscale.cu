// gradscale.cu -- dynamic gradient scaling and fp32 gradient accumulation (PAPER.md:126:
// "we applied the PyTorch dynamic gradient scaling mechanism [24] ... detects the value range of the computed gradient
// magnitude ... scale the gradient magnitudes to the proper value range representable in BFLOAT16, and then reverse the
// scaling during the parameters update").  Three steps of that mechanism as multi-tensor, HBM-bound kernels:
//   orbit_grads_unscale_check : g <- g / S in place over a list of gradient tensors; found_inf <- 1 on any non-finite value
//   orbit_grads_accumulate    : acc (fp32) += g / S over the list (gradient accumulation across micro-steps in fp32)
//   orbit_grad_scale_update   : S <- S * backoff on overflow, S <- S * growth after `interval` clean steps
// S, found_inf and the growth tracker live on the device: no host synchronisation anywhere.
#include "api_util.cuh"

namespace orbit {
namespace {

constexpr int MAXSEG = 24;
constexpr int CHUNK = 8192;                 // elements per block: 32 per thread
struct Seg { void* g; float* acc; unsigned long long n; unsigned int first_chunk; };
struct SegList { Seg s[MAXSEG]; int count; unsigned int chunks; };

// MODE 0: g <- g * inv in place;  MODE 1: acc += g * inv (g untouched)
template <typename T, int MODE>
__global__ void __launch_bounds__(256)
grads_kernel(SegList L, const float* __restrict__ scale, float* __restrict__ found_inf) {
  int si = 0;
#pragma unroll 1
  while (si + 1 < L.count && blockIdx.x >= L.s[si + 1].first_chunk) si++;
  const Seg sg = L.s[si];
  const float inv = scale ? 1.0f / *scale : 1.0f;
  const unsigned long long base = (unsigned long long)(blockIdx.x - sg.first_chunk) * CHUNK;
  const unsigned long long end = base + CHUNK < sg.n ? base + CHUNK : sg.n;
  bool bad = false;
  constexpr int VEC = 16 / sizeof(T);        // elements per 16-byte access
  T* g = (T*)sg.g;
  // the segment base is 16-byte aligned (checked by the entry point) and CHUNK is a multiple of VEC
  for (unsigned long long i = base + (unsigned long long)threadIdx.x * VEC; i < end; i += 256ull * VEC) {
    if (i + VEC <= end) {
      uint4 raw = *reinterpret_cast<const uint4*>(g + i);
      T* e = reinterpret_cast<T*>(&raw);
      float v[VEC];
#pragma unroll
      for (int k = 0; k < VEC; k++) { const float gk = to_f<T>(e[k]); bad |= !isfinite(gk); v[k] = gk * inv; }
      if (MODE == 0) {
#pragma unroll
        for (int k = 0; k < VEC; k++) e[k] = from_f<T>(v[k]);
        *reinterpret_cast<uint4*>(g + i) = raw;
      } else {
#pragma unroll
        for (int k = 0; k < VEC; k += 4) {
          float4 a = *reinterpret_cast<const float4*>(sg.acc + i + k);
          a.x += v[k]; a.y += v[k + 1]; a.z += v[k + 2]; a.w += v[k + 3];
          *reinterpret_cast<float4*>(sg.acc + i + k) = a;
        }
      }
    } else {
      for (unsigned long long j = i; j < end; j++) {
        const float gj = to_f<T>(g[j]);
        bad |= !isfinite(gj);                 // the test of [24]: on the computed gradient, before it is unscaled
        const float v = gj * inv;
        if (MODE == 0) g[j] = from_f<T>(v); else sg.acc[j] += v;
      }
    }
  }
  if (found_inf && __syncthreads_or(bad) && threadIdx.x == 0) *found_inf = 1.0f;
}

__global__ void scale_update_kernel(float* scale, int* tracker, const float* found_inf, float growth, float backoff, int interval) {
  if (*found_inf != 0.0f) {
    *scale = *scale * backoff;
    *tracker = 0;
  } else {
    const int t = *tracker + 1;
    if (t >= interval) { *scale = *scale * growth; *tracker = 0; }
    else *tracker = t;
  }
}

int run_list(int n, void* const* grads, float* const* acc, const size_t* counts, int dtype, const float* scale, float* found_inf,
             int mode, cudaStream_t s) {
  int i = 0;
  while (i < n) {
    SegList L;
    L.count = 0; L.chunks = 0;
    while (i < n && L.count < MAXSEG) {
      if (counts[i] > 0) {
        const unsigned long long nch = (counts[i] + CHUNK - 1) / CHUNK;
        if ((unsigned long long)L.chunks + nch > 0x7fffffffull) break;
        Seg& sg = L.s[L.count++];
        sg.g = grads[i]; sg.acc = acc ? acc[i] : nullptr; sg.n = counts[i]; sg.first_chunk = L.chunks;
        L.chunks += (unsigned int)nch;
      }
      i++;
    }
    if (!L.count) { if (i < n) { set_error("grads: tensor %d too large for one launch", i); return ORBIT_ERR_SHAPE; } break; }
    if (dtype == ORBIT_BF16) {
      if (mode == 0) grads_kernel<bf16, 0><<<L.chunks, 256, 0, s>>>(L, scale, found_inf);
      else grads_kernel<bf16, 1><<<L.chunks, 256, 0, s>>>(L, scale, found_inf);
    } else {
      if (mode == 0) grads_kernel<float, 0><<<L.chunks, 256, 0, s>>>(L, scale, found_inf);
      else grads_kernel<float, 1><<<L.chunks, 256, 0, s>>>(L, scale, found_inf);
    }
    ORBIT_LAUNCH_CHECK();
  }
  return ORBIT_OK;
}

int check_list(const char* who, int n, const void* const* grads, const float* const* acc, const size_t* counts, int dtype) {
  if (n < 0) { set_error("%s: negative tensor count", who); return ORBIT_ERR_SHAPE; }
  if (n > 0 && (!grads || !counts)) { set_error("%s: NULL list", who); return ORBIT_ERR_NULL; }
  if (!valid_dtype(dtype)) { set_error("%s: bad dtype", who); return ORBIT_ERR_DTYPE; }
  for (int i = 0; i < n; i++) {
    if (counts[i] == 0) continue;
    if (!grads[i] || (acc && !acc[i])) { set_error("%s: NULL tensor %d", who, i); return ORBIT_ERR_NULL; }
    if (!aligned16(grads[i]) || (acc && !aligned16(acc[i]))) { set_error("%s: tensor %d not 16B aligned", who, i); return ORBIT_ERR_ALIGN; }
  }
  return ORBIT_OK;
}
}  // namespace
}  // namespace orbit

using namespace orbit;

extern "C" {

int orbit_grads_unscale_check(int n, void* const* grads, const size_t* counts, orbit_dtype dtype, const float* scale,
                              float* found_inf, void* stream) {
  ORBIT_TRY(check_list("grads_unscale_check", n, grads, nullptr, counts, dtype));
  if (!found_inf) { set_error("grads_unscale_check: found_inf is NULL"); return ORBIT_ERR_NULL; }
  ORBIT_TRY(check_device());
  return run_list(n, grads, nullptr, counts, dtype, scale, found_inf, 0, (cudaStream_t)stream);
}

int orbit_grads_accumulate(int n, const void* const* grads, float* const* acc, const size_t* counts, orbit_dtype dtype,
                           const float* scale, float* found_inf, void* stream) {
  if (n > 0 && !acc) { set_error("grads_accumulate: NULL accumulator list"); return ORBIT_ERR_NULL; }
  ORBIT_TRY(check_list("grads_accumulate", n, grads, acc, counts, dtype));
  ORBIT_TRY(check_device());
  return run_list(n, const_cast<void* const*>(grads), acc, counts, dtype, scale, found_inf, 1, (cudaStream_t)stream);
}

int orbit_grad_scale_update(float* scale, int* growth_tracker, const float* found_inf, float growth_factor,
                            float backoff_factor, int growth_interval, void* stream) {
  if (!scale || !growth_tracker || !found_inf) { set_error("grad_scale_update: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!(growth_factor > 1.0f) || !(backoff_factor > 0.0f && backoff_factor < 1.0f) || growth_interval < 1) {
    set_error("grad_scale_update: need growth_factor > 1, 0 < backoff_factor < 1, growth_interval >= 1");
    return ORBIT_ERR_SHAPE;
  }
  ORBIT_TRY(check_device());
  scale_update_kernel<<<1, 1, 0, (cudaStream_t)stream>>>(scale, growth_tracker, found_inf, growth_factor, backoff_factor, growth_interval);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

}  // extern "C"
