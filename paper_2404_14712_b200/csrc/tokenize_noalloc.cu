// tokenize_noalloc.cu -- orbit_tokenize_bwd_noalloc: the a1' tokeniser backward for callers that
// cannot provide (i.e. cannot cudaMalloc) a workspace: code under CUDA graph capture, tight serving loops, harnesses
// that forbid allocation.  The fp32 accumulators of dWp / dbp that orbit_tokenize_bwd takes as `ws` live here in a
// file-scope device array instead.
//
//  * The array is ORBIT_TOKENIZE_BWD_NOALLOC_MAX_BYTES (16 MiB) of device memory on EVERY GPU that loads liborbit.so,
//    held until the process exits.  It covers V (p^2 + 1) D <= 4 Mi fp32 accumulators (config 3: 91 x 17 x 2048 = 3.2 Mi).
//  * In host code the array's name is a host-side stand-in, not a device address: the address is taken with
//    cudaGetSymbolAddress once per device, with that device current, and cached per device ordinal.
//  * Every call (and every stream) shares the one array.  A call clears what it accumulates into before using it, so
//    calls that follow one another on a stream are independent; calls that OVERLAP on the GPU (different streams, or
//    different host threads launching to different streams) race on it and must be serialised by the caller.
//  * No cudaMalloc / cudaFree / allocating library routine anywhere on the path (memset, kernels, tensor-map encoding
//    on the host only).
#include <atomic>
#include "api_util.cuh"

#define ORBIT_TOKENIZE_BWD_NOALLOC_MAX_BYTES (16u << 20)

static __device__ __align__(256) unsigned char g_tok_bwd_scratch[ORBIT_TOKENIZE_BWD_NOALLOC_MAX_BYTES];

namespace orbit {
namespace {

// device address of g_tok_bwd_scratch on the CURRENT device (each device that loads the module has its own copy)
int scratch_address(void** out) {
  static std::atomic<void*> cached[ORBIT_MAX_DEV];
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) {
    cudaGetLastError();
    set_error("tokenize_bwd_noalloc: no usable CUDA device");
    return ORBIT_ERR_ARCH;
  }
  const bool cacheable = dev >= 0 && dev < ORBIT_MAX_DEV;
  if (cacheable) {
    void* p = cached[dev].load(std::memory_order_acquire);
    if (p) { *out = p; return ORBIT_OK; }
  }
  void* p = nullptr;
  const cudaError_t e = cudaGetSymbolAddress(&p, g_tok_bwd_scratch);
  if (e != cudaSuccess || !p) {
    cudaGetLastError();
    set_error("tokenize_bwd_noalloc: cudaGetSymbolAddress failed on device %d: %s", dev, cudaGetErrorString(e));
    return ORBIT_ERR_CUDA;
  }
  if (cacheable) cached[dev].store(p, std::memory_order_release);
  *out = p;
  return ORBIT_OK;
}

}  // namespace
}  // namespace orbit

using namespace orbit;

extern "C" {

size_t orbit_tokenize_bwd_noalloc_max_bytes(void) { return ORBIT_TOKENIZE_BWD_NOALLOC_MAX_BYTES; }

int orbit_tokenize_bwd_noalloc(const orbit_embed_desc* d, const float* x, const void* dtok, void* dWp, void* dbp,
                               void* stream) {
  if (!d) { set_error("embed desc is NULL"); return ORBIT_ERR_NULL; }
  if (d->V <= 0 || d->p <= 0 || d->D <= 0) { set_error("tokenize_bwd_noalloc: bad shape V=%d p=%d D=%d", d->V, d->p, d->D); return ORBIT_ERR_SHAPE; }
  // in 64 bits before anything else: the product below is what orbit_tokenize_bwd_workspace_bytes() computes
  const unsigned long long need = ((unsigned long long)d->V * ((unsigned long long)d->p * d->p + 1ull) * (unsigned long long)d->D * sizeof(float) + 255ull) & ~255ull;
  if (need > ORBIT_TOKENIZE_BWD_NOALLOC_MAX_BYTES) {
    set_error("tokenize_bwd_noalloc: V (p^2 + 1) D fp32 accumulators = %llu bytes exceed the built-in scratch of %u bytes; "
              "use orbit_tokenize_bwd with a caller workspace", need, (unsigned)ORBIT_TOKENIZE_BWD_NOALLOC_MAX_BYTES);
    return ORBIT_ERR_WORKSPACE;
  }
  ORBIT_TRY(check_device());
  void* scratch = nullptr;
  ORBIT_TRY(scratch_address(&scratch));
  // same checks, same kernels, same order as the caller-workspace entry point; it zeroes the accumulators first
  return orbit_tokenize_bwd(d, x, dtok, dWp, dbp, scratch, ORBIT_TOKENIZE_BWD_NOALLOC_MAX_BYTES, stream);
}

}  // extern "C"
