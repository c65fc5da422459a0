// common.cuh -- shared device/host helpers of liborbit (sm_100a).  Not shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include <stdio.h>
#include <atomic>
#include <utility>
#include "../../include/orbit.h"

namespace orbit {

typedef __nv_bfloat16 bf16;

// ---- error state (thread-local) --------------------------------------------------------------
void set_error(const char* fmt, ...);
extern thread_local long long g_launches;
// A/B switch between kernel variants (0 = the product dispatch).  Compiled in only with -DORBIT_DEBUG_SWITCH
// (`ORBIT_DEBUG_SWITCH=1 python -m paper_2404_14712_b200.build` -> liborbit_dbg.so, which also exports
// orbit_set_debug_force_simt, declared in csrc/orbit_debug.h); in the shipped liborbit.so it is the constant 0, so the
// alternative branches fold away and no process-wide dispatch state exists.
#ifdef ORBIT_DEBUG_SWITCH
extern int g_force_simt;
#else
constexpr int g_force_simt = 0;
#endif
inline void count_launch(int n = 1) { g_launches += n; }

#define ORBIT_CUDA_CHECK(expr)                                                                   \
  do {                                                                                           \
    cudaError_t _e = (expr);                                                                     \
    if (_e != cudaSuccess) {                                                                     \
      orbit::set_error("%s:%d %s -> %s", __FILE__, __LINE__, #expr, cudaGetErrorString(_e));     \
      return ORBIT_ERR_CUDA;                                                                     \
    }                                                                                            \
  } while (0)

#define ORBIT_LAUNCH_CHECK()                                                                     \
  do {                                                                                           \
    orbit::count_launch();                                                                       \
    cudaError_t _e = cudaGetLastError();                                                         \
    if (_e != cudaSuccess) {                                                                     \
      orbit::set_error("%s:%d launch -> %s", __FILE__, __LINE__, cudaGetErrorString(_e));        \
      return ORBIT_ERR_CUDA;                                                                     \
    }                                                                                            \
  } while (0)

// ---- per-device one-time launch setup --------------------------------------------------------------
// cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the (function, device) pair, not to the process: the record is
// kept per device ordinal (atomics: two host threads may race, both then set the same value, which is harmless) and
// remembers the largest size requested so far, so call sites whose size depends on the shape stay correct.
constexpr int ORBIT_MAX_DEV = 64;
struct SmemAttrOnce { std::atomic<int> bytes[ORBIT_MAX_DEV]; };
int smem_attr_once(SmemAttrOnce& st, const void* fn, int bytes);
int device_ordinal();            // cudaGetDevice (0 when it fails; the launch that follows reports the error)
int num_sms();                   // multiprocessor count of the current device (cached per device)
#define ORBIT_SMEM_ATTR(fn, nbytes)                                                              \
  do {                                                                                           \
    static orbit::SmemAttrOnce _once;                                                            \
    ORBIT_TRY(orbit::smem_attr_once(_once, (const void*)(fn), (int)(nbytes)));                   \
  } while (0)

// ---- programmatic dependent launch (PDL) -------------------------------------------------------------------
// The block is a chain of 25-80 short dependent kernels; at C2 / C4 sizes the drain of one kernel plus the launch latency
// and on-chip prologue (barrier init, TMEM allocation, tensor-map fetch) of the next is a few microseconds per link.  Kernels
// launched through launch_pdl() may start while their predecessor is still running; they run their prologue, then
// pdl_wait() (griddepcontrol.wait: returns once every prerequisite grid has completed and its writes are visible) BEFORE
// their first global-memory access, then pdl_trigger() so that their own successor may be scheduled as soon as all their
// CTAs are resident.  A kernel launched without the attribute (or after a memset) behaves as usual: the two
// instructions are no-ops there.  ORBIT_PDL=0 disables the attribute (A/B).
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
bool pdl_enabled();
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = pdl_enabled() ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

#define ORBIT_TRY(expr)                                                                          \
  do {                                                                                           \
    int _s = (expr);                                                                             \
    if (_s != ORBIT_OK) return _s;                                                               \
  } while (0)

inline size_t dsize(int dt) { return dt == ORBIT_BF16 ? 2 : 4; }
inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline int cdiv(long long a, long long b) { return (int)((a + b - 1) / b); }

// ---- runtime-dtype scalar access (warp-uniform branch) ----------------------------------------
__device__ __forceinline__ float ldf(const void* p, size_t i, int dt) {
  return dt == ORBIT_BF16 ? __bfloat162float(((const bf16*)p)[i]) : ((const float*)p)[i];
}
__device__ __forceinline__ void stf(void* p, size_t i, float v, int dt) {
  if (dt == ORBIT_BF16) ((bf16*)p)[i] = __float2bfloat16_rn(v);
  else ((float*)p)[i] = v;
}
template <typename T> __device__ __forceinline__ float to_f(T v);
template <> __device__ __forceinline__ float to_f<float>(float v) { return v; }
template <> __device__ __forceinline__ float to_f<bf16>(bf16 v) { return __bfloat162float(v); }
template <typename T> __device__ __forceinline__ T from_f(float v);
template <> __device__ __forceinline__ float from_f<float>(float v) { return v; }
template <> __device__ __forceinline__ bf16 from_f<bf16>(float v) { return __float2bfloat16_rn(v); }

// ---- math --------------------------------------------------------------------------------------
// exact-erf GELU ("GeLU"; reading R7) and its derivative Phi(u) + u phi(u)
__device__ __forceinline__ float gelu_f(float u) { return 0.5f * u * (1.0f + erff(u * 0.70710678118654752f)); }
__device__ __forceinline__ float gelu_grad_f(float u) {
  float Phi = 0.5f * (1.0f + erff(u * 0.70710678118654752f));
  float phi = 0.39894228040143268f * __expf(-0.5f * u * u);
  return Phi + u * phi;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
// block-wide sum, blockDim.x multiple of 32, <= 1024 threads; `sh` >= 32 floats
__device__ __forceinline__ float block_sum(float v, float* sh) {
  int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  v = warp_sum(v);
  __syncthreads();
  if (lane == 0) sh[w] = v;
  __syncthreads();
  float r = lane < nw ? sh[lane] : 0.f;
  r = warp_sum(r);
  return r;
}

// ---- internal GEMM interface ---------------------------------------------------------------------
// C[m,n] = epi( alpha * sum_k A(m,k) B(k,n) ), A(m,k) = A[m*a_rs + k*a_cs], B(k,n) = B[k*b_rs + n*b_cs]
enum { ACT_NONE = 0, ACT_GELU = 1 /* C = gelu(v), aux_out = v */, ACT_GELU_GRAD = 2 /* C = v * gelu'(aux_in) */ };
struct GemmArgs {
  const void* A = nullptr; long long a_rs = 0, a_cs = 0;
  const void* B = nullptr; long long b_rs = 0, b_cs = 0;
  void* C = nullptr; long long ldc = 0;
  int M = 0, N = 0, K = 0;
  int in_dtype = ORBIT_F32;      // dtype of A and B
  int out_dtype = ORBIT_F32;     // dtype of C (and aux_out)
  float alpha = 1.f;
  const void* bias = nullptr; int bias_dtype = ORBIT_F32;              // [N]
  const void* resid = nullptr; int resid_dtype = ORBIT_F32; long long ldr = 0; int resid_row_mod = 0;
  int accumulate = 0;            // C += (only meaningful for fp32 C)
  int act = ACT_NONE;
  void* aux_out = nullptr; const void* aux_in = nullptr; long long ld_aux = 0; int aux_dtype = ORBIT_F32;
  // strided batch: problem i uses A + i*a_bs, B + i*b_bs, C + i*c_bs, bias + i*bias_bs (element offsets; the
  // per-head products of the front end).  resid / aux / accumulate must be unset when batch > 1.
  int batch = 1; long long a_bs = 0, b_bs = 0, c_bs = 0, bias_bs = 0;
};
int gemm(const GemmArgs& g, cudaStream_t s);           // dispatcher (tensor-core path or SIMT)
int gemm_simt(const GemmArgs& g, cudaStream_t s);      // fp32-FMA kernels, any dtype/stride
int gemm_tc(const GemmArgs& g, cudaStream_t s);        // tcgen05 + TMA, bf16 in / fp32 accumulate
bool gemm_tc_supported(const GemmArgs& g);

// ---- optional per-launch CUDA-event timing (bench.py's roofline legs) ------------------------------------------------
// When switched on, a ProfScope records an event pair on the launching stream around the kernel(s) issued inside it, tagged
// with a category and the algorithmic work of those launches (FLOPs for the tensor-bound categories, bytes for the
// HBM-bound ones).  Single-threaded use (bench.py); off by default: the scope then costs one load.
enum { PROF_GEMM = 0, PROF_ATTN_FWD = 1, PROF_ATTN_BWD = 2, PROF_LN = 3, PROF_FRONT = 4, PROF_NCAT = 5 };
int prof_enable(int on);
int prof_collect(int cat, double* ms, double* work, long long* launches);     // sums over the category; clears it
struct ProfScope {
  int slot; cudaStream_t s;
  ProfScope(int cat, double work, cudaStream_t stream);
  ~ProfScope();
};

// widest row the LayerNorm kernels take (backward: 4 chunks of 8 columns per thread, 512 threads); entry points reject
// wider models with ORBIT_ERR_SHAPE before the first launch
constexpr int ORBIT_LN_MAX_D = 16384;

// ---- row-wise / reduction kernels (rowops.cu) -----------------------------------------------------
int layernorm_fwd(const void* x, int x_dt, const void* gamma, const void* beta, int p_dt, void* out, int out_dt,
                  float* mean, float* rstd, int M, int D, float eps, void* x_copy, cudaStream_t s);
// dz from d(out); dx_out = add (nullable, add_dt) + dz, written as f32 to dx_f32 (nullable) and as out_dt to
// dx_out (nullable); dgamma/dbeta accumulated into fp32 acc buffers (zeroed by the caller).
int layernorm_bwd(const void* dout, int dout_dt, const void* x, int x_dt, const float* mean, const float* rstd,
                  const void* gamma, int p_dt, const void* add, int add_dt, float* dx_f32, void* dx_out,
                  int out_dt, float* dgamma_acc, float* dbeta_acc, int M, int D, cudaStream_t s);
// TMA-staged variants (layernorm_tma.cu), same contracts; used whenever two row stages fit in shared memory
bool layernorm_tma_supported(int D, int x_dt, int dout_dt /* -1: forward */, int add_dt, bool has_add);
int layernorm_fwd_tma(const void* x, int x_dt, const void* gamma, const void* beta, int p_dt, void* out, int out_dt,
                     float* mean, float* rstd, int M, int D, float eps, void* x_copy, cudaStream_t s);
int layernorm_bwd_tma(const void* dout, int dout_dt, const void* x, int x_dt, const float* mean, const float* rstd,
                     const void* gamma, int p_dt, const void* add, int add_dt, float* dx_f32, void* dx_out,
                     int out_dt, float* dgamma_acc, float* dbeta_acc, int M, int D, cudaStream_t s);
// out[n] = sum_m in[m*ld + n]  (fp32 atomics into acc, caller zeroes) ; optional bf16/f32 copy of `in`
int colsum(const void* in, int in_dt, long long ld, int M, int N, float* acc, void* copy_out, int copy_dt,
           long long ld_copy, cudaStream_t s);
int cast_copy(const void* in, int in_dt, void* out, int out_dt, size_t n, cudaStream_t s);
// up to 16 fp32 -> out_dt casts in one launch
struct CastSeg { const float* src; void* dst; size_t n; };
struct CastSegs {
  CastSeg s[16]; int count = 0;
  void add(const float* src, void* dst, size_t n) { s[count].src = src; s[count].dst = dst; s[count].n = n; count++; }
};
int cast_multi(const CastSegs& segs, int out_dt, cudaStream_t s);
// The tail of a block backward in ONE launch: up to 12 column sums (acc[n] += sum_m in[m, n], as colsum), each 256-column group
// cast to `out` (out_dt) by the LAST of its row blocks to finish (one ticket word per group, zero on entry and on exit), plus the
// fp32 -> out_dt casts of accumulators that were complete before the launch, spread over all blocks.
struct TailSeg { const void* in; int in_dt; long long ld; int M, N; float* acc; void* out; int first_block, first_group, gx, gy, rows_per_block; };
struct TailSegs {
  TailSeg s[12]; int count = 0;
  void add(const void* in, int in_dt, long long ld, int M, int N, float* acc, void* out) {
    TailSeg& t = s[count++]; t.in = in; t.in_dt = in_dt; t.ld = ld; t.M = M; t.N = N; t.acc = acc; t.out = out;
    t.first_block = t.first_group = t.gx = t.gy = t.rows_per_block = 0;
  }
};
inline size_t block_tail_tickets(size_t total_columns, int segments) { return total_columns / 256 + segments + 8; }
int block_tail(TailSegs& sums, const CastSegs& casts, int out_dt, unsigned int* tickets, cudaStream_t s);
int fill_zero(void* p, size_t bytes, cudaStream_t s);
// out = a (a_dt) + b_f32 + bias (p_dt)  (combine of fp32 Hybrid-STOP partials)
int add_partial(const void* a, int a_dt, const float* part, const void* bias, int p_dt, void* out, int out_dt,
                int M, int D, cudaStream_t s);

// ---- QK-LayerNorm (qknorm.cu): buffer layout [M, ld] with columns [Q | K | V | Q' | K'], dc each -------
bool qknorm_supported(int dh);
int qknorm_fwd(void* qkv, long long ld, int M, int hk, int dh, int dc, const void* qg, const void* qb, const void* kg,
               const void* kb, int p_dt, int dt, float eps, cudaStream_t s);
// dqkv holds dQ', dK' (columns 3dc, 4dc) on entry; dQ, dK are written to columns 0, dc; acc [4][dh] += dgamma/dbeta
int qknorm_bwd(const void* qkv, void* dqkv, long long ld, int M, int hk, int dh, int dc, const void* qg, const void* kg,
               int p_dt, int dt, float eps, float* acc, cudaStream_t s);

int mse_loss_grad(const void* y, const void* t, int dt, void* dy, float* loss, size_t n, cudaStream_t s);

// ---- attention (attention_simt.cu / attention_tc.cu) ------------------------------------------------
// qkv: [B*N, ld] with Q at column q_off + j*dh, K at k_off + j*dh, V at v_off + j*dh for head j
struct AttnArgs {
  const void* qkv = nullptr; long long ld = 0; int q_off = 0, k_off = 0, v_off = 0;
  int B = 0, N = 0, heads = 0, dh = 0; int dtype = ORBIT_F32;
  void* O = nullptr; long long ldo = 0;               // [B*N, heads*dh]
  float* lse = nullptr;                               // [B, heads, N] natural-log sum-exp of scaled logits
  // backward
  const void* dO = nullptr; long long lddo = 0;
  void* dqkv = nullptr;                               // same layout as qkv
  float* delta = nullptr;                             // [B, heads, N] workspace
  float* dq_acc = nullptr;                            // [B*N, heads*dh] fp32 workspace (tensor-core path)
};
int attention_fwd(const AttnArgs& a, cudaStream_t s);
int attention_bwd(const AttnArgs& a, cudaStream_t s);
int attention_fwd_simt(const AttnArgs& a, cudaStream_t s);
int attention_bwd_simt(const AttnArgs& a, cudaStream_t s);

}  // namespace orbit
