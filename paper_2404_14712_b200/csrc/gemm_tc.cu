// gemm_tc.cu -- bf16 GEMM on the 5th-gen tensor cores: TMA -> 128B-swizzled shared-memory ring -> tcgen05.mma
// (fp32 accumulators in TMEM, double buffered) -> tcgen05.ld epilogue with the fused bias / GELU / GELU' /
// residual / fp32-accumulate of GemmArgs.  Persistent, warp specialised: warp 0 = TMA producer, warp 1 = MMA
// issuer (+ TMEM allocation), warps 2..5 = epilogue (one TMEM lane quarter each).
//
// Operand majors: the forward GEMMs read W [in,out] as an N-major B; the dX GEMMs read it as a K-major B; the
// dW GEMMs read activations as an M-major A and an N-major B.  All four combinations go through
// the same kernel: only the TMA boxes, the UMMA descriptors' LBO/SBO and the per-k-step advance differ.
#include <cuda.h>
#include "common.cuh"
#include "ptx.cuh"

namespace orbit {
namespace {

constexpr int BM = 128, BN = 256, BK = 64, UK = 16;
constexpr int STAGES = 4;
constexpr int A_BYTES = BM * BK * 2;            // 16 KB
constexpr int B_BYTES = BN * BK * 2;            // 32 KB
constexpr int STAGE_BYTES = A_BYTES + B_BYTES;  // 48 KB
constexpr int NTHREADS = 192;
constexpr int TMEM_COLS = 512;                  // two 128x256 fp32 accumulators
constexpr size_t SMEM_BYTES = (size_t)STAGES * STAGE_BYTES + 1024 /*align*/ + 256 /*barriers*/;

struct Epi {
  void* C; long long ldc; int out_dt;
  const void* bias; int bias_dt;
  const void* resid; int resid_dt; long long ldr; int resid_row_mod;
  int accumulate; int act;
  void* aux_out; const void* aux_in; long long ld_aux; int aux_dt;
};

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

__device__ __forceinline__ void tile_coords(int t, int tiles_m, int tiles_n, int& mb, int& nb) {
  // groups of 16 M-blocks swept along N: concurrently running CTAs share A and B tiles through L2
  constexpr int GROUP = 16;
  const int group_size = GROUP * tiles_n;
  const int g = t / group_size, r = t - g * group_size;
  const int first_m = g * GROUP;
  const int gm = min(GROUP, tiles_m - first_m);
  mb = first_m + r % gm;
  nb = r / gm;
}

template <int A_MN, int B_MN>
__global__ void __launch_bounds__(NTHREADS, 1)
gemm_tc_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, Epi e, int M, int N, int K) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t bar_base = smem_base + STAGES * STAGE_BYTES;
  // barriers: full[STAGES], empty[STAGES], tmem_full[2], tmem_empty[2]; then the TMEM base address word
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
  auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * STAGES + a); };
  auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * STAGES + 2 + a); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * STAGES + 4);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int tiles_m = (M + BM - 1) / BM, tiles_n = (N + BN - 1) / BN;
  const int num_tiles = tiles_m * tiles_n;
  const int num_kb = (K + BK - 1) / BK;

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&tmA);
    ptx::prefetch_tmap(&tmB);
    for (int s = 0; s < STAGES; s++) { ptx::mbar_init(full_bar(s), 1); ptx::mbar_init(empty_bar(s), 1); }
    for (int a = 0; a < 2; a++) { ptx::mbar_init(tfull_bar(a), 1); ptx::mbar_init(tempty_bar(a), 4); }
    ptx::fence_barrier_init();
  }
  if (warp == 1) {
    ptx::tmem_alloc(tmem_slot, TMEM_COLS);
    ptx::tmem_relinquish();
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0) {
      int s = 0; uint32_t ph = 0;
      for (int t = blockIdx.x; t < num_tiles; t += gridDim.x) {
        int mb, nb;
        tile_coords(t, tiles_m, tiles_n, mb, nb);
        const int m0 = mb * BM, n0 = nb * BN;
        for (int kb = 0; kb < num_kb; kb++) {
          ptx::mbar_wait(empty_bar(s), ph ^ 1);
          ptx::mbar_expect_tx(full_bar(s), STAGE_BYTES);
          const uint32_t sa = smem_base + s * STAGE_BYTES, sb = sa + A_BYTES;
          const int k0 = kb * BK;
          if (A_MN) {  // A stored [K, M], M contiguous: boxes of 64 (M) x 64 (K)
#pragma unroll
            for (int i = 0; i < BM / 64; i++) ptx::tma_load_2d(sa + i * 8192, &tmA, full_bar(s), m0 + i * 64, k0);
          } else {     // A stored [M, K], K contiguous: one box of 64 (K) x 128 (M)
            ptx::tma_load_2d(sa, &tmA, full_bar(s), k0, m0);
          }
          if (B_MN) {  // B stored [K, N], N contiguous
#pragma unroll
            for (int i = 0; i < BN / 64; i++) ptx::tma_load_2d(sb + i * 8192, &tmB, full_bar(s), n0 + i * 64, k0);
          } else {     // B stored [N, K], K contiguous: one box of 64 (K) x 256 (N)
            ptx::tma_load_2d(sb, &tmB, full_bar(s), k0, n0);
          }
          if (++s == STAGES) { s = 0; ph ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (lane == 0) {
      constexpr uint32_t idesc = ptx::make_idesc_bf16(BM, BN, A_MN, B_MN);
      // K-major: 8-row groups 1024 B apart (SBO), k-step of 16 elements = +32 B inside the 128 B swizzle row.
      // MN-major: 64-wide MN chunks 8192 B apart (LBO), 8-k-row groups 1024 B apart (SBO), k-step = +2048 B.
      constexpr uint32_t a_lbo = A_MN ? 8192 : 16, a_sbo = 1024, a_step = A_MN ? 2048 : 32;
      constexpr uint32_t b_lbo = B_MN ? 8192 : 16, b_sbo = 1024, b_step = B_MN ? 2048 : 32;
      int s = 0; uint32_t ph = 0;
      int acc = 0; uint32_t aph = 0;
      for (int t = blockIdx.x; t < num_tiles; t += gridDim.x) {
        ptx::mbar_wait(tempty_bar(acc), aph ^ 1);
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + acc * BN;
        for (int kb = 0; kb < num_kb; kb++) {
          ptx::mbar_wait(full_bar(s), ph);
          ptx::tc_fence_after();
          const uint32_t sa = smem_base + s * STAGE_BYTES, sb = sa + A_BYTES;
#pragma unroll
          for (int k = 0; k < BK / UK; k++) {
            const uint64_t da = ptx::make_smem_desc(sa + k * a_step, a_lbo, a_sbo);
            const uint64_t db = ptx::make_smem_desc(sb + k * b_step, b_lbo, b_sbo);
            ptx::mma_f16_ss(d_tmem, da, db, idesc, (kb | k) != 0);
          }
          ptx::mma_commit(empty_bar(s));          // frees the smem stage once these MMAs have read it
          if (++s == STAGES) { s = 0; ph ^= 1; }
        }
        ptx::mma_commit(tfull_bar(acc));          // accumulator complete -> epilogue
        if (++acc == 2) { acc = 0; aph ^= 1; }
      }
    }
  } else {
    // ===================== epilogue: TMEM -> registers -> global =====================
    const int quarter = warp & 3;                 // TMEM lanes [32*quarter, +32) are this warp's
    int acc = 0; uint32_t aph = 0;
    for (int t = blockIdx.x; t < num_tiles; t += gridDim.x) {
      int mb, nb;
      tile_coords(t, tiles_m, tiles_n, mb, nb);
      const int row = mb * BM + quarter * 32 + lane;
      const int n0 = nb * BN;
      ptx::mbar_wait(tfull_bar(acc), aph);
      ptx::tc_fence_after();
      const uint32_t taddr = tmem_base + acc * BN + ((uint32_t)(quarter * 32) << 16);
      const int rrow = e.resid_row_mod > 0 ? (row % e.resid_row_mod) : row;
#pragma unroll 1
      for (int c = 0; c < BN / 32; c++) {
        uint32_t r[32];
        ptx::tmem_ld_32x32(taddr + c * 32, r);
        ptx::tmem_ld_wait();
        if (row < M) {
#pragma unroll
          for (int g8 = 0; g8 < 4; g8++) {
            const int col = n0 + c * 32 + g8 * 8;
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
      }
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(tempty_bar(acc));
      if (++acc == 2) { acc = 0; aph ^= 1; }
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc(tmem_base, TMEM_COLS);
  }
}

// ---- host side -------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn get_encode() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  }
  return fn;
}

// 2-D bf16 tensor map: `inner` contiguous elements, `outer` rows `ld` elements apart; 128B swizzle
int make_map(CUtensorMap* m, const void* base, long long inner, long long outer, long long ld, int box_inner,
             int box_outer) {
  EncodeTiledFn enc = get_encode();
  if (!enc) { set_error("cuTensorMapEncodeTiled entry point not found"); return ORBIT_ERR_CUDA; }
  cuuint64_t dims[2] = {(cuuint64_t)inner, (cuuint64_t)outer};
  cuuint64_t strides[1] = {(cuuint64_t)ld * 2};
  cuuint32_t box[2] = {(cuuint32_t)box_inner, (cuuint32_t)box_outer};
  cuuint32_t es[2] = {1, 1};
  CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    set_error("cuTensorMapEncodeTiled failed (%d): inner=%lld outer=%lld ld=%lld box=%dx%d", (int)r, inner, outer, ld,
              box_inner, box_outer);
    return ORBIT_ERR_CUDA;
  }
  return ORBIT_OK;
}

int num_sms() {
  static int n = 0;
  if (!n) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
    if (n <= 0) n = 148;
  }
  return n;
}

// ---- optional per-launch CUDA-event timing of the tensor-core GEMM (bench.py's roofline leg) ----------------
struct Prof {
  bool on = false;
  static constexpr int MAXP = 16384;
  cudaEvent_t* ev = nullptr;     // 2 * MAXP events, created lazily
  double* flops = nullptr;
  int n = 0;
};
Prof g_prof;

template <int A_MN, int B_MN>
int launch(const CUtensorMap& ma, const CUtensorMap& mb, const Epi& e, int M, int N, int K, cudaStream_t s) {
  static bool attr_set = false;
  if (!attr_set) {
    ORBIT_CUDA_CHECK(cudaFuncSetAttribute((const void*)gemm_tc_kernel<A_MN, B_MN>,
                                          cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES));
    attr_set = true;
  }
  const int tiles = cdiv(M, BM) * cdiv(N, BN);
  const int grid = tiles < num_sms() ? tiles : num_sms();
  gemm_tc_kernel<A_MN, B_MN><<<grid, NTHREADS, SMEM_BYTES, s>>>(ma, mb, e, M, N, K);
  return ORBIT_OK;
}
}  // namespace

int gemm_tc2_launch(const CUtensorMap& ma, const CUtensorMap& mb, const GemmArgs& g, bool a_mn, bool b_mn, int sms,
                    cudaStream_t s);   // gemm_tc2.cu

int gemm_profile_enable(int on) {
  if (on && !g_prof.ev) {
    g_prof.ev = new cudaEvent_t[2 * Prof::MAXP];
    g_prof.flops = new double[Prof::MAXP];
    for (int i = 0; i < 2 * Prof::MAXP; i++) ORBIT_CUDA_CHECK(cudaEventCreate(&g_prof.ev[i]));
  }
  g_prof.on = on != 0;
  g_prof.n = 0;
  return ORBIT_OK;
}
int gemm_profile_collect(double* ms, double* flops, long long* launches) {
  double t = 0, f = 0;
  for (int i = 0; i < g_prof.n; i++) {
    float e = 0.f;
    ORBIT_CUDA_CHECK(cudaEventSynchronize(g_prof.ev[2 * i + 1]));
    ORBIT_CUDA_CHECK(cudaEventElapsedTime(&e, g_prof.ev[2 * i], g_prof.ev[2 * i + 1]));
    t += e; f += g_prof.flops[i];
  }
  if (ms) *ms = t;
  if (flops) *flops = f;
  if (launches) *launches = g_prof.n;
  g_prof.n = 0;
  return ORBIT_OK;
}

bool gemm_tc_supported(const GemmArgs& g) {
  if (g.in_dtype != ORBIT_BF16 || g.alpha != 1.f) return false;
  if (g.M < 64 || g.N < 64 || g.K < 32 || (g.N % 8) != 0) return false;
  const bool a_k = (g.a_cs == 1 && g.a_rs % 8 == 0), a_m = (g.a_rs == 1 && g.a_cs % 8 == 0);
  const bool b_n = (g.b_cs == 1 && g.b_rs % 8 == 0), b_k = (g.b_rs == 1 && g.b_cs % 8 == 0);
  if (!(a_k || a_m) || !(b_n || b_k)) return false;
  auto al16 = [](const void* p) { return (((uintptr_t)p) & 15) == 0; };
  if (!al16(g.A) || !al16(g.B) || !al16(g.C)) return false;
  if (g.ldc % 8) return false;
  if (g.bias && !al16(g.bias)) return false;
  if (g.resid && (!al16(g.resid) || g.ldr % 8)) return false;
  if ((g.aux_out && (!al16(g.aux_out) || g.ld_aux % 8)) || (g.aux_in && (!al16(g.aux_in) || g.ld_aux % 8))) return false;
  if (g.accumulate && g.out_dtype != ORBIT_F32) return false;
  return true;
}

int gemm_tc(const GemmArgs& g, cudaStream_t s) {
  const bool a_mn = !(g.a_cs == 1 && g.a_rs % 8 == 0);
  const bool b_mn = (g.b_cs == 1 && g.b_rs % 8 == 0);
  // CTA-pair kernel (256 x 256 tiles) when the problem has at least one full pair tile; g_force_simt == 2
  // forces the single-CTA kernel (debug / A-B comparison)
  const bool pair = g_force_simt != 2 && g.M >= 256 && g.N >= 256;
  CUtensorMap ma, mb;
  if (a_mn) ORBIT_TRY(make_map(&ma, g.A, g.M, g.K, g.a_cs, 64, 64));               // [K rows, M contiguous]
  else      ORBIT_TRY(make_map(&ma, g.A, g.K, g.M, g.a_rs, 64, BM));               // [M rows, K contiguous]
  if (b_mn) ORBIT_TRY(make_map(&mb, g.B, g.N, g.K, g.b_rs, 64, 64));               // [K rows, N contiguous]
  else      ORBIT_TRY(make_map(&mb, g.B, g.K, g.N, g.b_cs, 64, pair ? 128 : BN));  // [N rows, K contiguous]
  const bool rec = g_prof.on && g_prof.n < Prof::MAXP;
  if (rec) ORBIT_CUDA_CHECK(cudaEventRecord(g_prof.ev[2 * g_prof.n], s));
  if (pair) {
    ORBIT_TRY(gemm_tc2_launch(ma, mb, g, a_mn, b_mn, num_sms(), s));
  } else {
    Epi e;
    e.C = g.C; e.ldc = g.ldc; e.out_dt = g.out_dtype; e.bias = g.bias; e.bias_dt = g.bias_dtype;
    e.resid = g.resid; e.resid_dt = g.resid_dtype; e.ldr = g.ldr; e.resid_row_mod = g.resid_row_mod;
    e.accumulate = g.accumulate; e.act = g.act; e.aux_out = g.aux_out; e.aux_in = g.aux_in; e.ld_aux = g.ld_aux;
    e.aux_dt = g.aux_dtype;
    if (!a_mn && b_mn) ORBIT_TRY((launch<0, 1>(ma, mb, e, g.M, g.N, g.K, s)));
    else if (!a_mn && !b_mn) ORBIT_TRY((launch<0, 0>(ma, mb, e, g.M, g.N, g.K, s)));
    else if (a_mn && b_mn) ORBIT_TRY((launch<1, 1>(ma, mb, e, g.M, g.N, g.K, s)));
    else ORBIT_TRY((launch<1, 0>(ma, mb, e, g.M, g.N, g.K, s)));
  }
  if (rec) {
    ORBIT_CUDA_CHECK(cudaEventRecord(g_prof.ev[2 * g_prof.n + 1], s));
    g_prof.flops[g_prof.n++] = 2.0 * g.M * g.N * g.K;
  }
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

}  // namespace orbit
