// gemm_tc.cu -- bf16 GEMM on the 5th-gen tensor cores: TMA -> 128B-swizzled shared-memory ring -> tcgen05.mma
// (fp32 accumulators in TMEM, double buffered) -> tcgen05.ld epilogue with the fused bias / GELU / GELU' /
// residual / fp32-accumulate of GemmArgs.  Persistent, warp specialised: warp 0 = TMA producer, warp 1 = MMA
// issuer (+ TMEM allocation), warps 2..5 = epilogue (one TMEM lane quarter each).
//
// Operand majors: the forward GEMMs read W [in,out] as an N-major B; the dX GEMMs read it as a K-major B; the
// dW GEMMs read activations as an M-major A and an N-major B.  All four combinations go through
// the same kernel: only the TMA boxes, the UMMA descriptors' LBO/SBO and the per-k-step advance differ.
#include <cuda.h>
#include <atomic>
#include "common.cuh"
#include "gemm_epi.cuh"
#include "ptx.cuh"

namespace orbit {
namespace {

constexpr int BM = 128, BK = 64, UK = 16;
constexpr int NTHREADS = 192;
constexpr int A_BYTES = BM * BK * 2;            // 16 KB
// per-BN configuration: BN = 256 (4 stages of 48 KB) for the wide GEMMs, BN = 128 (6 stages of 32 KB) for
// the d_a-wide per-head products of the front end
template <int BN> struct TcCfg {
  static constexpr int B_BYTES = BN * BK * 2;
  static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
  static constexpr int STAGES = BN == 256 ? 4 : 6;
  static constexpr int TMEM_COLS = 2 * BN;      // two 128 x BN fp32 accumulators
  static constexpr size_t SMEM_BYTES = (size_t)STAGES * STAGE_BYTES + 1024 /*align*/ + 256 /*barriers*/;
};

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

template <int A_MN, int B_MN, int BN>
__global__ void __launch_bounds__(NTHREADS, 1)
gemm_tc_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, epi::Args e0, int M, int N, int K,
               int batch, long long c_bs, long long bias_bs) {
  using Cf = TcCfg<BN>;
  constexpr int STAGES = Cf::STAGES, STAGE_BYTES = Cf::STAGE_BYTES;
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
  const int tiles_per_batch = tiles_m * tiles_n;
  const int num_tiles = tiles_per_batch * batch;
  const int num_kb = (K + BK - 1) / BK;

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&tmA);
    ptx::prefetch_tmap(&tmB);
    for (int s = 0; s < STAGES; s++) { ptx::mbar_init(full_bar(s), 1); ptx::mbar_init(empty_bar(s), 1); }
    for (int a = 0; a < 2; a++) { ptx::mbar_init(tfull_bar(a), 1); ptx::mbar_init(tempty_bar(a), 4); }
    ptx::fence_barrier_init();
  }
  if (warp == 1) {
    ptx::tmem_alloc(tmem_slot, Cf::TMEM_COLS);
    ptx::tmem_relinquish();
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));
  pdl_wait();                                    // only on-chip state and kernel parameters were touched above
  pdl_trigger();

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0) {
      int s = 0; uint32_t ph = 0;
      for (int t = blockIdx.x; t < num_tiles; t += gridDim.x) {
        const int bi = t / tiles_per_batch;
        int mb, nb;
        tile_coords(t - bi * tiles_per_batch, tiles_m, tiles_n, mb, nb);
        const int m0 = mb * BM, n0 = nb * BN;
        for (int kb = 0; kb < num_kb; kb++) {
          ptx::mbar_wait(empty_bar(s), ph ^ 1);
          ptx::mbar_expect_tx(full_bar(s), STAGE_BYTES);
          const uint32_t sa = smem_base + s * STAGE_BYTES, sb = sa + A_BYTES;
          const int k0 = kb * BK;
          if (A_MN) {  // A stored [K, M], M contiguous: boxes of 64 (M) x 64 (K)
#pragma unroll
            for (int i = 0; i < BM / 64; i++) ptx::tma_load_3d(sa + i * 8192, &tmA, full_bar(s), m0 + i * 64, k0, bi);
          } else {     // A stored [M, K], K contiguous: one box of 64 (K) x 128 (M)
            ptx::tma_load_3d(sa, &tmA, full_bar(s), k0, m0, bi);
          }
          if (B_MN) {  // B stored [K, N], N contiguous
#pragma unroll
            for (int i = 0; i < BN / 64; i++) ptx::tma_load_3d(sb + i * 8192, &tmB, full_bar(s), n0 + i * 64, k0, bi);
          } else {     // B stored [N, K], K contiguous: one box of 64 (K) x BN (N)
            ptx::tma_load_3d(sb, &tmB, full_bar(s), k0, n0, bi);
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
      const int bi = t / tiles_per_batch;
      int mb, nb;
      tile_coords(t - bi * tiles_per_batch, tiles_m, tiles_n, mb, nb);
      const int row = mb * BM + quarter * 32 + lane;
      const int n0 = nb * BN;
      epi::Args e = e0;
      if (batch > 1) epi::offset_batch(e, bi, c_bs, bias_bs);
      ptx::mbar_wait(tfull_bar(acc), aph);
      ptx::tc_fence_after();
      const uint32_t taddr = tmem_base + acc * BN + ((uint32_t)(quarter * 32) << 16);
      const int rrow = e.resid_row_mod > 0 ? (row % e.resid_row_mod) : row;
#pragma unroll 1
      for (int c = 0; c < BN / 32; c++) {
        uint32_t r[32];
        ptx::tmem_ld_32x32(taddr + c * 32, r);
        ptx::tmem_ld_wait();
        if (row < M) epi::chunk32(e, r, row, rrow, n0 + c * 32, N);
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
    ptx::tmem_dealloc(tmem_base, Cf::TMEM_COLS);
  }
}

// ---- host side -------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn get_encode() {
  static std::atomic<EncodeTiledFn> cached{nullptr};     // process-wide entry point; host threads may race to fill it (same value)
  EncodeTiledFn fn = cached.load(std::memory_order_relaxed);
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess) {
      fn = (EncodeTiledFn)p;
      cached.store(fn, std::memory_order_relaxed);
    }
  }
  return fn;
}

// bf16 tensor map over `batch` 2-D problems `bstride` elements apart: `inner` contiguous elements, `outer` rows `ld`
// elements apart; 128B swizzle; box = box_inner x box_outer x 1 (out-of-bounds elements read as zero per problem)
int make_map(CUtensorMap* m, const void* base, long long inner, long long outer, long long ld, int box_inner,
             int box_outer, int batch, long long bstride, CUtensorMapSwizzle swz = CU_TENSOR_MAP_SWIZZLE_128B, int esz = 2) {
  EncodeTiledFn enc = get_encode();
  if (!enc) { set_error("cuTensorMapEncodeTiled entry point not found"); return ORBIT_ERR_CUDA; }
  if (batch <= 1) { batch = 1; bstride = ld * outer; }
  cuuint64_t dims[3] = {(cuuint64_t)inner, (cuuint64_t)outer, (cuuint64_t)batch};
  cuuint64_t strides[2] = {(cuuint64_t)ld * esz, (cuuint64_t)bstride * esz};
  if (batch == 1) strides[1] = strides[0] * dims[1];
  cuuint32_t box[3] = {(cuuint32_t)box_inner, (cuuint32_t)box_outer, 1};
  cuuint32_t es[3] = {1, 1, 1};
  CUresult r = enc(m, esz == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims,
                   strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, swz, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    set_error("cuTensorMapEncodeTiled failed (%d): inner=%lld outer=%lld ld=%lld box=%dx%d batch=%d bstride=%lld", (int)r,
              inner, outer, ld, box_inner, box_outer, batch, bstride);
    return ORBIT_ERR_CUDA;
  }
  return ORBIT_OK;
}

template <int A_MN, int B_MN, int BN>
int launch(const CUtensorMap& ma, const CUtensorMap& mb, const GemmArgs& g, cudaStream_t s) {
  using Cf = TcCfg<BN>;
  ORBIT_SMEM_ATTR((gemm_tc_kernel<A_MN, B_MN, BN>), Cf::SMEM_BYTES);
  const int batch = g.batch > 1 ? g.batch : 1;
  const long long tiles = (long long)cdiv(g.M, BM) * cdiv(g.N, BN) * batch;
  const int grid = tiles < num_sms() ? (int)tiles : num_sms();
  ORBIT_CUDA_CHECK(launch_pdl(gemm_tc_kernel<A_MN, B_MN, BN>, dim3(grid), dim3(NTHREADS), Cf::SMEM_BYTES, s, ma, mb, epi::from_gemm(g),
                              g.M, g.N, g.K, batch, g.c_bs, g.bias_bs));
  return ORBIT_OK;
}
template <int BN>
int launch_bn(const CUtensorMap& ma, const CUtensorMap& mb, const GemmArgs& g, bool a_mn, bool b_mn, cudaStream_t s) {
  if (!a_mn && b_mn) return launch<0, 1, BN>(ma, mb, g, s);
  if (!a_mn && !b_mn) return launch<0, 0, BN>(ma, mb, g, s);
  if (a_mn && b_mn) return launch<1, 1, BN>(ma, mb, g, s);
  return launch<1, 0, BN>(ma, mb, g, s);
}
}  // namespace

int gemm_tc2_launch(const CUtensorMap& ma, const CUtensorMap& mb, const CUtensorMap* mc, const CUtensorMap* mx, const GemmArgs& g,
                    bool a_mn, bool b_mn, int sms, cudaStream_t s);   // gemm_tc2.cu

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
  if (g.batch > 1) {
    if (g.resid || g.aux_out || g.aux_in || g.accumulate) return false;
    if ((g.a_bs % 8) || (g.b_bs % 8) || (g.c_bs % 8) || (g.bias && (g.bias_bs % 8))) return false;
  }
  return true;
}

int gemm_tc(const GemmArgs& g, cudaStream_t s) {
  const bool a_mn = !(g.a_cs == 1 && g.a_rs % 8 == 0);
  const bool b_mn = (g.b_cs == 1 && g.b_rs % 8 == 0);
  // CTA-pair kernel (256 x 256 tiles) when the problem has at least one full pair tile; g_force_simt == 2
  // forces the single-CTA kernel (debug / A-B comparison).  Narrow outputs (N <= 128) use 128 x 128 tiles.
  const bool pair = g_force_simt != 2 && g.M >= 256 && g.N >= 256;
  const int bn = pair ? 128 : (g.N <= 128 ? 128 : 256);   // rows of a K-major B box
  CUtensorMap ma, mb;
  if (a_mn) ORBIT_TRY(make_map(&ma, g.A, g.M, g.K, g.a_cs, 64, 64, g.batch, g.a_bs));   // [K rows, M contiguous]
  else      ORBIT_TRY(make_map(&ma, g.A, g.K, g.M, g.a_rs, 64, BM, g.batch, g.a_bs));   // [M rows, K contiguous]
  if (b_mn) ORBIT_TRY(make_map(&mb, g.B, g.N, g.K, g.b_rs, 64, 64, g.batch, g.b_bs));   // [K rows, N contiguous]
  else      ORBIT_TRY(make_map(&mb, g.B, g.K, g.N, g.b_cs, 64, bn, g.batch, g.b_bs));   // [N rows, K contiguous]
  // bf16 outputs without residual (weight gradients, QKV, dO, fc1 with GELU, du with GELU') leave the CTA-pair kernel through TMA stores; g_force_simt == 5
  // keeps the direct row-per-thread stores (A/B comparison)
  CUtensorMap mc, mx;
  const bool store_bf16 = g.out_dtype == ORBIT_BF16 && !g.accumulate &&
                          (g.act == ACT_NONE ? (!g.aux_out && !g.aux_in)
                           : g.act == ACT_GELU ? (g.batch <= 1 && (!g.aux_out || g.aux_dtype == ORBIT_BF16))
                                               : (g.batch <= 1 && g.aux_in != nullptr));
  // fp32 outputs, stored or accumulated (the Hybrid-STOP partial sums and the fp32 dm / da of the backward): TMA store / reduce-add
  const bool store_f32 = g.out_dtype == ORBIT_F32 && !(g.resid && g.accumulate) && g.act == ACT_NONE && !g.aux_out && !g.aux_in &&
                         g.ldc % 4 == 0 && (!g.resid || g.ldr % 4 == 0);
  const bool store_map = pair && g_force_simt != 5 && (store_bf16 || store_f32);
  const bool aux_map = store_map && g.act == ACT_GELU && g.aux_out;
  if (store_map && store_f32) ORBIT_TRY(make_map(&mc, g.C, g.N, g.M, g.ldc, 16, 32, g.batch, g.c_bs, CU_TENSOR_MAP_SWIZZLE_64B, 4));
  else if (store_map) ORBIT_TRY(make_map(&mc, g.C, g.N, g.M, g.ldc, 32, 32, g.batch, g.c_bs, CU_TENSOR_MAP_SWIZZLE_64B));
  if (aux_map) ORBIT_TRY(make_map(&mx, g.aux_out, g.N, g.M, g.ld_aux, 32, 32, 1, 0, CU_TENSOR_MAP_SWIZZLE_64B));
  ProfScope prof(PROF_GEMM, 2.0 * g.M * g.N * g.K * (g.batch > 1 ? g.batch : 1), s);
  if (pair) ORBIT_TRY(gemm_tc2_launch(ma, mb, store_map ? &mc : nullptr, aux_map ? &mx : nullptr, g, a_mn, b_mn, num_sms(), s));
  else if (bn == 128) ORBIT_TRY(launch_bn<128>(ma, mb, g, a_mn, b_mn, s));
  else ORBIT_TRY(launch_bn<256>(ma, mb, g, a_mn, b_mn, s));
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

}  // namespace orbit
