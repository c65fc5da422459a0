// attention_tc5.cu -- flash attention FORWARD on the 5th-gen tensor cores (PAPER.md:88 softmax(QK^T)V, :114).
//
// One CTA = 128 query rows of one (batch, head); key/value tiles of 128 stream through a 2-stage TMA ring.
//   warp 0      : TMA producer (Q once, then K_j / V_j tiles; 128B-swizzled boxes of 64 columns x 128 rows)
//   warp 1      : single-thread tcgen05.mma issuer:  S_j = Q K_j^T  (fp32, TMEM, double buffered)
//                                                     O  += P_j V_j  (fp32, TMEM)
//   warps 2..5  : softmax; thread <-> query row <-> TMEM lane: tcgen05.ld the S row, row max / exp2 / row sum with
//                 no cross-thread traffic, P_j as bf16 into a swizzled K-major shared-memory tile (the A operand
//                 of the PV product), lazy rescale of O in TMEM (only when a row max grows by more than 2^8:
//                 stale maxima keep exp2 below 256, which is exact enough in fp32 accumulators), final O / l.
// S_{j+1} is issued before the softmax of tile j finishes, so the tensor pipe overlaps the exponentials.
// V tiles are consumed as an MN-major B operand straight from their row-major [keys, d] layout.
#include <cuda.h>
#include "common.cuh"
#include "ptx.cuh"

namespace orbit {
namespace {

constexpr int BQ = 128, BKV = 128;
constexpr int NTH = 192;
constexpr float LOG2E = 1.4426950408889634f;
constexpr float LN2 = 0.6931471805599453f;

template <int DH>
struct Cfg {
  static constexpr int NBLK = DH / 64;                  // 64-column blocks per tile row
  static constexpr int TILE = 128 * DH * 2;             // bytes of a [128 x DH] bf16 tile
  static constexpr int P_BYTES = 128 * BKV * 2;         // 32 KB
  static constexpr int SMEM = TILE /*Q*/ + 2 * 2 * TILE /*K,V x 2 stages*/ + P_BYTES + 1024 + 256;
};

template <int DH>
__global__ void __launch_bounds__(NTH, 1)
attn_fwd_tc5_kernel(const __grid_constant__ CUtensorMap tmQKV, AttnArgs a, float sl2) {
  using C = Cfg<DH>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sQ = base, sKV = sQ + C::TILE, sP = sKV + 4 * C::TILE, bar = sP + C::P_BYTES;
  auto sK = [&](int st) { return sKV + st * 2 * C::TILE; };
  auto sV = [&](int st) { return sKV + st * 2 * C::TILE + C::TILE; };
  const uint32_t q_full = bar, kv_full0 = bar + 8, kv_empty0 = bar + 24, s_full0 = bar + 40, s_empty0 = bar + 56,
                 p_full = bar + 72, o_done = bar + 80, tmem_slot = bar + 88;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int bh = blockIdx.y, b = bh / a.heads, h = bh - b * a.heads, N = a.N;
  const int q0 = blockIdx.x * BQ;
  const int ntiles = (N + BKV - 1) / BKV;
  const int row0 = b * N;                                   // first row of this batch in the [B*N, ld] matrix
  const int qc = a.q_off + h * DH, kc = a.k_off + h * DH, vc = a.v_off + h * DH;

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&tmQKV);
    ptx::mbar_init(q_full, 1);
    for (int i = 0; i < 2; i++) {
      ptx::mbar_init(kv_full0 + 8 * i, 1); ptx::mbar_init(kv_empty0 + 8 * i, 1);
      ptx::mbar_init(s_full0 + 8 * i, 1);  ptx::mbar_init(s_empty0 + 8 * i, 4);
    }
    ptx::mbar_init(p_full, 4);
    ptx::mbar_init(o_done, 1);
    ptx::fence_barrier_init();
  }
  if (warp == 1) { ptx::tmem_alloc(tmem_slot, 512); ptx::tmem_relinquish(); }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem) : "r"(tmem_slot));
  const uint32_t tS0 = tmem, tO = tmem + 256;

  if (warp == 0) {
    if (lane == 0) {
      ptx::mbar_expect_tx(q_full, C::TILE);
#pragma unroll
      for (int bk = 0; bk < C::NBLK; bk++) ptx::tma_load_2d(sQ + bk * 16384, &tmQKV, q_full, qc + bk * 64, row0 + q0);
      for (int j = 0; j < ntiles; j++) {
        const int st = j & 1;
        ptx::mbar_wait(kv_empty0 + 8 * st, ((j >> 1) & 1) ^ 1);
        ptx::mbar_expect_tx(kv_full0 + 8 * st, 2 * C::TILE);
#pragma unroll
        for (int bk = 0; bk < C::NBLK; bk++) {
          ptx::tma_load_2d(sK(st) + bk * 16384, &tmQKV, kv_full0 + 8 * st, kc + bk * 64, row0 + j * BKV);
          ptx::tma_load_2d(sV(st) + bk * 16384, &tmQKV, kv_full0 + 8 * st, vc + bk * 64, row0 + j * BKV);
        }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      constexpr uint32_t idesc_s = ptx::make_idesc_bf16(BQ, BKV, 0, 0);     // S = Q K^T: both K-major
      constexpr uint32_t idesc_o = ptx::make_idesc_bf16(BQ, DH, 0, 1);      // O += P V: V is MN-major
      auto issue_s = [&](int j) {
        const int st = j & 1, sb = j & 1;
        ptx::mbar_wait(kv_full0 + 8 * st, (j >> 1) & 1);
        ptx::mbar_wait(s_empty0 + 8 * sb, ((j >> 1) & 1) ^ 1);
        ptx::tc_fence_after();
#pragma unroll
        for (int ks = 0; ks < DH / 16; ks++) {
          const uint32_t off = (ks >> 2) * 16384 + (ks & 3) * 32;
          ptx::mma_f16_ss(tS0 + sb * 128, ptx::make_smem_desc(sQ + off, 16, 1024), ptx::make_smem_desc(sK(st) + off, 16, 1024),
                          idesc_s, ks != 0);
        }
        ptx::mma_commit(s_full0 + 8 * sb);
      };
      ptx::mbar_wait(q_full, 0);
      issue_s(0);
      for (int j = 0; j < ntiles; j++) {
        if (j + 1 < ntiles) issue_s(j + 1);
        ptx::mbar_wait(p_full, j & 1);
        ptx::tc_fence_after();
        const int st = j & 1;
#pragma unroll
        for (int ks = 0; ks < BKV / 16; ks++) {
          const uint32_t aoff = (ks >> 2) * 16384 + (ks & 3) * 32;          // P: K-major, two 64-key blocks
          ptx::mma_f16_ss(tO, ptx::make_smem_desc(sP + aoff, 16, 1024),
                          ptx::make_smem_desc(sV(st) + ks * 2048, 16384, 1024), idesc_o, (j | ks) != 0);
        }
        ptx::mma_commit(kv_empty0 + 8 * st);
        ptx::mma_commit(o_done);
      }
    }
  } else {
    // ===================== softmax / correction / epilogue =====================
    const int quarter = warp & 3;
    const int r = quarter * 32 + lane;                       // query row within the tile = TMEM lane
    const uint32_t lane_off = (uint32_t)(quarter * 32) << 16;
    float m_used = -INFINITY, l = 0.f;
    for (int j = 0; j < ntiles; j++) {
      const int sb = j & 1;
      ptx::mbar_wait(s_full0 + 8 * sb, (j >> 1) & 1);
      ptx::tc_fence_after();
      uint32_t s[128];
#pragma unroll
      for (int c = 0; c < 4; c++) ptx::tmem_ld_32x32(tS0 + sb * 128 + c * 32 + lane_off, s + c * 32);
      ptx::tmem_ld_wait();
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(s_empty0 + 8 * sb);   // S buffer may be overwritten by S_{j+2}
      float mx = -INFINITY;
      if ((j + 1) * BKV > N) {                               // last, ragged tile: mask keys >= N
#pragma unroll
        for (int c = 0; c < 128; c++) {
          float v = (j * BKV + c < N) ? __uint_as_float(s[c]) : -INFINITY;
          s[c] = __float_as_uint(v);
          mx = fmaxf(mx, v);
        }
      } else {
#pragma unroll
        for (int c = 0; c < 128; c++) mx = fmaxf(mx, __uint_as_float(s[c]));
      }
      const float m_tile = mx * sl2;
      // P buffer and O are free / final once PV_{j-1} has completed
      if (j > 0) { ptx::mbar_wait(o_done, (j - 1) & 1); ptx::tc_fence_after(); }
      float m_new = m_used;
      bool need = false;
      if (j == 0) m_new = m_tile;
      else if (m_tile > m_used + 8.f) { m_new = m_tile; need = true; }
      if (__any_sync(0xffffffffu, need)) {                    // lazy rescale of the O row in TMEM
        const float f = exp2f(m_used - m_new);
        l *= f;
#pragma unroll
        for (int c = 0; c < DH / 32; c++) {
          uint32_t o[32];
          ptx::tmem_ld_32x32(tO + c * 32 + lane_off, o);
          ptx::tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 32; i++) o[i] = __float_as_uint(__uint_as_float(o[i]) * f);
          ptx::tmem_st_32x32(tO + c * 32 + lane_off, o);
        }
        ptx::tmem_st_wait();
      }
      m_used = m_new;
      float sum = 0.f;
#pragma unroll
      for (int c = 0; c < 16; c++) {                          // 8 keys = one 16-byte chunk of the P row
        uint32_t pk[4];
#pragma unroll
        for (int i = 0; i < 4; i++) {
          const float p0 = exp2f(__uint_as_float(s[c * 8 + 2 * i]) * sl2 - m_used);
          const float p1 = exp2f(__uint_as_float(s[c * 8 + 2 * i + 1]) * sl2 - m_used);
          sum += p0 + p1;
          __nv_bfloat162 v = __floats2bfloat162_rn(p0, p1);
          pk[i] = *reinterpret_cast<uint32_t*>(&v);
        }
        const uint32_t addr = sP + (c >> 3) * 16384 + r * 128 + (((c & 7) ^ (r & 7)) << 4);
        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(pk[0]), "r"(pk[1]), "r"(pk[2]), "r"(pk[3]) : "memory");
      }
      l += sum;
      ptx::fence_proxy_async();                               // generic-proxy smem writes -> visible to the MMA
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(p_full);
    }
    // ---- epilogue: O / l -> bf16 -> global; logsumexp
    ptx::mbar_wait(o_done, (ntiles - 1) & 1);
    ptx::tc_fence_after();
    const int qrow = q0 + r;
    const float inv = 1.f / l;
    bf16* orow = (bf16*)a.O + (size_t)(row0 + qrow) * a.ldo + h * DH;
#pragma unroll
    for (int c = 0; c < DH / 32; c++) {
      uint32_t o[32];
      ptx::tmem_ld_32x32(tO + c * 32 + lane_off, o);
      ptx::tmem_ld_wait();
      if (qrow < N) {
#pragma unroll
        for (int g8 = 0; g8 < 4; g8++) {
          uint4 v;
          uint32_t* pv = reinterpret_cast<uint32_t*>(&v);
#pragma unroll
          for (int i = 0; i < 4; i++) {
            __nv_bfloat162 t2 = __floats2bfloat162_rn(__uint_as_float(o[g8 * 8 + 2 * i]) * inv, __uint_as_float(o[g8 * 8 + 2 * i + 1]) * inv);
            pv[i] = *reinterpret_cast<uint32_t*>(&t2);
          }
          *reinterpret_cast<uint4*>(orow + c * 32 + g8 * 8) = v;
        }
      }
    }
    if (qrow < N) a.lse[(size_t)bh * N + qrow] = (m_used + log2f(l)) * LN2;
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 1) { ptx::tc_fence_after(); ptx::tmem_dealloc(tmem, 512); }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn get_encode5() {
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

template <int DH>
int launch_fwd5(const AttnArgs& a, cudaStream_t s) {
  EncodeTiledFn enc = get_encode5();
  if (!enc) { set_error("cuTensorMapEncodeTiled entry point not found"); return ORBIT_ERR_CUDA; }
  CUtensorMap tm;
  cuuint64_t dims[2] = {(cuuint64_t)a.ld, (cuuint64_t)a.B * a.N};
  cuuint64_t strides[1] = {(cuuint64_t)a.ld * 2};
  cuuint32_t box[2] = {64, 128};
  cuuint32_t es[2] = {1, 1};
  CUresult r = enc(&tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(a.qkv), dims, strides, box, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { set_error("attention: cuTensorMapEncodeTiled failed (%d)", (int)r); return ORBIT_ERR_CUDA; }
  static bool set = false;
  if (!set) {
    ORBIT_CUDA_CHECK(cudaFuncSetAttribute((const void*)attn_fwd_tc5_kernel<DH>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg<DH>::SMEM));
    set = true;
  }
  dim3 grid(cdiv(a.N, BQ), a.B * a.heads);
  attn_fwd_tc5_kernel<DH><<<grid, NTH, Cfg<DH>::SMEM, s>>>(tm, a, LOG2E / sqrtf((float)DH));
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}
}  // namespace

bool attention_tc5_supported(const AttnArgs& a) {
  if (a.dtype != ORBIT_BF16 || (a.dh != 64 && a.dh != 128)) return false;
  auto al16 = [](const void* p) { return (((uintptr_t)p) & 15) == 0; };
  if (a.ld % 8 || a.ldo % 8 || a.q_off % 8 || a.k_off % 8 || a.v_off % 8) return false;
  if (!al16(a.qkv) || !al16(a.O)) return false;
  return a.N >= 128;
}
int attention_fwd_tc5(const AttnArgs& a, cudaStream_t s) {
  return a.dh == 64 ? launch_fwd5<64>(a, s) : launch_fwd5<128>(a, s);
}

}  // namespace orbit
