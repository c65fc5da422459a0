// attention_tc5.cu -- flash attention FORWARD on the 5th-gen tensor cores (PAPER.md:88 softmax(QK^T)V, :114).
//
// One CTA = 128 query rows of one (batch, head); key/value tiles of 128 stream through a 2-stage TMA ring.
//   warp 0      : TMA producer (Q once, then K_j / V_j tiles; 128B-swizzled boxes of 64 columns x 128 rows)
//   warp 1      : single-thread tcgen05.mma issuer:  S_j = Q K_j^T  (fp32, TMEM, double buffered)
//                                                     O  += P_j V_j  (fp32, TMEM)
//   warps 2..9  : softmax; two warps share a TMEM lane quarter (thread <-> query row <-> TMEM lane) and split the
//                 tile's 128 key columns: tcgen05.ld of the S half-row, row max (agreed between the pair through
//                 shared memory as ceil(max), a float), exp2 / row sum, P_j as packed bf16 pairs written with tcgen05.st
//                 over the S columns just read (the A operand of the PV product, read from TENSOR MEMORY); the two key
//                 halves are published separately (PV_j starts on the first half while the second is still being written),
//                 lazy rescale of O in TMEM (only when a row max grows by more than 2^8: stale maxima keep exp2
//                 below 256, which is exact enough in fp32 accumulators), final O / l.
// clock64 stamps (C5, one CTA per SM, 16 tiles): ~2200 cycles per tile against ~1050 of MMA; the softmax warps are
// the critical path: 128 MUFU.EX2 per row and tile = ~1024 cycles of the sub-partition's quarter-rate unit, plus the
// serial tcgen05.ld / fence.proxy.async / barrier latencies of a tile.  Tried and measured no faster: a max-only warp
// running one tile ahead of an exp-only warp (291 us vs 284), P packed by truncation instead of cvt (311 us).
// Round-2 probes (A/B build, C4, per-launch CUDA events) of the version that kept P in shared memory: with the exponentials removed
// (ORBIT_PROBE_NOEXP) 54.0 -> 54.7 us, with half of the tcgen05.ld traffic removed (ORBIT_PROBE_HALFLD) 52.0 us, with the K / V
// tiles TMA-multicast across a cluster of two query tiles (half the L2 -> SM traffic) 54 -> 58 us: none of MUFU, TMEM reads or L2
// bandwidth bounded it.  The timeline probe (ORBIT_PROBE_TIMELINE: cycles per mbarrier wait of each agent) then showed the
// MMA-issuing thread busy ~1850 of 2350 cycles per tile OUTSIDE its waits while the softmax warps waited 550 cycles per tile for
// S: the tensor pipe was starved by shared-memory bandwidth (Cfg above).  With P in tensor memory: 2090 cycles per tile, MMA thread
// 1540 busy, softmax wait for S 240; same-box A/B of the kernel: 53.3 -> 48.0 us at C4 (644 -> 715 TFLOP/s), 370 -> 344 us at C5,
// 195 -> 180 us at C3.  Both agents are now about equally loaded (softmax ~1850 busy cycles per tile).
// Four softmax warps per lane quarter (32 key columns each, a four-way row-max exchange) measured SLOWER: 175 vs 166 us at C3.
// S_{j+1} is issued before the softmax of tile j finishes, so the tensor pipe overlaps the exponentials.
// V tiles are consumed as an MN-major B operand straight from their row-major [keys, d] layout.
#include <cuda.h>
#include <atomic>
#include "common.cuh"
#include "ptx.cuh"

namespace orbit {
namespace {

constexpr int BQ = 128;

// ---- timeline probe of the forward kernel (A/B build with ORBIT_NVCC_EXTRA=-DORBIT_PROBE_TIMELINE only) ---------------------
// Cycles the three agents of CTA (0, 0) spend in each mbarrier wait, summed over its tiles, read back with
// orbit_debug_read_probe (csrc/orbit_debug.h).  Slots: 0 producer k_empty, 1 producer v_empty, 2 mma k_full, 3 mma s_empty,
// 4 mma v_full, 5 mma p_full[0], 6 mma p_full[1], 7 softmax s_full, 8 softmax o_done (rescale), 9 softmax p_free, 10 softmax
// loop total, 11 mma loop total, 12 tiles, 13 producer loop total, 14 softmax pair barrier, 15 softmax final o_done wait.
#ifdef ORBIT_PROBE_TIMELINE
__device__ unsigned long long g_attn_probe[32];
#define PROBE_DECL long long pw_[16] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}; const bool pon_ = blockIdx.x == 0 && blockIdx.y == 0
#define PWAIT(slot, bar, par) do { long long t0_ = clock64(); ptx::mbar_wait(bar, par); pw_[slot] += clock64() - t0_; } while (0)
#define PTIME(slot, stmt) do { long long t0_ = clock64(); stmt; pw_[slot] += clock64() - t0_; } while (0)
#define PFLUSH(a, b) do { if (pon_) for (int i_ = a; i_ <= b; i_++) atomicAdd(&g_attn_probe[i_], (unsigned long long)pw_[i_]); } while (0)
#define PROBE_T0 const long long pt0_ = clock64()
#define PSINCE(slot) pw_[slot] = clock64() - pt0_
#define PSET(slot, v) pw_[slot] = (v)
#else
#define PROBE_T0
#define PSINCE(slot)
#define PSET(slot, v)
#define PROBE_DECL
#define PWAIT(slot, bar, par) ptx::mbar_wait(bar, par)
#define PTIME(slot, stmt) stmt
#define PFLUSH(a, b)
#endif
constexpr int NTH = 320;   // forward: warp 0 TMA, warp 1 MMA issuer, warps 2..9 softmax (two per TMEM lane quarter, 64 key columns each)
constexpr float LOG2E = 1.4426950408889634f;
constexpr float LN2 = 0.6931471805599453f;

// one MUFU.EX2 (ex2.approx.ftz): exp2f() adds a range fix-up of ~5 instructions per element, which made the softmax
// warps issue-bound; the arguments here are <= 8 and results below 2^-126 may flush to zero
__device__ __forceinline__ float fast_ex2(float x) {
#ifdef ORBIT_PROBE_NOEXP       // measurement probe (A/B build only, ORBIT_NVCC_EXTRA): no MUFU work, wrong results
  return x * 0.001f;
#else
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
#endif
}

// descriptor of the same tile `bytes` further on: the start-address field (bits [0,14), in 16-byte units) never carries
// out for shared-memory addresses, so this is one 64-bit add instead of rebuilding the descriptor (the single MMA-issuing
// thread is latency-bound: ~13 dependent uniform-datapath instructions per tcgen05.mma otherwise)
__device__ __forceinline__ uint64_t desc_adv(uint64_t d, uint32_t bytes) { return d + (uint64_t)(bytes >> 4); }

__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

template <int DH>
struct Cfg {
  // head widths up to 128 stream key / value tiles of 128 rows; 192 and 256 (the paper's 113B / 1B / 10B shapes,
  // PAPER.md:140) stream 64-row tiles so that Q + the K / V rings + P still fit 227 KB and S (double buffered) + O fit
  // the 512 TMEM columns (2 * 64 + 256)
  static constexpr int BKV = DH <= 128 ? 128 : 64;
  static constexpr int NBLK = DH / 64;                  // 64-column blocks per tile row
  static constexpr int QBLK = 128 * 128;                // bytes of one 64-column block of the Q tile (128 rows)
  static constexpr int KBLK = BKV * 128;                // ... of a K / V tile (BKV rows)
  static constexpr int QTILE = 128 * DH * 2;            // bytes of the [128 x DH] bf16 query tile
  static constexpr int TILE = BKV * DH * 2;             // bytes of a [BKV x DH] bf16 key / value tile
  // P never touches shared memory: the softmax threads write it (packed bf16 pairs, tcgen05.st) over the S columns they have
  // just read and O += P V is a tcgen05.mma with the A operand in tensor memory.  The timeline probe (below) showed the
  // MMA-issuing thread busy ~1850 of 2350 cycles per tile with the softmax warps WAITING for S: the tensor pipe was starved by
  // shared-memory bandwidth -- per 128-key tile the MMAs read 128 KB of operands (8 KB per 64-cycle instruction = the whole
  // 128 B/clk of the SM), the softmax warps wrote 32 KB of P and TMA 64 KB of K / V: 224 KB = 1750 cycles against 1024 cycles
  // of MMA.  Without the P tile it is 160 KB.  S is then free only after PV has read P, hence THREE S buffers (S_{j+1} is
  // issued before PV_j, S_{j+2} must not wait for it): 3 BKV + DH <= 512 TMEM columns.
  static constexpr int NSB = 3;
  // K and V stream through separate rings: a K stage is free as soon as S_j = Q K_j^T has been computed, a V stage
  // only after O += P_j V_j
  static constexpr int KST = DH == 256 ? 2 : 3, VST = DH == 256 ? 2 : 3;
  static constexpr int SMEM = QTILE + (KST + VST) * TILE + 256 /*alignment slack, see the kernel*/ + 256 + 2048 /*row-max exchange*/;
  static_assert(SMEM <= 227 * 1024, "attention forward: shared memory budget");
  static_assert(NSB * BKV + DH <= 512, "attention forward: TMEM budget");
};

template <int DH>
__global__ void __launch_bounds__(NTH, 1)
attn_fwd_tc5_kernel(const __grid_constant__ CUtensorMap tmQKV, const __grid_constant__ CUtensorMap tmKV, AttnArgs a, float sl2) {
  using C = Cfg<DH>;
  // the 128B-swizzled tiles need 1024-byte aligned shared addresses: the alignment is requested on the declaration
  // (dynamic shared memory starts at the window's 1 KB-aligned base when the kernel has no static shared memory) and
  // the budget keeps only 256 bytes of slack, so a base that is further off fails loudly instead of overrunning
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  if (base - ptx::smem_u32(smem_raw) > 256u) __trap();
  constexpr int KST = C::KST, VST = C::VST, BKV = C::BKV;
  constexpr int NSB = C::NSB;
  const uint32_t sQ = base, sK0 = sQ + C::QTILE, sV0 = sK0 + KST * C::TILE, bar = sV0 + VST * C::TILE;
  auto sK = [&](int st) { return sK0 + st * C::TILE; };
  auto sV = [&](int st) { return sV0 + st * C::TILE; };
  const uint32_t q_full = bar, k_full0 = bar + 8, k_empty0 = k_full0 + 8 * KST, v_full0 = k_empty0 + 8 * KST,
                 v_empty0 = v_full0 + 8 * VST, s_full0 = v_empty0 + 8 * VST, s_empty0 = s_full0 + 8 * NSB, p_full0 = s_empty0 + 8 * NSB,
                 o_done = p_full0 + 16, tmem_slot = o_done + 8, xmax = bar + 256;   // xmax: fp32 [2 parity][2 halves][128 rows]
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int bh = blockIdx.y, b = bh / a.heads, h = bh - b * a.heads, N = a.N;
  const int q0 = blockIdx.x * BQ;
  const int ntiles = (N + BKV - 1) / BKV;
  const int row0 = b * N;                                   // first row of this batch in the [B*N, ld] matrix
  const int qc = a.q_off + h * DH, kc = a.k_off + h * DH, vc = a.v_off + h * DH;

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&tmQKV); ptx::prefetch_tmap(&tmKV);
    ptx::mbar_init(q_full, 1);
    for (int i = 0; i < KST; i++) { ptx::mbar_init(k_full0 + 8 * i, 1); ptx::mbar_init(k_empty0 + 8 * i, 1); }
    for (int i = 0; i < VST; i++) { ptx::mbar_init(v_full0 + 8 * i, 1); ptx::mbar_init(v_empty0 + 8 * i, 1); }
    for (int i = 0; i < NSB; i++) { ptx::mbar_init(s_full0 + 8 * i, 1);  ptx::mbar_init(s_empty0 + 8 * i, 1); }   // empty: commit of the PV that read P
    for (int i = 0; i < 2; i++) ptx::mbar_init(p_full0 + 8 * i, 4);
    ptx::mbar_init(o_done, 1);
    ptx::fence_barrier_init();
  }
  if (warp == 1) { ptx::tmem_alloc(tmem_slot, 512); ptx::tmem_relinquish(); }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem) : "r"(tmem_slot));
  pdl_wait();                                    // on-chip prologue done; first global access is below
  pdl_trigger();
  const uint32_t tS0 = tmem, tO = tmem + NSB * BKV;

  PROBE_DECL;
  if (warp == 0) {
    if (lane == 0) {
      ptx::mbar_expect_tx(q_full, C::QTILE);
#pragma unroll
      for (int bk = 0; bk < C::NBLK; bk++) ptx::tma_load_2d(sQ + bk * C::QBLK, &tmQKV, q_full, qc + bk * 64, row0 + q0);
      auto load_k = [&](int j) {
        const int st = j % KST;
        PWAIT(0, k_empty0 + 8 * st, ((j / KST) & 1) ^ 1);
        ptx::mbar_expect_tx(k_full0 + 8 * st, C::TILE);
#pragma unroll
        for (int bk = 0; bk < C::NBLK; bk++) ptx::tma_load_2d(sK(st) + bk * C::KBLK, &tmKV, k_full0 + 8 * st, kc + bk * 64, row0 + j * BKV);
      };
      load_k(0);
      for (int j = 0; j < ntiles; j++) {                      // K runs one tile ahead of V
        if (j + 1 < ntiles) load_k(j + 1);
        const int st = j % VST;
        PWAIT(1, v_empty0 + 8 * st, ((j / VST) & 1) ^ 1);
        ptx::mbar_expect_tx(v_full0 + 8 * st, C::TILE);
#pragma unroll
        for (int bk = 0; bk < C::NBLK; bk++) ptx::tma_load_2d(sV(st) + bk * C::KBLK, &tmKV, v_full0 + 8 * st, vc + bk * 64, row0 + j * BKV);
      }
      PFLUSH(0, 1);
    }
  } else if (warp == 1) {
    if (lane == 0) {
      constexpr uint32_t idesc_s = ptx::make_idesc_bf16(BQ, BKV, 0, 0);     // S = Q K^T: both K-major
      constexpr uint32_t idesc_o = ptx::make_idesc_bf16(BQ, DH, 0, 1);      // O += P V: V is MN-major
      const uint64_t dQ0 = ptx::make_smem_desc(sQ, 16, 1024);
      auto issue_s = [&](int j) {
        const int st = j % KST, sb = j % NSB;
        PWAIT(2, k_full0 + 8 * st, (j / KST) & 1);
        PWAIT(3, s_empty0 + 8 * sb, ((j / NSB) & 1) ^ 1);
        ptx::tc_fence_after();
        const uint64_t dK0 = ptx::make_smem_desc(sK(st), 16, 1024);
#pragma unroll
        for (int ks = 0; ks < DH / 16; ks++) {
          const uint32_t qoff = (ks >> 2) * C::QBLK + (ks & 3) * 32, koff = (ks >> 2) * C::KBLK + (ks & 3) * 32;
          ptx::mma_f16_ss(tS0 + sb * BKV, desc_adv(dQ0, qoff), desc_adv(dK0, koff), idesc_s, ks != 0);
        }
        ptx::mma_commit(k_empty0 + 8 * st);          // K stage free once these MMAs have read it
        ptx::mma_commit(s_full0 + 8 * sb);
      };
      ptx::mbar_wait(q_full, 0);
#ifdef ORBIT_PROBE_TIMELINE
      const long long pt_m0 = clock64();
#endif
      issue_s(0);
      for (int j = 0; j < ntiles; j++) {
        if (j + 1 < ntiles) issue_s(j + 1);
        const int st = j % VST;
        PWAIT(4, v_full0 + 8 * st, (j / VST) & 1);
        const uint64_t dV0 = ptx::make_smem_desc(sV(st), C::KBLK, 1024);
        const uint32_t tP = tS0 + (j % NSB) * BKV;            // P_j lives in the columns of S_j
#pragma unroll
        for (int hh = 0; hh < 2; hh++) {                      // the two key halves of P are written by different warps
          PWAIT(5 + hh, p_full0 + 8 * hh, j & 1);
          ptx::tc_fence_after();
#pragma unroll
          for (int k4 = 0; k4 < BKV / 32; k4++) {             // k-step (16 keys) k4 of half hh: 8 columns of packed bf16 pairs
            const int ks = hh * (BKV / 32) + k4;
            ptx::mma_f16_ts(tO, tP + hh * (BKV / 2) + k4 * 8, desc_adv(dV0, ks * 2048), idesc_o, (j | ks) != 0);
          }
        }
        ptx::mma_commit(s_empty0 + 8 * (j % NSB));            // S_j / P_j columns may be overwritten by S_{j+3}
        ptx::mma_commit(v_empty0 + 8 * st);
        ptx::mma_commit(o_done);
      }
#ifdef ORBIT_PROBE_TIMELINE
      pw_[11] = clock64() - pt_m0;
      PFLUSH(2, 6); PFLUSH(11, 11);
#endif
    }
  } else {
    // ===================== softmax / correction / epilogue =====================
    // Two warps share a TMEM lane quarter (32 query rows) and split the tile's 128 key columns: the exponentials of a
    // row are issued from two schedulers' worth of warps instead of one (with 4 softmax warps the single warp per SM
    // sub-partition could not hide its own MUFU / TMEM latencies: ~2900 cycles per tile against ~1050 of MMA).
    // The pair agrees on the row maximum through shared memory as ceil(max): any common reference >= the true
    // maximum is exact for softmax (it cancels in P / l); exchanged as fp32 so runaway logits (the regime QK-LayerNorm
    // targets) do not saturate the reference.
    const int quarter = warp & 3, half = (warp - 2) >> 2;   // warps 2..9
    const int r = quarter * 32 + lane;                       // query row within the tile = TMEM lane
    const uint32_t lane_off = (uint32_t)(quarter * 32) << 16;
    const int pair_bar = 1 + quarter;                        // named barrier of the two warps of this quarter
    float m_used = -INFINITY, l = 0.f;                       // l: this thread's half of the row sum
#ifdef ORBIT_PROBE_TIMELINE
    const long long pt_sm0 = clock64();
#endif
    for (int j = 0; j < ntiles; j++) {
      const int sb = j % NSB;
      PWAIT(7, s_full0 + 8 * sb, (j / NSB) & 1);
      ptx::tc_fence_after();
      constexpr int HC = BKV / 2;                             // key columns of this warp
      uint32_t s[HC];
#pragma unroll
#ifdef ORBIT_PROBE_HALFLD      // measurement probe (A/B build only): half of the tcgen05.ld traffic, wrong results
      ptx::tmem_ld_32x32(tS0 + sb * BKV + half * HC + lane_off, s);
      if (HC == 64) { ptx::tmem_ld_wait(); for (int c = 0; c < 32; c++) s[32 + c] = s[c]; }
#else
      for (int c = 0; c < HC / 32; c++) ptx::tmem_ld_32x32(tS0 + sb * BKV + half * HC + c * 32 + lane_off, s + c * 32);
#endif
      ptx::tmem_ld_wait();
      float mx = -INFINITY;
      if ((j + 1) * BKV > N) {                               // last, ragged tile: mask keys >= N
#pragma unroll
        for (int c = 0; c < HC; c++) {
          float v = (j * BKV + half * HC + c < N) ? __uint_as_float(s[c]) : -INFINITY;
          s[c] = __float_as_uint(v);
          mx = fmaxf(mx, v);
        }
      } else {
#pragma unroll
        for (int c = 0; c < HC; c++) mx = fmaxf(mx, __uint_as_float(s[c]));
      }
      const float mi = ceilf(mx * sl2);                                  // -inf when this half of a ragged tile is fully masked
      const uint32_t xm = xmax + (uint32_t)((j & 1) * 256 + r) * 4;     // [parity][half][row] fp32 (no range limit on the logits)
      asm volatile("st.shared.f32 [%0], %1;" ::"r"(xm + half * 512), "f"(mi) : "memory");
      PTIME(14, named_bar_sync(pair_bar, 64));
      float mo;
      asm volatile("ld.shared.f32 %0, [%1];" : "=f"(mo) : "r"(xm + (half ^ 1) * 512) : "memory");
      const float m_tile = fmaxf(mi, mo);
      float m_new = m_used;
      bool need = false;
      if (j == 0) m_new = m_tile;
      else if (m_tile > m_used + 8.f) { m_new = m_tile; need = true; }
      if (__any_sync(0xffffffffu, need)) {                    // lazy rescale: this thread's half of the O row in TMEM
        // O is final only once PV_{j-1} has completed, and PV_j (which starts as soon as the FIRST half of P_j is
        // published) must not begin before BOTH warps of the pair have rescaled: pair barrier after the rescale.
        // The partner takes the same branch: it sees the same maxima.
        PWAIT(8, o_done, (j - 1) & 1);
        ptx::tc_fence_after();
        const float f = exp2f(m_used - m_new);
        l *= f;
#pragma unroll
        for (int c = 0; c < DH / 64; c++) {
          uint32_t o[32];
          ptx::tmem_ld_32x32(tO + half * (DH / 2) + c * 32 + lane_off, o);
          ptx::tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 32; i++) o[i] = __float_as_uint(__uint_as_float(o[i]) * f);
          ptx::tmem_st_32x32(tO + half * (DH / 2) + c * 32 + lane_off, o);
        }
        ptx::tmem_st_wait();
        ptx::tc_fence_before();
        named_bar_sync(pair_bar, 64);
      }
      m_used = m_new;
      float sum = 0.f;
      // P_j: packed bf16 pairs over the first half of this thread's own S columns (k-step of 16 keys = 8 columns); nobody else
      // reads or writes this lane's columns [half HC, half HC + HC) of the buffer until PV_j has consumed them
      const uint32_t tPh = tS0 + sb * BKV + half * HC + lane_off;
#pragma unroll
      for (int c = 0; c < HC / 16; c++) {
        uint32_t pk[8];
#pragma unroll
        for (int i = 0; i < 8; i++) {
          const float p0 = fast_ex2(__uint_as_float(s[c * 16 + 2 * i]) * sl2 - m_used);
          const float p1 = fast_ex2(__uint_as_float(s[c * 16 + 2 * i + 1]) * sl2 - m_used);
          sum += p0 + p1;
          __nv_bfloat162 v = __floats2bfloat162_rn(p0, p1);
          pk[i] = *reinterpret_cast<uint32_t*>(&v);
        }
        ptx::tmem_st_32x8(tPh + c * 8, pk);
      }
      l += sum;
      ptx::tmem_st_wait();
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(p_full0 + 8 * half);
    }
    // ---- epilogue: O / l -> bf16 -> global; logsumexp.  All MMAs and TMA loads are done: the pair adds its half sums through K stage 0
    PWAIT(15, o_done, (ntiles - 1) & 1);
#ifdef ORBIT_PROBE_TIMELINE
    pw_[10] = clock64() - pt_sm0; pw_[12] = ntiles;
    if (warp == 2 && lane == 0) { PFLUSH(7, 10); PFLUSH(12, 12); PFLUSH(14, 15); }
#endif
    ptx::tc_fence_after();
    asm volatile("st.shared.f32 [%0], %1;" ::"r"(sK0 + (uint32_t)(half * 128 + r) * 4), "f"(l) : "memory");
    named_bar_sync(pair_bar, 64);
    float lo;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(lo) : "r"(sK0 + (uint32_t)((half ^ 1) * 128 + r) * 4) : "memory");
    l += lo;
    const int qrow = q0 + r;
    const float inv = 1.f / l;
    bf16* orow = (bf16*)a.O + (size_t)(row0 + qrow) * a.ldo + h * DH + half * (DH / 2);
#pragma unroll
    for (int c = 0; c < DH / 64; c++) {
      uint32_t o[32];
      ptx::tmem_ld_32x32(tO + half * (DH / 2) + c * 32 + lane_off, o);
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
    if (half == 0 && qrow < N) a.lse[(size_t)bh * N + qrow] = (m_used + log2f(l)) * LN2;
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 1) { ptx::tc_fence_after(); ptx::tmem_dealloc(tmem, 512); }
}

// =====================================================================================================
// Backward on tcgen05 (split as in attention_tc.cu: a dK/dV kernel with rows = keys and a dQ kernel with rows =
// queries; 7 tile products, no atomics).  The stationary operand (128 rows) stays in shared memory; the other
// index streams in tiles of 64 rows through a 2-stage TMA ring.  S^T / dP^T (resp. S / dP) accumulate in TMEM
// (double buffered, 64 columns each); the 128 "softmax" threads (thread <-> TMEM lane <-> row) turn them into
// P^T and dS^T (resp. dS) as bf16 K-major operand tiles in shared memory; the gradient accumulators live in TMEM.
// A streamed [64 x d_h] tile is used twice from the same bytes: as a K-major B operand (contraction over d_h)
// and as an MN-major B operand (contraction over its 64 rows).
// =====================================================================================================
// warp 0 TMA, warp 1 gradient MMAs, warps 2..17 softmax, warp 18 dP MMAs, warp 19 S MMAs.  The 16 softmax warps form two
// groups of 8 (two per TMEM lane quarter, BT / 2 columns each); group g owns the tiles of parity g, i.e. the S / dP
// accumulator buffer g and the operand-tile buffer g.  A tile's softmax is a serial chain (tcgen05.ld latency -> exponentials
// -> shared-memory stores -> proxy fence -> barrier) of about a tile's MMA time; with one group that chain sat between the
// S^T / dP^T products and the gradient products of every tile (tensor pipe 47-53 % active, profiles/r1_full_ncu.md); with
// two groups the chains of consecutive tiles overlap.  The backward has no running maximum (logsumexp is saved), so tiles
// are independent and the groups never exchange anything.
constexpr int NTHB = 640;
// TS_DKV: in the dK / dV kernel the operand tiles P^T and dS^T stay in TENSOR MEMORY (tcgen05.mma with the A operand in
// TMEM), written by the softmax threads with tcgen05.st over the S^T / dP^T columns they have just read (16 fp32 columns
// -> 8 columns of packed bf16 pairs, in place).  The kernels were shared-memory-bandwidth bound: per 64-query tile the
// MMAs read 160 KB of operands from shared memory, the softmax warps wrote 32 KB of operand tiles and TMA 32 KB of Q / dO,
// i.e. 224 KB = 1750 cycles at 128 B/clk against 1024 cycles of MMA; without the operand tiles (written and read once
// each) it is 160 KB.  A buffer of S^T / dP^T is then free only once the gradient MMAs that read it have completed.
constexpr bool TS_DKV = true;
// the same for dS in the dQ kernel measured no gain, with two S / dP buffers (C5: attention backward 417 vs 423-429 TFLOP/s of
// model FLOPs) and with three (ncu, same box: 312.4 vs 312.5 us at C5, 207.6 vs 207.7 us at C3 / C4).
constexpr bool TS_DQ = false;
// Q / dO as tensor-memory A operands of the S / dP products (dQ kernel): SLOWER, 339 us vs 312 us at C5 (368 us with dS in
// tensor memory as well).  What the round-2 probes of this kernel say (A/B builds, C5, ncu per-launch times):
//   timeline (ORBIT_PROBE_TIMELINE): 1565 cycles per 64-key tile; the S-issuing thread waits 150 of them on barriers and sits in
//   tcgen05.mma issue for the rest (back-pressure of the tensor pipe), the softmax warps wait 640 cycles per tile for S / dP, the
//   dQ issuer 570 for dS: the MMAs themselves take ~1400 cycles per tile against a floor of 768 (3 products of 128 x 64 x 128);
//   no softmax work at all (ORBIT_PROBE_DQ_NOSM) 313 -> 282 us; no exponentials (.._NOEXP) 317 us; half the tcgen05.ld (.._HALFLD)
//   319 us; one of eight k-steps of S / dP (.._NOS) 252 us; no dQ product (.._NOG) 280 us.
// A model that fits all of these: one tcgen05.mma of M = 128, K = 16 costs max(N / 2, shared-memory operand bytes / 128 B/clk,
// tensor-memory A bytes / 64 B/clk) cycles.  The A operand is 4 KB either way, so an SS product needs N >= 128 to reach the
// floor (N = 64: 6 KB = 48 cycles against 32, i.e. 67 %) and a TS product costs 64 cycles whatever N is: equal to SS at
// N = 128 (P V, dV, dK, dQ: no gain, no loss, less shared-memory traffic), slower at N = 64 (S, dP here).  Per tile: S 384 +
// dP 384 + dQ 256 = 1024 cycles of operand reads, + 256 of TMA writes of K / V + 128 of dS writes ~ 1400.  The N = 64 of the
// S / dP products is set by tensor memory (2 x 2 x 64 S / dP columns + 128 dQ columns; 128-key tiles would leave one buffer),
// so this kernel stays at ~55 % of its tensor floor; the remedy is a CTA pair per 256 queries (cta_group::2 halves the B
// operand and the K / V stream per SM: 40 cycles per S / dP instruction instead of 48) -- not built, see DESIGN.md §13.
constexpr bool TSA_DQ = false;

template <int DH>
struct CfgB {
  // streamed tile rows: 64 up to d_h = 128; 32 for d_h = 192 / 256 (PAPER.md:140 shapes) so that S / dP (double
  // buffered, 4 BT columns) + the gradient accumulators fit the 512 TMEM columns and two stationary [128 x DH] tiles +
  // the ring fit 227 KB.  d_h = 256: dK + dV alone would fill TMEM, so the dK/dV kernel computes one 128-column slice
  // of both per CTA (grid z = NSPLIT; S^T and dP^T are recomputed per slice: 6 tile products instead of 4).
  static constexpr int BT = DH <= 128 ? 64 : 32;
  static constexpr int NBLK = DH / 64;
  static constexpr int BBLK = 128 * 128;          // bytes of one 64-column block of a stationary [128 x DH] tile
  static constexpr int SBLK = BT * 128;           // ... of a streamed [BT x DH] tile
  static constexpr int BIG = 128 * DH * 2;        // stationary [128 x DH] tile
  static constexpr int SMALL = BT * DH * 2;       // streamed [BT x DH] tile
  static constexpr int PT = 128 * BT * 2;         // [128 x BT] bf16 operand tile written by the softmax threads (rows of 2 BT bytes:
                                                  // 128B swizzle at BT = 64, 64B swizzle at BT = 32)
  static constexpr int NSPLIT = DH == 256 ? 2 : 1;
  static constexpr int DHO = DH / NSPLIT;         // dK / dV columns per CTA
  // stages of the streamed (two-tile) ring: hide the TMA round trip.  The operand tiles written by the softmax warps
  // (P^T, dS^T resp. dS) are double buffered so that tile j+1 is written while the MMAs of tile j still read tile j.
  static constexpr int NST_DKV = DH == 256 ? 2 : 3, NST_DQ = DH == 256 ? 2 : 4;
  // + statistics [2 groups][2 buffers][lse2 | delta][BT] floats, 256 bytes of alignment slack (see the kernels), barriers
  static constexpr int SMEM_DKV = 2 * BIG + 2 * NST_DKV * SMALL + 4 * PT + 2048 /*stats*/ + 256 + 256;
  static constexpr int SMEM_DQ = 2 * BIG + 2 * NST_DQ * SMALL + 2 * PT + 256 + 256;
  static_assert(SMEM_DKV <= 227 * 1024 && SMEM_DQ <= 227 * 1024, "attention backward: shared memory budget");
  static_assert(4 * BT + 2 * DHO <= 512 && 4 * BT + DH <= 512, "attention backward: TMEM budget");
};

// write 64 bf16 (this thread's row r) into a K-major [128 x 64] operand tile (128-byte rows, 128B swizzle)
__device__ __forceinline__ void write_row64(uint32_t tile, int r, const float* v) {
#pragma unroll
  for (int c = 0; c < 8; c++) {
    uint32_t pk[4];
#pragma unroll
    for (int i = 0; i < 4; i++) {
      __nv_bfloat162 t2 = __floats2bfloat162_rn(v[c * 8 + 2 * i], v[c * 8 + 2 * i + 1]);
      pk[i] = *reinterpret_cast<uint32_t*>(&t2);
    }
    const uint32_t addr = tile + r * 128 + ((c ^ (r & 7)) << 4);
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(pk[0]), "r"(pk[1]), "r"(pk[2]), "r"(pk[3]) : "memory");
  }
}
// same for 32 of the 64 columns (chunks 4*half .. 4*half + 3): two warps share a row (backward softmax warps)
__device__ __forceinline__ void write_row32(uint32_t tile, int r, const float* v, int half) {
#pragma unroll
  for (int c = 0; c < 4; c++) {
    uint32_t pk[4];
#pragma unroll
    for (int i = 0; i < 4; i++) {
      __nv_bfloat162 t2 = __floats2bfloat162_rn(v[c * 8 + 2 * i], v[c * 8 + 2 * i + 1]);
      pk[i] = *reinterpret_cast<uint32_t*>(&t2);
    }
    const uint32_t addr = tile + r * 128 + (((half * 4 + c) ^ (r & 7)) << 4);
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(pk[0]), "r"(pk[1]), "r"(pk[2]), "r"(pk[3]) : "memory");
  }
}
// 16 of the 32 columns of a [128 x 32] K-major operand tile with 64-byte rows (64B swizzle: 16-byte chunk index ^ ((row >> 1) & 3))
__device__ __forceinline__ void write_row16_sw64(uint32_t tile, int r, const float* v, int half) {
#pragma unroll
  for (int c = 0; c < 2; c++) {
    uint32_t pk[4];
#pragma unroll
    for (int i = 0; i < 4; i++) {
      __nv_bfloat162 t2 = __floats2bfloat162_rn(v[c * 8 + 2 * i], v[c * 8 + 2 * i + 1]);
      pk[i] = *reinterpret_cast<uint32_t*>(&t2);
    }
    const uint32_t addr = tile + r * 64 + (((half * 2 + c) ^ ((r >> 1) & 3)) << 4);
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(pk[0]), "r"(pk[1]), "r"(pk[2]), "r"(pk[3]) : "memory");
  }
}
// 16 columns (two 16-byte chunks, column group g16 of the row) of a [128 x BT] K-major operand tile: 128-byte rows with 128B
// swizzle at BT = 64, 64-byte rows with 64B swizzle at BT = 32
template <int BT>
__device__ __forceinline__ void write_cols16(uint32_t tile, int r, const float* v, int g16) {
#pragma unroll
  for (int c = 0; c < 2; c++) {
    uint32_t pk[4];
#pragma unroll
    for (int i = 0; i < 4; i++) {
      __nv_bfloat162 t2 = __floats2bfloat162_rn(v[c * 8 + 2 * i], v[c * 8 + 2 * i + 1]);
      pk[i] = *reinterpret_cast<uint32_t*>(&t2);
    }
    const uint32_t addr = BT == 64 ? tile + r * 128 + (((g16 * 2 + c) ^ (r & 7)) << 4)
                                   : tile + r * 64 + (((g16 * 2 + c) ^ ((r >> 1) & 3)) << 4);
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(pk[0]), "r"(pk[1]), "r"(pk[2]), "r"(pk[3]) : "memory");
  }
}
// K-major descriptor of a [128 x BT] operand tile
template <int BT>
__device__ __forceinline__ uint64_t optile_desc(uint32_t saddr) {
  return BT == 64 ? ptx::make_smem_desc(saddr, 16, 1024) : ptx::make_smem_desc_sw64(saddr, 16, 512);
}
// TMEM accumulator row (DH fp32 columns of this thread's lane) * scale -> bf16 -> global row
template <int DH>
__device__ __forceinline__ void store_acc_row(uint32_t taddr, bf16* dst, float scale, bool ok) {
#pragma unroll
  for (int c = 0; c < DH / 32; c++) {
    uint32_t o[32];
    ptx::tmem_ld_32x32(taddr + c * 32, o);
    ptx::tmem_ld_wait();
    if (ok) {
#pragma unroll
      for (int g8 = 0; g8 < 4; g8++) {
        uint4 v;
        uint32_t* pv = reinterpret_cast<uint32_t*>(&v);
#pragma unroll
        for (int i = 0; i < 4; i++) {
          __nv_bfloat162 t2 = __floats2bfloat162_rn(__uint_as_float(o[g8 * 8 + 2 * i]) * scale, __uint_as_float(o[g8 * 8 + 2 * i + 1]) * scale);
          pv[i] = *reinterpret_cast<uint32_t*>(&t2);
        }
        *reinterpret_cast<uint4*>(dst + c * 32 + g8 * 8) = v;
      }
    }
  }
}

// ---------------------------------------------------------------- dK, dV : rows = keys -------------------
template <int DH>
__global__ void __launch_bounds__(NTHB, 1)
attn_bwd_dkv_tc5_kernel(const __grid_constant__ CUtensorMap tmBig, const __grid_constant__ CUtensorMap tmSmall,
                        const __grid_constant__ CUtensorMap tmdO, AttnArgs a, float scale, float sl2) {
  using C = CfgB<DH>;
  constexpr int BT = C::BT, CW = BT / 2, DHO = C::DHO;       // streamed rows; columns per softmax warp; dK / dV columns of this CTA
  const int slice = blockIdx.z;                              // which DHO-column slice of dK / dV (d_h = 256: two)
  extern __shared__ __align__(1024) uint8_t smem_raw[];     // see attn_fwd_tc5_kernel: 256 bytes of slack budgeted, fail loudly beyond
  const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  if (base - ptx::smem_u32(smem_raw) > 256u) __trap();
  const uint32_t sK = base, sV = sK + C::BIG, sRing = sV + C::BIG, sPt0 = sRing + 2 * C::NST_DKV * C::SMALL,
                 sStat = sPt0 + 4 * C::PT, bar = sStat + 2048;
  auto sQ = [&](int st) { return sRing + st * 2 * C::SMALL; };
  auto sdO = [&](int st) { return sRing + st * 2 * C::SMALL + C::SMALL; };
  float* stat = reinterpret_cast<float*>(smem_raw + (sStat - ptx::smem_u32(smem_raw)));   // [2 groups][2 uses][lse2 | delta][BT]
  constexpr int NST = C::NST_DKV;
  const uint32_t kv_full = bar, qdo_full0 = bar + 8, qdo_empty0 = qdo_full0 + 8 * NST, st_full0 = qdo_empty0 + 8 * NST,
                 st_empty0 = st_full0 + 16, p_full0 = st_empty0 + 16, p_done0 = p_full0 + 16, tmem_slot = p_done0 + 16;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int bh = blockIdx.y, b = bh / a.heads, h = bh - b * a.heads, N = a.N;
  const int k0 = blockIdx.x * 128;
  const int ntiles = (N + BT - 1) / BT;
  const int row0 = b * N;
  const int qc = a.q_off + h * DH, kc = a.k_off + h * DH, vc = a.v_off + h * DH;

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&tmBig); ptx::prefetch_tmap(&tmSmall); ptx::prefetch_tmap(&tmdO);
    ptx::mbar_init(kv_full, 1);
    for (int i = 0; i < NST; i++) { ptx::mbar_init(qdo_full0 + 8 * i, 1); ptx::mbar_init(qdo_empty0 + 8 * i, 1); }
    // st_empty: released by the 8 softmax warps once S^T / dP^T are in registers, or (TS_DKV: the operands live in those
    // columns) by the commit of the gradient MMAs that read them
    for (int i = 0; i < 2; i++) { ptx::mbar_init(st_full0 + 8 * i, 2);  ptx::mbar_init(st_empty0 + 8 * i, TS_DKV ? 1 : 8); }
    for (int i = 0; i < 2; i++) { ptx::mbar_init(p_full0 + 8 * i, 8); ptx::mbar_init(p_done0 + 8 * i, 1); }
    ptx::fence_barrier_init();
  }
  if (warp == 1) { ptx::tmem_alloc(tmem_slot, 512); ptx::tmem_relinquish(); }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem) : "r"(tmem_slot));
  pdl_wait();                                    // on-chip prologue done; first global access is below
  pdl_trigger();
  const uint32_t tSt = tmem, tdPt = tmem + 2 * BT, tdV = tmem + 4 * BT, tdK = tdV + DHO;

  if (warp == 0) {
    if (lane == 0) {
      ptx::mbar_expect_tx(kv_full, 2 * C::BIG);
#pragma unroll
      for (int bk = 0; bk < C::NBLK; bk++) {
        ptx::tma_load_2d(sK + bk * C::BBLK, &tmBig, kv_full, kc + bk * 64, row0 + k0);
        ptx::tma_load_2d(sV + bk * C::BBLK, &tmBig, kv_full, vc + bk * 64, row0 + k0);
      }
      for (int j = 0; j < ntiles; j++) {
        const int st = j % NST;
        ptx::mbar_wait(qdo_empty0 + 8 * st, ((j / NST) & 1) ^ 1);
        ptx::mbar_expect_tx(qdo_full0 + 8 * st, 2 * C::SMALL);
#pragma unroll
        for (int bk = 0; bk < C::NBLK; bk++) {
          ptx::tma_load_2d(sQ(st) + bk * C::SBLK, &tmSmall, qdo_full0 + 8 * st, qc + bk * 64, row0 + j * BT);
          ptx::tma_load_2d(sdO(st) + bk * C::SBLK, &tmdO, qdo_full0 + 8 * st, h * DH + bk * 64, row0 + j * BT);
        }
      }
    }
  } else if (warp == 1 || warp >= NTHB / 32 - 2) {   // warp 1: gradient MMAs; last warp: S^T / dP^T MMAs (issue-bound otherwise)
    if (lane == 0) {
      constexpr uint32_t idesc_s = ptx::make_idesc_bf16(128, BT, 0, 0);
      constexpr uint32_t idesc_g = ptx::make_idesc_bf16(128, DHO, 0, 1);
      auto issue_s = [&](int j) {
        const int st = j % NST, tb = j & 1;
        ptx::mbar_wait(qdo_full0 + 8 * st, (j / NST) & 1);
        ptx::mbar_wait(st_empty0 + 8 * tb, ((j >> 1) & 1) ^ 1);
        ptx::tc_fence_after();
        const uint64_t dK0 = ptx::make_smem_desc(sK, 16, 1024), dV0 = ptx::make_smem_desc(sV, 16, 1024);
        const uint64_t dQs = ptx::make_smem_desc(sQ(st), 16, 1024), dOs = ptx::make_smem_desc(sdO(st), 16, 1024);
        if (warp == NTHB / 32 - 1) {
#pragma unroll
          for (int ks = 0; ks < DH / 16; ks++) {
            const uint32_t ob = (ks >> 2) * C::BBLK + (ks & 3) * 32, os = (ks >> 2) * C::SBLK + (ks & 3) * 32;
            ptx::mma_f16_ss(tSt + tb * BT, desc_adv(dK0, ob), desc_adv(dQs, os), idesc_s, ks != 0);
          }
        } else {
#pragma unroll
          for (int ks = 0; ks < DH / 16; ks++) {
            const uint32_t ob = (ks >> 2) * C::BBLK + (ks & 3) * 32, os = (ks >> 2) * C::SBLK + (ks & 3) * 32;
            ptx::mma_f16_ss(tdPt + tb * BT, desc_adv(dV0, ob), desc_adv(dOs, os), idesc_s, ks != 0);
          }
        }
        ptx::mma_commit(st_full0 + 8 * tb);
      };
      ptx::mbar_wait(kv_full, 0);
      if (warp != 1) {
        for (int j = 0; j < ntiles; j++) issue_s(j);
      } else
      for (int j = 0; j < ntiles; j++) {
        ptx::mbar_wait(qdo_full0 + 8 * (j % NST), (j / NST) & 1);
        const int pb = j & 1;
        const uint32_t sPt = sPt0 + pb * 2 * C::PT, sdSt = sPt + C::PT;
        ptx::mbar_wait(p_full0 + 8 * pb, (j >> 1) & 1);
        ptx::tc_fence_after();
        const int st = j % NST;
        const uint64_t dPt = optile_desc<BT>(sPt), dSt = optile_desc<BT>(sdSt);
        // streamed tiles as MN-major B operands: this CTA's DHO columns start (slice * DHO / 64) blocks in
        const uint32_t so = slice * (DHO / 64) * C::SBLK;
        const uint64_t dOm = ptx::make_smem_desc(sdO(st) + so, C::SBLK, 1024), dQm = ptx::make_smem_desc(sQ(st) + so, C::SBLK, 1024);
        if (TS_DKV) {                             // A operands in TMEM: k-step ks (16 queries) = 8 columns at offset 16 ks of the buffer
#pragma unroll
          for (int ks = 0; ks < BT / 16; ks++)    // dV += P^T dO_j   (contraction over the tile's queries)
            ptx::mma_f16_ts(tdV, tSt + pb * BT + ks * 16, desc_adv(dOm, ks * 2048), idesc_g, (j | ks) != 0);
#pragma unroll
          for (int ks = 0; ks < BT / 16; ks++)    // dK += dS^T Q_j
            ptx::mma_f16_ts(tdK, tdPt + pb * BT + ks * 16, desc_adv(dQm, ks * 2048), idesc_g, (j | ks) != 0);
          ptx::mma_commit(st_empty0 + 8 * pb);    // the S^T / dP^T columns of this buffer may be overwritten
        } else {
#pragma unroll
          for (int ks = 0; ks < BT / 16; ks++)    // dV += P^T dO_j   (contraction over the tile's 64 queries)
            ptx::mma_f16_ss(tdV, desc_adv(dPt, ks * 32), desc_adv(dOm, ks * 2048), idesc_g, (j | ks) != 0);
#pragma unroll
          for (int ks = 0; ks < BT / 16; ks++)    // dK += dS^T Q_j
            ptx::mma_f16_ss(tdK, desc_adv(dSt, ks * 32), desc_adv(dQm, ks * 2048), idesc_g, (j | ks) != 0);
        }
        ptx::mma_commit(qdo_empty0 + 8 * st);
        ptx::mma_commit(p_done0 + 8 * pb);
      }
    }
  } else {
    const int sw = warp - 2, grp = sw >> 3;                  // softmax warp 0..15; group = parity of the tiles it works on
    const int quarter = warp & 3, half = (sw & 7) >> 2;      // this warp: 32 key rows x CW of the tile's BT query columns
    const int r = quarter * 32 + lane;                       // key row within the CTA tile = TMEM lane
    const uint32_t lane_off = (uint32_t)(quarter * 32) << 16;
    const int gi = (sw & 7) * 32 + lane;                     // 0..255 within the group: the first 2 BT load the statistics
    auto load_stat = [&](int j) -> float {
      const int q = j * BT + (gi % BT);
      if (gi >= 2 * BT || j >= ntiles || q >= N) return 0.f;
      return (gi / BT) ? a.delta[(size_t)bh * N + q] : a.lse[(size_t)bh * N + q] * LOG2E;
    };
    float nxt = load_stat(grp);
    for (int j = grp; j < ntiles; j += 2) {
      const int st = grp;                                    // accumulator / operand-tile buffer of this group (= j & 1)
      float* sbuf = stat + (grp * 2 + ((j >> 1) & 1)) * 2 * BT;   // [group][use parity][0][c] = lse2, [..][1][c] = delta
      if (gi < 2 * BT) sbuf[gi] = nxt;
      named_bar_sync(1 + grp, 256);                          // a buffer is rewritten two barriers of the group later
      nxt = load_stat(j + 2);
      const float* lse2 = sbuf + half * CW;
      const float* dl = lse2 + BT;
      ptx::mbar_wait(st_full0 + 8 * st, (j >> 1) & 1);
      ptx::tc_fence_after();
      const uint32_t sPt = sPt0 + st * 2 * C::PT, sdSt = sPt + C::PT;
      const int nvalid = N - j * BT - half * CW;             // queries (columns) >= N are masked (ragged last tile only)
#pragma unroll
      for (int g = 0; g < CW / 16; g++) {                    // 16 columns at a time: 48 live values instead of 96
        uint32_t s[16], dp[16];
        ptx::tmem_ld_32x16(tSt + st * BT + half * CW + g * 16 + lane_off, s);
        ptx::tmem_ld_32x16(tdPt + st * BT + half * CW + g * 16 + lane_off, dp);
        ptx::tmem_ld_wait();
        if (!TS_DKV && g == CW / 16 - 1) {                   // both accumulators of this tile are in registers
          ptx::tc_fence_before();
          __syncwarp();
          if (lane == 0) ptx::mbar_arrive(st_empty0 + 8 * st);
        }
        float p[16];
#pragma unroll
        for (int c = 0; c < 16; c++) {
          const float e = fast_ex2(__uint_as_float(s[c]) * sl2 - lse2[g * 16 + c]);
          p[c] = (g * 16 + c < nvalid) ? e : 0.f;
        }
        if (TS_DKV) {
          // P^T / dS^T of these 16 queries as 8 columns of packed bf16 pairs over the first half of the 16 fp32 columns
          // just read (this thread's own lane and columns: no other thread reads or writes them)
          const uint32_t c0 = st * BT + half * CW + g * 16 + lane_off;
          uint32_t pk[8];
#pragma unroll
          for (int i = 0; i < 8; i++) { __nv_bfloat162 t2 = __floats2bfloat162_rn(p[2 * i], p[2 * i + 1]); pk[i] = *reinterpret_cast<uint32_t*>(&t2); }
          ptx::tmem_st_32x8(tSt + c0, pk);
#pragma unroll
          for (int c = 0; c < 16; c++) p[c] *= __uint_as_float(dp[c]) - dl[g * 16 + c];
#pragma unroll
          for (int i = 0; i < 8; i++) { __nv_bfloat162 t2 = __floats2bfloat162_rn(p[2 * i], p[2 * i + 1]); pk[i] = *reinterpret_cast<uint32_t*>(&t2); }
          ptx::tmem_st_32x8(tdPt + c0, pk);
        } else {
          if (g == 0 && j > 1) ptx::mbar_wait(p_done0 + 8 * st, ((j >> 1) & 1) ^ 1);   // this buffer's P^T / dS^T tiles are free again
          write_cols16<BT>(sPt, r, p, half * (CW / 16) + g);
#pragma unroll
          for (int c = 0; c < 16; c++) p[c] *= __uint_as_float(dp[c]) - dl[g * 16 + c];
          write_cols16<BT>(sdSt, r, p, half * (CW / 16) + g);
        }
      }
      if (TS_DKV) ptx::tmem_st_wait(); else ptx::fence_proxy_async();
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(p_full0 + 8 * st);
    }
    // every group waits for the gradient MMAs of ITS OWN last tile (a barrier whose phases it has followed one by one:
    // a group that never waited on the other buffer's barrier could not tell its phase k from phase k - 2), then the two
    // groups meet, and the first one drains the accumulators
    if (ntiles > grp) { const int jl = ((ntiles - 1 - grp) & ~1) + grp; ptx::mbar_wait(p_done0 + 8 * grp, (jl >> 1) & 1); }
    named_bar_sync(3, 512);
    if (grp == 0) {                                          // epilogue: DHO / 2 columns of both gradients per warp
      ptx::tc_fence_after();
      const int krow = k0 + r;
      bf16* out = (bf16*)a.dqkv + (size_t)(row0 + krow) * a.ld + slice * DHO + half * (DHO / 2);
      store_acc_row<DHO / 2>(tdV + half * (DHO / 2) + lane_off, out + vc, 1.f, krow < N);
      store_acc_row<DHO / 2>(tdK + half * (DHO / 2) + lane_off, out + kc, scale, krow < N);
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 1) { ptx::tc_fence_after(); ptx::tmem_dealloc(tmem, 512); }
}

// ---- measurement probes of the dQ kernel (A/B build only, ORBIT_NVCC_EXTRA; wrong results) ----------------------------
#ifdef ORBIT_PROBE_DQ_NOS
#define DQ_PROBE_KS(n) 1
#else
#define DQ_PROBE_KS(n) (n)
#endif
#ifdef ORBIT_PROBE_DQ_NOG
#define DQ_PROBE_KG(n) 0
#else
#define DQ_PROBE_KG(n) (n)
#endif
#ifdef ORBIT_PROBE_DQ_NOEXP
#define DQ_PROBE_EX2(x) (x)
#else
#define DQ_PROBE_EX2(x) fast_ex2(x)
#endif
#ifdef ORBIT_PROBE_DQ_NOSM
#define DQ_PROBE_NG(n) 0
#else
#define DQ_PROBE_NG(n) (n)
#endif

// ---------------------------------------------------------------- dQ : rows = queries -------------------
template <int DH>
__global__ void __launch_bounds__(NTHB, 1)
attn_bwd_dq_tc5_kernel(const __grid_constant__ CUtensorMap tmBig, const __grid_constant__ CUtensorMap tmSmall,
                       const __grid_constant__ CUtensorMap tmdOBig, AttnArgs a, float scale, float sl2, int delta_here) {
  using C = CfgB<DH>;
  constexpr int BT = C::BT, CW = BT / 2;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  if (base - ptx::smem_u32(smem_raw) > 256u) __trap();
  const uint32_t sQ = base, sdO = sQ + C::BIG, sRing = sdO + C::BIG, sdS0 = sRing + 2 * C::NST_DQ * C::SMALL, bar = sdS0 + 2 * C::PT;
  auto sK = [&](int st) { return sRing + st * 2 * C::SMALL; };
  auto sV = [&](int st) { return sRing + st * 2 * C::SMALL + C::SMALL; };
  constexpr int NST = C::NST_DQ;
  // S / dP buffers: with dS kept in tensor memory a buffer stays busy until the dQ MMAs of its tile have read it, so a
  // third one keeps the S / dP products of tile j+2 from waiting on them
  // Q and dO (stationary) as tensor-memory A operands of the S / dP products where the columns allow it: those products
  // then read only the streamed K / V tile from shared memory
  constexpr int NB = !TS_DQ ? 2 : (TSA_DQ && 4 * BT + 2 * DH <= 512 && 6 * BT + 2 * DH > 512) ? 2 : 3;
  constexpr bool TSA = TSA_DQ && 2 * NB * BT + 2 * DH <= 512;
  static_assert(2 * NB * BT + DH <= 512, "attention backward (dQ): TMEM budget");
  const uint32_t q_full = bar, kv_full0 = bar + 8, kv_empty0 = kv_full0 + 8 * NST, s_full0 = kv_empty0 + 8 * NST,
                 s_empty0 = s_full0 + 8 * NB, p_full0 = s_empty0 + 8 * NB, p_done0 = p_full0 + 8 * NB, tmem_slot = p_done0 + 8 * NB;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  PROBE_DECL;
  PROBE_T0;
  const int bh = blockIdx.y, b = bh / a.heads, h = bh - b * a.heads, N = a.N;
  const int q0 = blockIdx.x * 128;
  const int ntiles = (N + BT - 1) / BT;
  const int row0 = b * N;
  const int qc = a.q_off + h * DH, kc = a.k_off + h * DH, vc = a.v_off + h * DH;

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&tmBig); ptx::prefetch_tmap(&tmSmall); ptx::prefetch_tmap(&tmdOBig);
    ptx::mbar_init(q_full, TSA ? 16 : 1);
    for (int i = 0; i < NST; i++) { ptx::mbar_init(kv_full0 + 8 * i, 1); ptx::mbar_init(kv_empty0 + 8 * i, 1); }
    for (int i = 0; i < NB; i++) { ptx::mbar_init(s_full0 + 8 * i, 2);  ptx::mbar_init(s_empty0 + 8 * i, TS_DQ ? 1 : 8); }   // as in the dK / dV kernel
    for (int i = 0; i < NB; i++) { ptx::mbar_init(p_full0 + 8 * i, 8); ptx::mbar_init(p_done0 + 8 * i, 1); }
    ptx::fence_barrier_init();
  }
  if (warp == 1) { ptx::tmem_alloc(tmem_slot, 512); ptx::tmem_relinquish(); }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem) : "r"(tmem_slot));
  pdl_wait();                                    // on-chip prologue done; first global access is below
  pdl_trigger();
  const uint32_t tS = tmem, tdP = tmem + NB * BT, tdQ = tmem + 2 * NB * BT, tQ = tdQ + DH, tdO = tQ + DH / 2;

  if (warp == 0) {
    if (lane == 0) {
      if (!TSA) ptx::mbar_expect_tx(q_full, 2 * C::BIG);
#pragma unroll
      for (int bk = 0; bk < (TSA ? 0 : C::NBLK); bk++) {
        ptx::tma_load_2d(sQ + bk * C::BBLK, &tmBig, q_full, qc + bk * 64, row0 + q0);
        ptx::tma_load_2d(sdO + bk * C::BBLK, &tmdOBig, q_full, h * DH + bk * 64, row0 + q0);
      }
      for (int j = 0; j < ntiles; j++) {
        const int st = j % NST;
        PWAIT(0, kv_empty0 + 8 * st, ((j / NST) & 1) ^ 1);
        ptx::mbar_expect_tx(kv_full0 + 8 * st, 2 * C::SMALL);
#pragma unroll
        for (int bk = 0; bk < C::NBLK; bk++) {
          ptx::tma_load_2d(sK(st) + bk * C::SBLK, &tmSmall, kv_full0 + 8 * st, kc + bk * 64, row0 + j * BT);
          ptx::tma_load_2d(sV(st) + bk * C::SBLK, &tmSmall, kv_full0 + 8 * st, vc + bk * 64, row0 + j * BT);
        }
      }
      PSINCE(11); PFLUSH(0, 0); PFLUSH(11, 11);
    }
  } else if (warp == 1 || warp >= NTHB / 32 - 2) {   // warp 1: dQ MMAs; last warp: S / dP MMAs
    if (lane == 0) {
      constexpr uint32_t idesc_s = ptx::make_idesc_bf16(128, BT, 0, 0);
      constexpr uint32_t idesc_g = ptx::make_idesc_bf16(128, DH, 0, 1);
      auto issue_s = [&](int j) {
        const int st = j % NST, tb = j % NB;
        PWAIT(1, kv_full0 + 8 * st, (j / NST) & 1);
        PWAIT(2, s_empty0 + 8 * tb, ((j / NB) & 1) ^ 1);
        ptx::tc_fence_after();
        const uint64_t dQ0 = ptx::make_smem_desc(sQ, 16, 1024), dO0 = ptx::make_smem_desc(sdO, 16, 1024);
        const uint64_t dKs = ptx::make_smem_desc(sK(st), 16, 1024), dVs = ptx::make_smem_desc(sV(st), 16, 1024);
        if (warp == NTHB / 32 - 1) {
#pragma unroll
          for (int ks = 0; ks < DQ_PROBE_KS(DH / 16); ks++) {
            const uint32_t ob = (ks >> 2) * C::BBLK + (ks & 3) * 32, os = (ks >> 2) * C::SBLK + (ks & 3) * 32;
            if (TSA) ptx::mma_f16_ts(tS + tb * BT, tQ + ks * 8, desc_adv(dKs, os), idesc_s, ks != 0);
            else ptx::mma_f16_ss(tS + tb * BT, desc_adv(dQ0, ob), desc_adv(dKs, os), idesc_s, ks != 0);
          }
        } else {
#pragma unroll
          for (int ks = 0; ks < DQ_PROBE_KS(DH / 16); ks++) {
            const uint32_t ob = (ks >> 2) * C::BBLK + (ks & 3) * 32, os = (ks >> 2) * C::SBLK + (ks & 3) * 32;
            if (TSA) ptx::mma_f16_ts(tdP + tb * BT, tdO + ks * 8, desc_adv(dVs, os), idesc_s, ks != 0);
            else ptx::mma_f16_ss(tdP + tb * BT, desc_adv(dO0, ob), desc_adv(dVs, os), idesc_s, ks != 0);
          }
        }
        ptx::mma_commit(s_full0 + 8 * tb);
      };
      PWAIT(15, q_full, 0);
      if (warp != 1) {
        for (int j = 0; j < ntiles; j++) issue_s(j);
        if (warp == NTHB / 32 - 1) { PSINCE(8); PFLUSH(1, 2); PFLUSH(8, 8); PFLUSH(15, 15); }
      } else
      for (int j = 0; j < ntiles; j++) {
        PWAIT(3, kv_full0 + 8 * (j % NST), (j / NST) & 1);
        const int pb = j % NB;
        const uint32_t sdS = sdS0 + (pb & 1) * C::PT;
        PWAIT(4, p_full0 + 8 * pb, (j / NB) & 1);
        ptx::tc_fence_after();
        const int st = j % NST;
        const uint64_t dSd = optile_desc<BT>(sdS), dKm = ptx::make_smem_desc(sK(st), C::SBLK, 1024);
        if (TS_DQ) {                             // dS stays in TMEM over the dP columns (A operand from tensor memory)
#pragma unroll
          for (int ks = 0; ks < BT / 16; ks++)    // dQ += dS K_j   (contraction over the tile's keys)
            ptx::mma_f16_ts(tdQ, tdP + pb * BT + ks * 16, desc_adv(dKm, ks * 2048), idesc_g, (j | ks) != 0);
          ptx::mma_commit(s_empty0 + 8 * pb);
        } else {
#pragma unroll
          for (int ks = 0; ks < DQ_PROBE_KG(BT / 16); ks++)    // dQ += dS K_j   (contraction over the tile's 64 keys)
            ptx::mma_f16_ss(tdQ, desc_adv(dSd, ks * 32), desc_adv(dKm, ks * 2048), idesc_g, (j | ks) != 0);
        }
        ptx::mma_commit(kv_empty0 + 8 * st);
        ptx::mma_commit(p_done0 + 8 * pb);
      }
      if (warp == 1) { PSINCE(9); PFLUSH(3, 4); PFLUSH(9, 9); }
    }
  } else {
    const int sw = warp - 2, grp = sw >> 3;                  // two groups of 8 warps alternate over the tiles (see NTHB)
    const int quarter = warp & 3, half = (sw & 7) >> 2;      // 32 query rows x CW of the tile's BT key columns
    const int r = quarter * 32 + lane;
    const uint32_t lane_off = (uint32_t)(quarter * 32) << 16;
    const int qrow = q0 + r;
    const float lse2 = qrow < N ? a.lse[(size_t)bh * N + qrow] * LOG2E : 0.f;
    // delta[row] = sum_d dO[row, d] O[row, d]: read from the delta kernel's output, or -- short sequences (N <= 1024), where a
    // launch of its own costs more than it computes (C2: +10 % on the attention backward, one launch less per block) --
    // computed HERE: the four threads that share a query row (two groups x two column halves) take a quarter of the head's
    // columns each while the first K / V tiles are in flight, exchange the partial sums through the (not yet used) dS tile,
    // and the row's value is written out for the dK / dV kernel, which runs after this one.  At N = 2048 the in-kernel
    // version delays the first softmax tile by more than the separate kernel takes (C5: 417 -> 409 TFLOP/s; a coalesced
    // warp-per-row variant: 407, and 184 instead of 207 at C2).
    float dl = 0.f;
    if (!delta_here) {
      dl = qrow < N ? a.delta[(size_t)bh * N + qrow] : 0.f;
    } else {
      const int part = grp * 2 + half;
      float acc = 0.f;
      if (qrow < N) {
        const bf16* po = (const bf16*)a.O + (size_t)(row0 + qrow) * a.ldo + h * DH + part * (DH / 4);
        const bf16* pd = (const bf16*)a.dO + (size_t)(row0 + qrow) * a.lddo + h * DH + part * (DH / 4);
#pragma unroll
        for (int c = 0; c < DH / 32; c++) {
          const uint4 xo = __ldg(reinterpret_cast<const uint4*>(po) + c), xd = __ldg(reinterpret_cast<const uint4*>(pd) + c);
          const uint32_t wo[4] = {xo.x, xo.y, xo.z, xo.w}, wd[4] = {xd.x, xd.y, xd.z, xd.w};
#pragma unroll
          for (int q = 0; q < 4; q++) {
            const float2 fo = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&wo[q]));
            const float2 fd = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&wd[q]));
            acc += fo.x * fd.x + fo.y * fd.y;
          }
        }
      }
      asm volatile("st.shared.f32 [%0], %1;" ::"r"(sdS0 + (uint32_t)(part * 128 + r) * 4), "f"(acc) : "memory");
      named_bar_sync(3, 512);
#pragma unroll
      for (int q = 0; q < 4; q++) {
        float v;
        asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(sdS0 + (uint32_t)(q * 128 + r) * 4) : "memory");
        dl += v;
      }
      named_bar_sync(3, 512);                                // the dS tile may be written from here on
      if (part == 0 && qrow < N) a.delta[(size_t)bh * N + qrow] = dl;
    }
    if (TSA) {                                               // this thread's row of Q / dO, a quarter of the columns per warp
      const int part = sw >> 2;
      const bf16* src = part < 2 ? (const bf16*)a.qkv + (size_t)(row0 + qrow) * a.ld + qc + part * (DH / 2)
                                 : (const bf16*)a.dO + (size_t)(row0 + qrow) * a.lddo + h * DH + (part - 2) * (DH / 2);
      const uint32_t dst = (part < 2 ? tQ + part * (DH / 4) : tdO + (part - 2) * (DH / 4)) + lane_off;
#pragma unroll
      for (int c = 0; c < DH / 32; c++) {                    // 8 columns = 16 bf16 per store
        uint4 v0 = make_uint4(0, 0, 0, 0), v1 = v0;
        if (qrow < N) { v0 = __ldg(reinterpret_cast<const uint4*>(src + c * 16)); v1 = __ldg(reinterpret_cast<const uint4*>(src + c * 16 + 8)); }
        const uint32_t pk[8] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w};
        ptx::tmem_st_32x8(dst + c * 8, pk);
      }
      ptx::tmem_st_wait();
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(q_full);
    }
    for (int j = grp; j < ntiles; j += 2) {
      const int st = j % NB, ph = (j / NB) & 1;
      PWAIT(5, s_full0 + 8 * st, ph);
      ptx::tc_fence_after();
      const int nvalid = N - j * BT - half * CW;             // keys (columns) >= N are masked (ragged last tile only)
#pragma unroll
      for (int g = 0; g < DQ_PROBE_NG(CW / 16); g++) {
        uint32_t s[16], dp[16];
        ptx::tmem_ld_32x16(tS + st * BT + half * CW + g * 16 + lane_off, s);
#ifndef ORBIT_PROBE_DQ_HALFLD
        ptx::tmem_ld_32x16(tdP + st * BT + half * CW + g * 16 + lane_off, dp);
#endif
        ptx::tmem_ld_wait();
#ifdef ORBIT_PROBE_DQ_HALFLD
#pragma unroll
        for (int c = 0; c < 16; c++) dp[c] = s[c];
#endif
        if (!TS_DQ && g == CW / 16 - 1) {
          ptx::tc_fence_before();
          __syncwarp();
          if (lane == 0) ptx::mbar_arrive(s_empty0 + 8 * st);
        }
        float ds[16];
#pragma unroll
        for (int c = 0; c < 16; c++) {
          const float pv = DQ_PROBE_EX2(__uint_as_float(s[c]) * sl2 - lse2);
          ds[c] = (g * 16 + c < nvalid) ? pv * (__uint_as_float(dp[c]) - dl) : 0.f;
        }
        if (TS_DQ) {
          uint32_t pk[8];
#pragma unroll
          for (int i = 0; i < 8; i++) { __nv_bfloat162 t2 = __floats2bfloat162_rn(ds[2 * i], ds[2 * i + 1]); pk[i] = *reinterpret_cast<uint32_t*>(&t2); }
          ptx::tmem_st_32x8(tdP + st * BT + half * CW + g * 16 + lane_off, pk);
        } else {
          if (g == 0 && j >= NB) PWAIT(6, p_done0 + 8 * st, ph ^ 1);
          write_cols16<BT>(sdS0 + st * C::PT, r, ds, half * (CW / 16) + g);
        }
      }
#ifdef ORBIT_PROBE_DQ_NOSM
      if (j >= NB) ptx::mbar_wait(p_done0 + 8 * st, ph ^ 1);
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(s_empty0 + 8 * st);
#endif
      if (TS_DQ) ptx::tmem_st_wait(); else ptx::fence_proxy_async();
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(p_full0 + 8 * st);
    }
    PSINCE(7);
    if (ntiles > grp) { const int jl = ((ntiles - 1 - grp) & ~1) + grp; PWAIT(12, p_done0 + 8 * (jl % NB), (jl / NB) & 1); }
    named_bar_sync(3, 512);                                  // see the dK / dV kernel
    if (grp == 0) {
      ptx::tc_fence_after();
      store_acc_row<DH / 2>(tdQ + half * (DH / 2) + lane_off,
                            (bf16*)a.dqkv + (size_t)(row0 + qrow) * a.ld + qc + half * (DH / 2), scale, qrow < N);
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2 && lane == 0) { PSINCE(13); PSET(10, ntiles); PFLUSH(5, 7); PFLUSH(10, 10); PFLUSH(12, 13); }
  if (warp == 1) { ptx::tc_fence_after(); ptx::tmem_dealloc(tmem, 512); }
}

// delta[b,h,i] = sum_d dO[i, h*dh+d] * O[i, h*dh+d].  A lane takes 16 bytes of a row (8 of its d_h values); a warp covers 4 rows
// (d_h 64), 2 (d_h 128) or 1 (d_h 192 / 256) per pass: 4-byte loads with one row per warp ran at 2.6 TB/s.
__global__ void attn_delta5_kernel(AttnArgs a) {
  pdl_wait();
  pdl_trigger();
  const int nchunk = a.dh >> 3;                                  // 16-byte pieces per row
  const int rpw = nchunk <= 8 ? 4 : (nchunk <= 16 ? 2 : 1), gs = 32 / rpw;
  const int lane = threadIdx.x & 31, sub = lane / gs, ch = lane - sub * gs;
  const long long w = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const long long total = (long long)a.B * a.heads * a.N;
  const long long row_id = w * rpw + sub;
  float s = 0.f;
  if (row_id < total && ch < nchunk) {
    const int bh = (int)(row_id / a.N), i = (int)(row_id - (long long)bh * a.N), b = bh / a.heads, h = bh - b * a.heads;
    const size_t row = (size_t)b * a.N + i;
    const uint4 xo = __ldg(reinterpret_cast<const uint4*>((const bf16*)a.O + row * a.ldo + h * a.dh) + ch);
    const uint4 xd = __ldg(reinterpret_cast<const uint4*>((const bf16*)a.dO + row * a.lddo + h * a.dh) + ch);
    const uint32_t wo[4] = {xo.x, xo.y, xo.z, xo.w}, wd[4] = {xd.x, xd.y, xd.z, xd.w};
#pragma unroll
    for (int q = 0; q < 4; q++) {
      const float2 fo = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&wo[q]));
      const float2 fd = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&wd[q]));
      s += fo.x * fd.x + fo.y * fd.y;
    }
  }
  for (int o = gs >> 1; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (ch == 0 && row_id < total) a.delta[row_id] = s;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn get_encode5() {
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

int make_map5(CUtensorMap* tm, const void* basep, long long ld, long long rows, int box_rows) {
  EncodeTiledFn enc = get_encode5();
  if (!enc) { set_error("cuTensorMapEncodeTiled entry point not found"); return ORBIT_ERR_CUDA; }
  cuuint64_t dims[2] = {(cuuint64_t)ld, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)ld * 2};
  cuuint32_t box[2] = {64, (cuuint32_t)box_rows};
  cuuint32_t es[2] = {1, 1};
  CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(basep), dims, strides, box, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { set_error("attention: cuTensorMapEncodeTiled failed (%d)", (int)r); return ORBIT_ERR_CUDA; }
  return ORBIT_OK;
}

template <int DH>
int launch_fwd5(const AttnArgs& a, cudaStream_t s) {
  const long long rows = (long long)a.B * a.N;
  CUtensorMap tmQ, tmKV;                                   // boxes of 64 columns x 128 (query) / Cfg::BKV (key, value) rows
  ORBIT_TRY(make_map5(&tmQ, a.qkv, a.ld, rows, 128));
  ORBIT_TRY(make_map5(&tmKV, a.qkv, a.ld, rows, Cfg<DH>::BKV));
  ORBIT_SMEM_ATTR(attn_fwd_tc5_kernel<DH>, Cfg<DH>::SMEM);
  dim3 grid(cdiv(a.N, BQ), a.B * a.heads);
  ORBIT_CUDA_CHECK(launch_pdl(attn_fwd_tc5_kernel<DH>, grid, dim3(NTH), Cfg<DH>::SMEM, s, tmQ, tmKV, a, LOG2E / sqrtf((float)DH)));
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

template <int DH>
int launch_bwd5(const AttnArgs& a, cudaStream_t s) {
  using C = CfgB<DH>;
  const long long rows = (long long)a.B * a.N;
  CUtensorMap tmBig, tmSmall, tmdOBig, tmdOSmall;
  ORBIT_TRY(make_map5(&tmBig, a.qkv, a.ld, rows, 128));
  ORBIT_TRY(make_map5(&tmSmall, a.qkv, a.ld, rows, C::BT));
  ORBIT_TRY(make_map5(&tmdOBig, a.dO, a.lddo, rows, 128));
  ORBIT_TRY(make_map5(&tmdOSmall, a.dO, a.lddo, rows, C::BT));
  ORBIT_SMEM_ATTR(attn_bwd_dkv_tc5_kernel<DH>, C::SMEM_DKV);
  ORBIT_SMEM_ATTR(attn_bwd_dq_tc5_kernel<DH>, C::SMEM_DQ);
  const int delta_here = a.N <= 1024;
  if (!delta_here) {
    const long long rows_d = (long long)a.B * a.heads * a.N;
    const int rpw = (a.dh >> 3) <= 8 ? 4 : ((a.dh >> 3) <= 16 ? 2 : 1);
    ORBIT_CUDA_CHECK(launch_pdl(attn_delta5_kernel, dim3(cdiv((rows_d + rpw - 1) / rpw * 32, 256)), dim3(256), 0, s, a));
    ORBIT_LAUNCH_CHECK();
  }
  dim3 grid(cdiv(a.N, 128), a.B * a.heads);
  const float scale = 1.0f / sqrtf((float)DH);
  ORBIT_CUDA_CHECK(launch_pdl(attn_bwd_dq_tc5_kernel<DH>, grid, dim3(NTHB), C::SMEM_DQ, s, tmBig, tmSmall, tmdOBig, a, scale, scale * LOG2E, delta_here));
  ORBIT_LAUNCH_CHECK();
  dim3 grid_kv(cdiv(a.N, 128), a.B * a.heads, C::NSPLIT);
  ORBIT_CUDA_CHECK(launch_pdl(attn_bwd_dkv_tc5_kernel<DH>, grid_kv, dim3(NTHB), C::SMEM_DKV, s, tmBig, tmSmall, tmdOSmall, a, scale, scale * LOG2E));
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}
}  // namespace

int attention_bwd_tc5(const AttnArgs& a, cudaStream_t s) {
  switch (a.dh) {
    case 64: return launch_bwd5<64>(a, s);
    case 128: return launch_bwd5<128>(a, s);
    case 192: return launch_bwd5<192>(a, s);
    default: return launch_bwd5<256>(a, s);
  }
}
bool attention_bwd_tc5_supported(const AttnArgs& a) {
  auto al16 = [](const void* p) { return (((uintptr_t)p) & 15) == 0; };
  return a.dO && al16(a.dO) && a.lddo % 8 == 0 && al16(a.dqkv);
}

bool attention_tc5_supported(const AttnArgs& a) {
  if (a.dtype != ORBIT_BF16 || (a.dh != 64 && a.dh != 128 && a.dh != 192 && a.dh != 256)) return false;
  auto al16 = [](const void* p) { return (((uintptr_t)p) & 15) == 0; };
  if (a.ld % 8 || a.ldo % 8 || a.q_off % 8 || a.k_off % 8 || a.v_off % 8) return false;
  if (!al16(a.qkv) || !al16(a.O)) return false;
  return a.N >= 128;
}
#ifdef ORBIT_PROBE_TIMELINE
int attention_probe_read(unsigned long long* out, int n, int reset) {
  unsigned long long h[32] = {0};
  if (cudaMemcpyFromSymbol(h, g_attn_probe, sizeof(h)) != cudaSuccess) return ORBIT_ERR_CUDA;
  for (int i = 0; i < n && i < 32; i++) out[i] = h[i];
  if (reset) { unsigned long long z[32] = {0}; cudaMemcpyToSymbol(g_attn_probe, z, sizeof(z)); }
  return ORBIT_OK;
}
#endif
int attention_fwd_tc5(const AttnArgs& a, cudaStream_t s) {
  switch (a.dh) {
    case 64: return launch_fwd5<64>(a, s);
    case 128: return launch_fwd5<128>(a, s);
    case 192: return launch_fwd5<192>(a, s);
    default: return launch_fwd5<256>(a, s);
  }
}

}  // namespace orbit
