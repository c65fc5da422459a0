// gemm_tc2.cu -- CTA-pair (cta_group::2) variant of the tcgen05 bf16 GEMM: a cluster of two CTAs on one TPC
// computes a 256 x 256 output tile.  Each CTA loads its own 128 rows of A and its own 128 columns of B (so the
// per-SM shared-memory traffic per MMA is halved), the leader CTA issues tcgen05.mma.cta_group::2 (M = 256),
// and each CTA drains its own 128 x 256 half of the accumulator from its own TMEM.
// Stage = 16 KB (A half) + 16 KB (B half) -> 6 stages in 192 KB.  Same operand-major handling and fused epilogue math
// as gemm_tc.cu; the results leave through 32 KB of shared-memory staging and TMA: per epilogue warp two 2 KB boxes
// (32 rows x 32 bf16 or 32 rows x 16 fp32, 64B swizzle) in flight as bulk store groups -- plain stores, or reduce-add for
// the fp32 partial sums of the Hybrid-STOP shard mode.  Direct row-per-thread stores remain as the
// fallback (aux outputs that are not bf16, resid + accumulate) and for A/B timing (orbit_set_debug_force_simt(5)).
// Synchronisation:
//   full[s]   (leader's, count 1): the leader's producer arrives expecting the bytes of BOTH CTAs; the peer's TMA
//                                  complete_tx on it too (a remote arrive per stage costs ~1400 cycles: measured)
//   empty[s]  (per CTA, count 1) : tcgen05.commit multicast to both CTAs frees the stage
//   tfull[a]  (per CTA, count 1) : tcgen05.commit multicast -> both epilogues
//   tempty[a] (leader's, count 16): the 8 epilogue warps of both CTAs release the accumulator
#include <cuda.h>
#include <stdlib.h>
#include "common.cuh"
#include "gemm_epi.cuh"
#include "ptx.cuh"

namespace orbit {
namespace {

constexpr int BM2 = 256, BN2 = 256, BK = 64, UK = 16;
constexpr int STAGES = 6;
constexpr int A_BYTES = 128 * BK * 2;           // this CTA's half of A
constexpr int B_BYTES = 128 * BK * 2;           // this CTA's half of B
constexpr int STAGE_BYTES = A_BYTES + B_BYTES;  // 32 KB
constexpr int NTHREADS = 320;                   // warp 0 TMA, warp 1 MMA, warps 2..9 epilogue (2 per TMEM lane quarter)
constexpr int TMEM_COLS = 512;
// epilogue staging for the TMA-store path: per epilogue warp two [32 rows x 32 bf16] boxes (64-byte rows, 64B swizzle)
constexpr int EPI_BOX_BYTES = 32 * 32 * 2;
constexpr int EPI_BYTES = 8 * 2 * EPI_BOX_BYTES;    // 32 KB
constexpr size_t SMEM_BYTES = (size_t)STAGES * STAGE_BYTES + EPI_BYTES + 1024 + 256;

__device__ __forceinline__ void tma_store_3d(const CUtensorMap* m, uint32_t src, int c0, int c1, int c2, uint64_t policy) {
  asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group.L2::cache_hint [%0, {%2, %3, %4}], [%1], %5;" ::"l"(m), "r"(src), "r"(c0),
               "r"(c1), "r"(c2), "l"(policy)
               : "memory");
}
__device__ __forceinline__ void tma_reduce_add_3d(const CUtensorMap* m, uint32_t src, int c0, int c1, int c2) {
  asm volatile("cp.reduce.async.bulk.tensor.3d.global.shared::cta.add.tile.bulk_group [%0, {%2, %3, %4}], [%1];" ::"l"(m), "r"(src),
               "r"(c0), "r"(c1), "r"(c2)
               : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

// Raster: groups of `group` row blocks, all column blocks of a group before the next group.  The A panels of a group
// (group x 256 x K) are what concurrent clusters share through L2; B is streamed once per group (host heuristic in launch2).
__device__ __forceinline__ void tile_coords2(int t, int tiles_m, int tiles_n, int GROUP, int& mb, int& nb) {
  const int group_size = GROUP * tiles_n;
  const int g = t / group_size, r = t - g * group_size;
  const int first_m = g * GROUP;
  const int gm = min(GROUP, tiles_m - first_m);
  mb = first_m + r % gm;
  nb = r / gm;
}
// Work units of the persistent loop.  Units [0, full) are whole 256 x 256 tiles, dealt round-robin to the clusters.  The
// tiles of the last, partial round (num_tiles % num_clusters of them: 14 of 384 at N = 12288 on 74 clusters, i.e. a sixth
// round that keeps 19 % of the SMs busy) are split into `parts` column sub-tiles of W = 256 / parts columns each, so that
// the last round takes 1 / parts of a tile time on parts x as many clusters.
// hint_a / hint_b / hint_c: L2 eviction priority of the A loads, B loads and C stores (0 normal, 1 evict_first, 2 evict_last)
// round_bar: the TMA producers of all clusters meet at a counter in global memory before each round of tiles, so that the 8-9
// clusters sharing an operand panel sweep K in step and fetch it from DRAM once: without it they drift apart and re-fetch (C5: 30.0
// -> 23.4 GB of DRAM traffic per step, fc2 4.1 -> 2.6 GB; step time unchanged on a typical box, profiles/r2_gemm_schedule.md; some
// boxes of the pool move 40 GB without it).  The wait is BOUNDED (20 us): the grid is not a cooperative launch, and a cluster that
// cannot become resident (another stream's kernel holds its SMs) must not hang the others; after a timeout the cluster stops waiting
// but keeps arriving.  ORBIT_GEMM_ROUND_SYNC=0 switches it off.
struct Sched { int full, parts, total, group_m, hint_a, hint_b, hint_c; unsigned int* round_bar; };
__device__ unsigned int g_round_bar[2 * 64];     // per slot: [arrivals, exits]; the last cluster to leave zeroes its slot
__device__ __forceinline__ void unit_of(const Sched& sc, int u, int& t, int& part, int& W) {
  if (u < sc.full) { t = u; part = 0; W = BN2; }
  else { const int r = u - sc.full; t = sc.full + r / sc.parts; part = r % sc.parts; W = BN2 / sc.parts; }
}

template <int A_MN, int B_MN>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(NTHREADS, 1)
gemm_tc2_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                const __grid_constant__ CUtensorMap tmC, const __grid_constant__ CUtensorMap tmX, int tma_store, epi::Args e0,
                int M, int N, int K,
                int batch, long long c_bs, long long bias_bs, Sched sc) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t epi_base = smem_base + STAGES * STAGE_BYTES;
  const uint32_t bar_base = epi_base + EPI_BYTES;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
  auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * STAGES + a); };
  auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * STAGES + 2 + a); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * STAGES + 4);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = ptx::cluster_ctarank();
  const bool leader = rank == 0;
  const int tiles_m = (M + BM2 - 1) / BM2, tiles_n = (N + BN2 - 1) / BN2;
  const int tiles_per_batch = tiles_m * tiles_n;
  const int num_tiles = tiles_per_batch * batch;
  const int num_kb = (K + BK - 1) / BK;
  const int cluster_id = blockIdx.x >> 1, num_clusters = gridDim.x >> 1;

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&tmA);
    ptx::prefetch_tmap(&tmB);
    if (tma_store) ptx::prefetch_tmap(&tmC);
    if (tma_store & 2) ptx::prefetch_tmap(&tmX);
    for (int s = 0; s < STAGES; s++) { ptx::mbar_init(full_bar(s), 1); ptx::mbar_init(empty_bar(s), 1); }
    for (int a = 0; a < 2; a++) { ptx::mbar_init(tfull_bar(a), 1); ptx::mbar_init(tempty_bar(a), 16); }
    ptx::fence_barrier_init();
  }
  if (warp == 1) {
    ptx::tmem_alloc_2sm(tmem_slot, TMEM_COLS);
    ptx::tmem_relinquish_2sm();
  }
  ptx::tc_fence_before();
  ptx::cluster_sync_all();                       // barrier inits and TMEM allocation visible in both CTAs
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));
  pdl_wait();                                    // everything above touched only on-chip state and kernel parameters
  pdl_trigger();

  if (warp == 0) {
    // ===================== TMA producer (both CTAs) =====================
    if (lane == 0) {
      int s = 0; uint32_t ph = 0;
      const uint64_t pol_a = ptx::l2_policy(sc.hint_a), pol_b = ptx::l2_policy(sc.hint_b);
      unsigned int target = 0;
      bool gave_up = false;
      for (int u = cluster_id, round = 0; u < sc.total; u += num_clusters, round++) {
        if (sc.round_bar && round > 0) {         // all clusters that have a unit in this round start it together
          const int left = sc.total - round * num_clusters;
          target += (unsigned int)(left < num_clusters ? left : num_clusters);
          if (leader) atomicAdd(sc.round_bar, 1u);
          if (!gave_up) {
            unsigned long long t0, t1;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
            unsigned int seen;
            do {
              asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(sc.round_bar) : "memory");
              asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
              if (t1 - t0 > 20000ull) { gave_up = true; break; }
            } while (seen < target);
          }
        }
        int t, part, W;
        unit_of(sc, u, t, part, W);
        const int bi = t / tiles_per_batch;
        int mb, nb;
        tile_coords2(t - bi * tiles_per_batch, tiles_m, tiles_n, sc.group_m, mb, nb);
        // a sub-tile loads the same boxes (expect_tx unchanged) from its own column origin and uses the first W / 2 of them
        const int m0 = mb * BM2 + (int)rank * 128, n0 = nb * BN2 + part * W + (int)rank * (W / 2);
        for (int kb = 0; kb < num_kb; kb++) {
          ptx::mbar_wait(empty_bar(s), ph ^ 1);
          const uint32_t lfull = ptx::mapa(full_bar(s), 0);
          if (leader) ptx::mbar_expect_tx(full_bar(s), 2 * STAGE_BYTES);
          const uint32_t sa = smem_base + s * STAGE_BYTES, sb = sa + A_BYTES;
          const int k0 = kb * BK;
          if (A_MN) {
#pragma unroll
            for (int i = 0; i < 2; i++) ptx::tma_load_3d_2sm_hint(sa + i * 8192, &tmA, lfull, m0 + i * 64, k0, bi, pol_a);
          } else {
            ptx::tma_load_3d_2sm_hint(sa, &tmA, lfull, k0, m0, bi, pol_a);
          }
          if (B_MN) {
#pragma unroll
            for (int i = 0; i < 2; i++) ptx::tma_load_3d_2sm_hint(sb + i * 8192, &tmB, lfull, n0 + i * 64, k0, bi, pol_b);
          } else {
            ptx::tma_load_3d_2sm_hint(sb, &tmB, lfull, k0, n0, bi, pol_b);
          }
          if (++s == STAGES) { s = 0; ph ^= 1; }
        }
      }
      if (sc.round_bar && leader) {            // every cluster has passed its last meeting point once all have left: reset the slot
        __threadfence();
        if (atomicAdd(sc.round_bar + 1, 1u) == (unsigned int)num_clusters - 1) { sc.round_bar[0] = 0; sc.round_bar[1] = 0; __threadfence(); }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (leader CTA only) =====================
    if (leader && lane == 0) {
      constexpr uint32_t a_lbo = A_MN ? 8192 : 16, a_sbo = 1024, a_step = A_MN ? 2048 : 32;
      constexpr uint32_t b_lbo = B_MN ? 8192 : 16, b_sbo = 1024, b_step = B_MN ? 2048 : 32;
      int s = 0; uint32_t ph = 0;
      int acc = 0; uint32_t aph = 0;
      for (int u = cluster_id; u < sc.total; u += num_clusters) {
        const uint32_t idesc = ptx::make_idesc_bf16(BM2, u < sc.full ? BN2 : BN2 / sc.parts, A_MN, B_MN);
        ptx::mbar_wait(tempty_bar(acc), aph ^ 1);
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + acc * BN2;
        for (int kb = 0; kb < num_kb; kb++) {
          ptx::mbar_wait(full_bar(s), ph);
          ptx::tc_fence_after();
          const uint32_t sa = smem_base + s * STAGE_BYTES, sb = sa + A_BYTES;
#pragma unroll
          for (int k = 0; k < BK / UK; k++) {
            const uint64_t da = ptx::make_smem_desc(sa + k * a_step, a_lbo, a_sbo);
            const uint64_t db = ptx::make_smem_desc(sb + k * b_step, b_lbo, b_sbo);
            ptx::mma_f16_ss_2sm(d_tmem, da, db, idesc, (kb | k) != 0);
          }
          ptx::mma_commit_2sm(empty_bar(s), 3);
          if (++s == STAGES) { s = 0; ph ^= 1; }
        }
        ptx::mma_commit_2sm(tfull_bar(acc), 3);
        if (++acc == 2) { acc = 0; aph ^= 1; }
      }
    }
  } else {
    // ===================== epilogue (both CTAs, own half of the rows) =====================
    const int quarter = warp & 3;                // TMEM lanes [32*quarter, +32)
    const int chalf = (warp - 2) >> 2;           // which 128 of the 256 accumulator columns
    int acc = 0; uint32_t aph = 0;
    uint32_t ebuf = 0;
    const uint64_t pol_c = ptx::l2_policy(sc.hint_c);
    for (int u = cluster_id; u < sc.total; u += num_clusters) {
      int t, part, W;
      unit_of(sc, u, t, part, W);
      const int bi = t / tiles_per_batch;
      int mb, nb;
      tile_coords2(t - bi * tiles_per_batch, tiles_m, tiles_n, sc.group_m, mb, nb);
      epi::Args e = e0;
      if (batch > 1) epi::offset_batch(e, bi, c_bs, bias_bs);
      const int row = mb * BM2 + (int)rank * 128 + quarter * 32 + lane;
      const int n0 = nb * BN2 + part * W;
      const int c_lo = chalf * (W / 64), c_hi = (chalf + 1) * (W / 64);     // this warp's 32-column chunks of the (sub-)tile
      ptx::mbar_wait(tfull_bar(acc), aph);
      ptx::tc_fence_after();
      const uint32_t taddr = tmem_base + acc * BN2 + ((uint32_t)(quarter * 32) << 16);
      const int rrow = e.resid_row_mod > 0 ? (row % e.resid_row_mod) : row;
      if (tma_store & 4) {
        // fp32 output (+ bias), stored or ACCUMULATED (Hybrid-STOP partial sums): 32 rows x 16 columns boxes
        // through shared memory; the accumulate is a TMA reduce-add performed at the L2 instead of a row-per-thread
        // read-modify-write of C in the SM
        const int wrow0 = mb * BM2 + (int)rank * 128 + quarter * 32;
#pragma unroll 1
        for (int c = c_lo; c < c_hi; c++) {
          uint32_t r[32];
          ptx::tmem_ld_32x32(taddr + c * 32, r);
          ptx::tmem_ld_wait();
          const int col0 = n0 + c * 32;
#pragma unroll
          for (int hh = 0; hh < 2; hh++) {
            if (lane == 0) bulk_wait_read<1>();
            __syncwarp();
            const uint32_t buf = epi_base + (uint32_t)(warp - 2) * (2 * EPI_BOX_BYTES) + ebuf * EPI_BOX_BYTES;
#pragma unroll
            for (int g4 = 0; g4 < 4; g4++) {
              float v[4];
#pragma unroll
              for (int j = 0; j < 4; j++) v[j] = __uint_as_float(r[hh * 16 + g4 * 4 + j]);
              const int col = col0 + hh * 16 + g4 * 4;
              if (e.bias && col < N) {
                if (e.bias_dt == ORBIT_BF16) {
                  const uint2 raw = *reinterpret_cast<const uint2*>((const bf16*)e.bias + col);
                  const float2 b0 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&raw.x));
                  const float2 b1 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&raw.y));
                  v[0] += b0.x; v[1] += b0.y; v[2] += b1.x; v[3] += b1.y;
                } else {
                  const float4 b = *reinterpret_cast<const float4*>((const float*)e.bias + col);
                  v[0] += b.x; v[1] += b.y; v[2] += b.z; v[3] += b.w;
                }
              }
              if (e.resid && row < M && col < N) {                // residual (+ positional embedding rows): direct loads
                if (e.resid_dt == ORBIT_BF16) {
                  const uint2 raw = *reinterpret_cast<const uint2*>((const bf16*)e.resid + (size_t)rrow * e.ldr + col);
                  const float2 q0 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&raw.x));
                  const float2 q1 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&raw.y));
                  v[0] += q0.x; v[1] += q0.y; v[2] += q1.x; v[3] += q1.y;
                } else {
                  const float4 q = *reinterpret_cast<const float4*>((const float*)e.resid + (size_t)rrow * e.ldr + col);
                  v[0] += q.x; v[1] += q.y; v[2] += q.z; v[3] += q.w;
                }
              }
              const uint32_t addr = buf + lane * 64 + ((g4 ^ ((lane >> 1) & 3)) << 4);
              asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]) : "memory");
            }
            ptx::fence_proxy_async();
            __syncwarp();
            if (lane == 0) {
              if (e.accumulate) tma_reduce_add_3d(&tmC, buf, col0 + hh * 16, wrow0, bi);
              else tma_store_3d(&tmC, buf, col0 + hh * 16, wrow0, bi, pol_c);
              bulk_commit();
            }
            ebuf ^= 1;
          }
        }
      } else if (tma_store) {
        // bf16 outputs (+ bias, GELU with its pre-activation side output, GELU'): 32 x 32 boxes through shared memory,
        // written back by TMA as full 64-byte row segments (the row-per-thread direct stores below touch 32 different
        // lines per instruction, which made the K = 2048 weight-gradient GEMMs epilogue-bound)
        const int wrow0 = mb * BM2 + (int)rank * 128 + quarter * 32;
        auto stage_store = [&](const CUtensorMap* tm, const float (&v)[32], int col0) {
          if (lane == 0) bulk_wait_read<1>();            // the store issued two boxes ago has left this buffer
          __syncwarp();
          const uint32_t buf = epi_base + (uint32_t)(warp - 2) * (2 * EPI_BOX_BYTES) + ebuf * EPI_BOX_BYTES;
#pragma unroll
          for (int g8 = 0; g8 < 4; g8++) {
            uint32_t pk[4];
#pragma unroll
            for (int j = 0; j < 4; j++) {
              __nv_bfloat162 t2 = __floats2bfloat162_rn(v[g8 * 8 + 2 * j], v[g8 * 8 + 2 * j + 1]);
              pk[j] = *reinterpret_cast<uint32_t*>(&t2);
            }
            const uint32_t addr = buf + lane * 64 + ((g8 ^ ((lane >> 1) & 3)) << 4);
            asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(pk[0]), "r"(pk[1]), "r"(pk[2]), "r"(pk[3]) : "memory");
          }
          ptx::fence_proxy_async();
          __syncwarp();
          if (lane == 0) { tma_store_3d(tm, buf, col0, wrow0, bi, pol_c); bulk_commit(); }
          ebuf ^= 1;
        };
#pragma unroll 1
        for (int c = c_lo; c < c_hi; c++) {
          uint32_t r[32];
          ptx::tmem_ld_32x32(taddr + c * 32, r);
          ptx::tmem_ld_wait();
          const int col0 = n0 + c * 32;
          float v[32];
#pragma unroll
          for (int g8 = 0; g8 < 4; g8++) {
#pragma unroll
            for (int j = 0; j < 8; j++) v[g8 * 8 + j] = __uint_as_float(r[g8 * 8 + j]);
            if (e.bias && col0 + g8 * 8 < N) {
              float b[8];
              epi::load8(e.bias, col0 + g8 * 8, e.bias_dt, b);
#pragma unroll
              for (int j = 0; j < 8; j++) v[g8 * 8 + j] += b[j];
            }
          }
          if (e.act == ACT_GELU) {
            if (tma_store & 2) {                                  // pre-activation u (bf16); g = GELU(bf16(u)) (reading R25)
              stage_store(&tmX, v, col0);
#pragma unroll
              for (int j = 0; j < 32; j++) v[j] = __bfloat162float(__float2bfloat16_rn(v[j]));
            }
#pragma unroll
            for (int j = 0; j < 32; j++) v[j] = gelu_f(v[j]);
          } else if (e.act == ACT_GELU_GRAD) {
            if (row < M) {
#pragma unroll
              for (int g8 = 0; g8 < 4; g8++) {
                if (col0 + g8 * 8 < N) {
                  float u[8];
                  epi::load8(e.aux_in, (size_t)row * e.ld_aux + col0 + g8 * 8, e.aux_dt, u);
#pragma unroll
                  for (int j = 0; j < 8; j++) v[g8 * 8 + j] *= gelu_grad_f(u[j]);
                }
              }
            }
          }
          if (e.resid && row < M) {
#pragma unroll
            for (int g8 = 0; g8 < 4; g8++) {
              if (col0 + g8 * 8 < N) {
                float q[8];
                epi::load8(e.resid, (size_t)rrow * e.ldr + col0 + g8 * 8, e.resid_dt, q);
#pragma unroll
                for (int j = 0; j < 8; j++) v[g8 * 8 + j] += q[j];
              }
            }
          }
          stage_store(&tmC, v, col0);
        }
      } else {
#pragma unroll 1
      for (int c = c_lo; c < c_hi; c++) {
        uint32_t r[32];
        ptx::tmem_ld_32x32(taddr + c * 32, r);
        ptx::tmem_ld_wait();
        if (row < M) epi::chunk32(e, r, row, rrow, n0 + c * 32, N);
      }
      }
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive_cluster(ptx::mapa(tempty_bar(acc), 0));
      if (++acc == 2) { acc = 0; aph ^= 1; }
    }
    if (tma_store && lane == 0) bulk_wait_all();   // the staging buffers (and the writes) outlive the last store
  }
  ptx::tc_fence_before();
  ptx::cluster_sync_all();                       // peer smem / barriers stay alive until both CTAs are done
  if (warp == 1) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc_2sm(tmem_base, TMEM_COLS);
  }
}

// A/B switches of the schedule (read once; profiles/r2_gemm_schedule.md): ORBIT_GEMM_TAIL_SPLIT=0 keeps whole tiles in
// the last round; ORBIT_GEMM_GROUP_M=<n> forces the raster group height; ORBIT_GEMM_L2HINT=<bits> selects the L2 eviction
// hints (default 1).
bool tail_split_enabled() {
  static const int v = [] { const char* e = getenv("ORBIT_GEMM_TAIL_SPLIT"); return (e && e[0] == '0') ? 0 : 1; }();
  return v != 0;
}
double round_sync_min_bytes() {
  static const double v = [] { const char* e = getenv("ORBIT_GEMM_ROUND_SYNC_MINMB"); return (e ? atof(e) : 256.0) * 1e6; }();
  return v;
}
bool round_sync_enabled() {
  static const int v = [] { const char* e = getenv("ORBIT_GEMM_ROUND_SYNC"); return (e && e[0] == '0') ? 0 : 1; }();
  return v != 0;
}
int l2_hint_mode() {
  static const int v = [] { const char* e = getenv("ORBIT_GEMM_L2HINT"); return e ? atoi(e) : 1; }();
  return v;
}
int raster_group_m(int tiles_m, int M, int K) {
  static const int forced = [] { const char* e = getenv("ORBIT_GEMM_GROUP_M"); return e ? atoi(e) : 0; }();
  if (forced > 0) return forced < tiles_m ? forced : tiles_m;
  (void)M; (void)K;
  return 8 < tiles_m ? 8 : tiles_m;
}

template <int A_MN, int B_MN>
int launch2(const CUtensorMap& ma, const CUtensorMap& mb, const CUtensorMap* mc, const CUtensorMap* mx, const GemmArgs& g, int sms,
            cudaStream_t s) {
  const epi::Args e = epi::from_gemm(g);
  const int M = g.M, N = g.N, K = g.K, batch = g.batch > 1 ? g.batch : 1;
  ORBIT_SMEM_ATTR((gemm_tc2_kernel<A_MN, B_MN>), SMEM_BYTES);
  const int tiles_m = cdiv(M, BM2);
  const long long tiles = (long long)tiles_m * cdiv(N, BN2) * batch;
  int clusters = sms / 2;
  if (tiles < clusters) clusters = (int)tiles;
  Sched sc;
  // last partial round: split its tiles into two 256 x 128 sub-tiles when they then still fit one round
  const int rem = (int)(tiles % clusters);
  sc.parts = (rem > 0 && 2 * rem <= clusters && tiles > clusters && tail_split_enabled()) ? 2 : 1;
  sc.full = sc.parts > 1 ? (int)(tiles - rem) : (int)tiles;
  sc.total = sc.full + (sc.parts > 1 ? rem * sc.parts : 0);
  sc.group_m = raster_group_m(tiles_m, M, K);
  // L2 policy (A/B on one box, profiles/r2_gemm_schedule.md): evict_last on the SMALLER operand (the activation panel every
  // round re-reads: C5 fc1 needs its 50 MB `a` in all 21 rounds while 1.2 GB of weights stream through the L2) is worth
  // ~1 % of the C5 step; evict_first on the larger operand RAISES the DRAM traffic (27 -> 37 GB per step: the clusters that
  // share a panel inside a round then miss it) and evict_first on large outputs changes nothing; both stay off.
  sc.hint_a = sc.hint_b = sc.hint_c = 0;
  const int hm = l2_hint_mode();                // bit 0: smaller operand evict_last; bit 1: large outputs evict_first; bit 2: larger operand evict_first
  if (hm) {
    const double bytes_a = 2.0 * M * K * batch, bytes_b = 2.0 * N * K * batch, bytes_c = (double)dsize(g.out_dtype) * M * N * batch;
    const double small = bytes_a < bytes_b ? bytes_a : bytes_b, big = bytes_a < bytes_b ? bytes_b : bytes_a;
    if (small <= 80e6 && big > 100e6) {
      if (hm & 1) (bytes_a < bytes_b ? sc.hint_a : sc.hint_b) = 2;
      if (hm & 4) (bytes_a < bytes_b ? sc.hint_b : sc.hint_a) = 1;
    }
    if ((hm & 2) && bytes_c > 100e6) sc.hint_c = 1;
  }
  sc.round_bar = nullptr;
  // only where the operands cannot stay in the 126 MB L2 anyway (C5: 1.2-1.4 GB per GEMM); at C3 / C4 sizes (< 70 MB per GEMM) the
  // panels are L2-resident whatever the skew and the meeting costs 1-2 % of the step
  if (round_sync_enabled() && tiles > 2 * clusters && 2.0 * K * ((double)M + N) * batch >= round_sync_min_bytes()) {
    static std::atomic<unsigned int> next_slot{0};
    static std::atomic<unsigned int*> base_c{nullptr};
    unsigned int* base = base_c.load(std::memory_order_relaxed);
    if (!base) { ORBIT_CUDA_CHECK(cudaGetSymbolAddress((void**)&base, g_round_bar)); base_c.store(base, std::memory_order_relaxed); }
    sc.round_bar = base + 2 * (next_slot.fetch_add(1) % 64);      // zero on entry: static storage, then reset by the last cluster out
  }
  ORBIT_CUDA_CHECK(launch_pdl(gemm_tc2_kernel<A_MN, B_MN>, dim3(2 * clusters), dim3(NTHREADS), SMEM_BYTES, s, ma, mb, mc ? *mc : ma,
                              mx ? *mx : ma, (mc ? (g.out_dtype == ORBIT_F32 ? 4 : 1) : 0) | (mx ? 2 : 0), e, M, N, K, batch, g.c_bs,
                              g.bias_bs, sc));
  return ORBIT_OK;
}
}  // namespace

// called by gemm_tc() (gemm_tc.cu), which builds the tensor maps: A boxes as in the 1-CTA kernel, B boxes with
// 128 rows (K-major) or 64 x 64 (N-major)
// mc / mx: tensor maps of C / of the GELU pre-activation side output for the TMA-store epilogue (32 x 32 bf16 boxes, 64B
// swizzle), or null for direct stores
int gemm_tc2_launch(const CUtensorMap& ma, const CUtensorMap& mb, const CUtensorMap* mc, const CUtensorMap* mx, const GemmArgs& g,
                    bool a_mn, bool b_mn, int sms, cudaStream_t s) {
  if (!a_mn && b_mn) return launch2<0, 1>(ma, mb, mc, mx, g, sms, s);
  if (!a_mn && !b_mn) return launch2<0, 0>(ma, mb, mc, mx, g, sms, s);
  if (a_mn && b_mn) return launch2<1, 1>(ma, mb, mc, mx, g, sms, s);
  return launch2<1, 0>(ma, mb, mc, mx, g, sms, s);
}

}  // namespace orbit
