// aggregate_tc.cu -- tensor-core versions of the per-patch aggregation kernels (a2 / a2'; collapsed
// form of DESIGN.md §4).  bf16 storage, heads <= 16, V <= 128, D % 64 == 0.
//
// A CTA streams one patch's token tile X [V x D] through shared memory in D-chunks (TMA box copies into a ring of
// mbarrier-guarded stages, 128-byte swizzle) and runs the small products on mma.sync.m16n8k16 (bf16 in, fp32 accumulate):
//   forward : S = X Ut^T  (scores, [V x h])  -> warp softmax over V -> Xbar = alpha^T X  ([h x D])
//   backward: dA = X dXbar^T ([V x h]) -> ds -> dX = [alpha | ds] [dXbar ; Ut]  ([V x D]),  dUt^T += ds^T X
// X is read twice per direction (second pass mostly from L2); everything else is tiny.  This makes the kernels
// HBM/L2-bound instead of fp32-ALU-bound (2*heads .. 4*heads FMA per token element on CUDA cores).
#include <cuda.h>
#include <atomic>
#include "frontend.cuh"
#include "ptx.cuh"

namespace orbit {
namespace {
using namespace ptx;

constexpr int NT = 256;            // 8 warps
constexpr int VP_MAX = 128;
constexpr int HP = 16;             // heads padded to 16

__device__ __forceinline__ uint32_t s_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void ldsm4(uint32_t addr, uint32_t* r) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void ldsm4t(uint32_t addr, uint32_t* r) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void mma16816(float* c, const uint32_t* a, uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}

// bf16 tile with rows of DC elements (DC*2 bytes, a multiple of 128), 16-byte chunks XOR-swizzled with (row & 7)
template <int DC>
struct Tl {
  static constexpr int CH = DC / 8;
  static constexpr int ROWB = DC * 2;
  __device__ static __forceinline__ uint32_t addr(uint32_t base, int row, int chunk) {
    return base + row * ROWB + ((chunk ^ (row & 7)) << 4);
  }
  // B(k, n) = T[k][n]: 16 k from k0, 8 n from n0 -> r[0..1]
  __device__ static __forceinline__ void ldB_nmajor8(uint32_t base, int k0, int n0, uint32_t* r) {
    int lane = threadIdx.x & 31;
    asm volatile("ldmatrix.sync.aligned.m8n8.x2.trans.shared.b16 {%0,%1}, [%2];"
                 : "=r"(r[0]), "=r"(r[1]) : "r"(addr(base, k0 + (lane & 7) + ((lane >> 3) & 1) * 8, n0 >> 3)));
  }
  __device__ static __forceinline__ void ldA(uint32_t base, int r0, int k0, uint32_t* a) {
    int lane = threadIdx.x & 31;
    ldsm4(addr(base, r0 + (lane & 7) + ((lane >> 3) & 1) * 8, (k0 >> 3) + (lane >> 4)), a);
  }
  // B(k, n) = T[n][k]: 16 n from n0, 16 k from k0 -> r[0..1] n-tile n0, r[2..3] n-tile n0+8
  __device__ static __forceinline__ void ldB_kmajor(uint32_t base, int n0, int k0, uint32_t* r) {
    int lane = threadIdx.x & 31;
    ldsm4(addr(base, n0 + (lane & 7) + (lane >> 4) * 8, (k0 >> 3) + ((lane >> 3) & 1)), r);
  }
  // B(k, n) = T[k][n]: 16 k from k0, 16 n from n0
  __device__ static __forceinline__ void ldB_nmajor(uint32_t base, int k0, int n0, uint32_t* r) {
    int lane = threadIdx.x & 31;
    ldsm4t(addr(base, k0 + (lane & 7) + ((lane >> 3) & 1) * 8, (n0 >> 3) + (lane >> 4)), r);
  }
};

// small un-swizzled bf16 matrix in smem with padded rows (ROWB bytes): A fragments (16 rows from r0, 16 k from k0)
__device__ __forceinline__ void ldA_plain(uint32_t base, int rowb, int r0, int k0, uint32_t* a) {
  int lane = threadIdx.x & 31;
  ldsm4(base + (r0 + (lane & 7) + ((lane >> 3) & 1) * 8) * rowb + (k0 + (lane >> 4) * 8) * 2, a);
}

// scores-like product: acc[2][4] (16 rows of this warp x 16 heads) += Xc[rows, :] * Bc[0..15, :]^T over one chunk
template <int DC>
__device__ __forceinline__ void chunk_scores(float (*acc)[4], uint32_t xc, int r0, uint32_t bc) {
#pragma unroll
  for (int ks = 0; ks < DC / 16; ks++) {
    uint32_t a[4], b[4];
    Tl<DC>::ldA(xc, r0, ks * 16, a);
    Tl<DC>::ldB_kmajor(bc, 0, ks * 16, b);
    mma16816(acc[0], a, b[0], b[1]);
    mma16816(acc[1], a, b[2], b[3]);
  }
}

constexpr int SROW = HP + 1;   // fp32 score matrix row stride (floats)

// Both kernels stream their operands with TMA (cp.async.bulk.tensor, 128-byte swizzle = the XOR layout of Tl<64>): one
// thread issues a few box copies per step instead of every thread issuing ~10 cp.async with their address arithmetic
// (which was ~2/3 of the instructions of the cp.async versions; ncu: issue-bound at 2 warps per scheduler, not
// HBM-bound).  The chunks of all patches of a CTA form ONE stream (n = patch_iter * 2 nch + i) through an STG-deep ring
// of mbarrier-guarded stages, so the ring stays full across the softmax phase and across patch boundaries.
// Box rows = V exactly (the next patch's rows must not land in the tile); tile rows V..Vp-1 are zeroed once.
constexpr int TB = 64;                       // columns per TMA box / smem sub-tile (128 bytes: one swizzle span)
constexpr int XT = VP_MAX * TB * 2;          // bytes of an X sub-tile   (16 KB)
constexpr int UT = HP * TB * 2;              // bytes of a [16 x 64] sub-tile (2 KB)

__device__ __forceinline__ void zero_tail_rows(uint8_t* tile, int r0, int r1, int nthreads) {
  for (int i = r0 * 8 + threadIdx.x; i < r1 * 8; i += nthreads) reinterpret_cast<uint4*>(tile)[i] = make_uint4(0, 0, 0, 0);
}

// ============================================ forward ============================================
// A step is NSUB = 2 sub-tiles (128 columns); 16 warps = two groups of 8, group wh works on sub-tile wh.  Pass 1: warp
// (wh, wt < mtiles) accumulates the scores of its 16 rows over its sub-tiles (the two groups' halves are summed through
// shared memory).  Pass 2: warp (wh, wt) owns 8 columns of sub-tile wh.
constexpr int NTF = 512;                    // consumer threads; warp 16 is the TMA producer
__device__ __forceinline__ void consumer_sync() { asm volatile("bar.sync 1, 512;" ::: "memory"); }
template <int STG>
__global__ void __launch_bounds__(NTF + 32) agg_fwd_tma_kernel(const __grid_constant__ CUtensorMap tmX,
    const __grid_constant__ CUtensorMap tmU, float* __restrict__ alpha, bf16* __restrict__ Xbar, int BL, int V, int D, int h) {
  constexpr int NSUB = 2;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = smem_raw + ((1024 - (s_u32(smem_raw) & 1023)) & 1023);
  const int Vp = (V + 15) & ~15;
  const uint32_t sX = s_u32(smem), sU = sX + STG * NSUB * XT;               // [STG][NSUB] tiles each
  uint8_t* rest = smem + STG * NSUB * (XT + UT);
  float* sS = reinterpret_cast<float*>(rest);                               // [VP_MAX][SROW]
  bf16* sAT = reinterpret_cast<bf16*>(sS + VP_MAX * SROW);                  // alpha^T [HP][ATROW]
  constexpr int ATROW = VP_MAX + 8;
  const uint32_t sATu = s_u32(sAT);
  const uint32_t bar0 = s_u32(sAT + HP * ATROW), ebar0 = bar0 + 8 * STG;    // full[STG], empty[STG]
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int wt = warp & 7, wh = warp >> 3;
  const int nch = D / (TB * NSUB), mtiles = Vp / 16;

  for (int j = 0; j < STG * NSUB; j++) zero_tail_rows(smem + j * XT, V, Vp, NTF + 32);
  if (threadIdx.x == 0) {
    for (int i = 0; i < STG; i++) { mbar_init(bar0 + 8 * i, 1); mbar_init(ebar0 + 8 * i, NTF / 32); }
    fence_barrier_init();
  }
  fence_proxy_async();
  __syncthreads();

  const int npat = blockIdx.x < BL ? (BL - 1 - blockIdx.x) / gridDim.x + 1 : 0;
  const int per = 2 * nch, total = npat * per;
  auto issue = [&](int n) {             // producer lane: n-th step of this CTA: pass 1 (scores) then pass 2 (Xbar) of each patch
    const int pi = n / per, i = n - pi * per, c = i < nch ? i : per - 1 - i, st = n % STG;   // pass 2 walks back
    const int row0 = (blockIdx.x + pi * gridDim.x) * V;
    const uint32_t bar = bar0 + 8 * st;
    mbar_expect_tx(bar, NSUB * (V * TB * 2 + (i < nch ? UT : 0)));
#pragma unroll
    for (int j = 0; j < NSUB; j++) {
      tma_load_2d(sX + (st * NSUB + j) * XT, &tmX, bar, (c * NSUB + j) * TB, row0);
      if (i < nch) tma_load_2d(sU + (st * NSUB + j) * UT, &tmU, bar, (c * NSUB + j) * TB, 0);
    }
  };
  // Producer warp: refills a stage as soon as all 16 consumer warps have released it (empty[st]); inside a pass the
  // consumer warps never meet at a CTA barrier.
  if (warp == NTF / 32) {
    if (lane == 0)
      for (int n = 0; n < total; n++) {
        if (n >= STG) mbar_wait(ebar0 + 8 * (n % STG), ((n / STG) + 1) & 1);
        issue(n);
      }
    return;
  }

  for (int pi = 0; pi < npat; pi++) {
    const int bl = blockIdx.x + pi * gridDim.x, n0 = pi * per;
    float acc[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
    // ---- pass 1: S[v, a] = X_v . Ut[a, :]
    for (int i = 0; i < nch; i++) {
      const int n = n0 + i, st = n % STG;
      mbar_wait(bar0 + 8 * st, (n / STG) & 1);
      if (wt < mtiles) chunk_scores<TB>(acc, sX + (st * NSUB + wh) * XT, wt * 16, sU + (st * NSUB + wh) * UT);
      __syncwarp();
      if (lane == 0) mbar_arrive(ebar0 + 8 * st);
    }
    consumer_sync();                    // the previous patch's pass 2 is finished everywhere: sS / sAT may be rewritten
    if (wt < mtiles && wh == 0) {
#pragma unroll
      for (int nt = 0; nt < 2; nt++) {
        int r = wt * 16 + g, c = nt * 8 + 2 * t;
        sS[r * SROW + c] = acc[nt][0]; sS[r * SROW + c + 1] = acc[nt][1];
        sS[(r + 8) * SROW + c] = acc[nt][2]; sS[(r + 8) * SROW + c + 1] = acc[nt][3];
      }
    }
    consumer_sync();
    if (wt < mtiles && wh == 1) {
#pragma unroll
      for (int nt = 0; nt < 2; nt++) {
        int r = wt * 16 + g, c = nt * 8 + 2 * t;
        sS[r * SROW + c] += acc[nt][0]; sS[r * SROW + c + 1] += acc[nt][1];
        sS[(r + 8) * SROW + c] += acc[nt][2]; sS[(r + 8) * SROW + c + 1] += acc[nt][3];
      }
    }
    consumer_sync();
    // ---- softmax over v per head; alpha -> global (fp32) and alpha^T (bf16) -> smem
    for (int a = warp; a < HP; a += NTF / 32) {
      if (a < h) {
        float m = -INFINITY;
        for (int v = lane; v < V; v += 32) m = fmaxf(m, sS[v * SROW + a]);
        m = warp_max(m);
        float l = 0.f;
        for (int v = lane; v < V; v += 32) l += __expf(sS[v * SROW + a] - m);
        l = warp_sum(l);
        const float inv = 1.f / l;
        for (int v = lane; v < Vp; v += 32) {
          float p = v < V ? __expf(sS[v * SROW + a] - m) * inv : 0.f;
          if (v < V) alpha[((size_t)bl * h + a) * V + v] = p;
          sAT[a * ATROW + v] = __float2bfloat16_rn(p);
        }
      } else {
        for (int v = lane; v < Vp; v += 32) sAT[a * ATROW + v] = __float2bfloat16_rn(0.f);
      }
    }
    consumer_sync();
    // ---- pass 2: Xbar[a, d] = sum_v alpha[v, a] X[v, d]
    uint32_t af[VP_MAX / 16][4];
#pragma unroll
    for (int ks = 0; ks < VP_MAX / 16; ks++)
      if (ks < mtiles) ldA_plain(sATu, ATROW * 2, 0, ks * 16, af[ks]);
    for (int i = nch; i < 2 * nch; i++) {
      const int n = n0 + i, st = n % STG;
      mbar_wait(bar0 + 8 * st, (n / STG) & 1);
      const uint32_t xc = sX + (st * NSUB + wh) * XT;
      float o[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};      // two accumulation chains (even / odd k-steps)
#pragma unroll
      for (int ks = 0; ks < VP_MAX / 16; ks++) {
        if (ks < mtiles) {
          uint32_t b[2];
          Tl<TB>::ldB_nmajor8(xc, ks * 16, wt * 8, b);
          mma16816(o[ks & 1], af[ks], b[0], b[1]);
        }
      }
      const int d = (per - 1 - i) * (TB * NSUB) + wh * TB + wt * 8 + 2 * t;   // pass 2 runs from the last chunk back (L2 reuse distance)
      if (g < h) __stcs(reinterpret_cast<uint32_t*>(Xbar + ((size_t)bl * h + g) * D + d), pack_bf16(o[0][0] + o[1][0], o[0][1] + o[1][1]));
      if (g + 8 < h) __stcs(reinterpret_cast<uint32_t*>(Xbar + ((size_t)bl * h + g + 8) * D + d), pack_bf16(o[0][2] + o[1][2], o[0][3] + o[1][3]));
      __syncwarp();
      if (lane == 0) mbar_arrive(ebar0 + 8 * st);
    }
  }
}

// ============================================ backward ============================================
// 16 warps, one 64-column sub-tile per step (the [HP][D] fp32 dUt accumulator takes most of the shared memory).  Pass 1:
// warp w takes row tile (w & 7) and k half (w >> 3) of the chunk; pass 2: warps 0-7 produce dX (one 16-row tile each)
// while warps 8-15 accumulate dUt^T (one 8-column group of the chunk each).  dX leaves through a per-warp XOR-swizzled
// staging tile (aliasing the dalpha / alpha score buffers, dead in pass 2) as 16-byte pieces, 128 contiguous bytes of a
// token row per 8 lanes, instead of 4-byte pieces of 16 rows.
constexpr int NTB = 512;                    // consumer threads; warp 16 is the TMA producer
constexpr int TMEM_ACC_COLS = 512;          // dUt^T accumulator: 2 warps per lane quarter x (D / 64 chunks) x 4 columns -> D <= 4096
constexpr int BT = 2 * UT;                   // B tile: rows 0-15 dXbar chunk, 16-31 Ut chunk
template <int STG>
__global__ void __launch_bounds__(NTB + 32) agg_bwd_tma_kernel(const __grid_constant__ CUtensorMap tmX,
    const __grid_constant__ CUtensorMap tmG, const __grid_constant__ CUtensorMap tmU,
    const float* __restrict__ alpha, bf16* __restrict__ dtok, float* __restrict__ dUt_acc, int BL, int V, int D, int h) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = smem_raw + ((1024 - (s_u32(smem_raw) & 1023)) & 1023);
  const int Vp = (V + 15) & ~15;
  const int XTb = Vp * TB * 2;                                                // X tile sized for this V: more stages fit
  const uint32_t sX = s_u32(smem), sB = sX + STG * XTb;
  float* sS = reinterpret_cast<float*>(smem + STG * (XTb + BT));             // [Vp][SROW] dalpha
  float* sAl = sS + Vp * SROW;                                                // [Vp][SROW] alpha
  bf16* sAD = reinterpret_cast<bf16*>(sAl + Vp * SROW);                      // [Vp][ADROW]  (alpha | ds)
  constexpr int ADROW = 2 * HP + 8;
  bf16* sDT = sAD + Vp * ADROW;                                              // ds^T [HP][DTROW]
  constexpr int DTROW = VP_MAX + 8;
  // The block-private dUt^T accumulator [HP][D] fp32 (131 KB at D = 2048) lives in TENSOR MEMORY, not in shared memory: every
  // thread of the 8 accumulating warps owns 4 values per 64-column chunk, kept in 4 columns of its own TMEM lane (tcgen05.ld /
  // add / tcgen05.st, no hazards: nobody else touches the cell).  The shared memory it occupied now holds a 12-stage ring
  // instead of 4 stages: the kernel was bound by the mbarrier waits of the shallow ring (3.6 TB/s of DRAM traffic).
  const uint32_t tslot = s_u32(sDT + HP * DTROW);                             // TMEM base address word (+ padding to 16 bytes)
  const uint32_t bar0 = tslot + 16, ebar0 = bar0 + 8 * STG;                   // full[STG], empty[STG]
  const uint32_t sADu = s_u32(sAD), sDTu = s_u32(sDT);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int wt = warp & 7, wh = warp >> 3;
  const int nch = D / TB, mtiles = Vp / 16;
  uint8_t* sO = reinterpret_cast<uint8_t*>(sS) + wt * (16 * 128);            // [16][64] bf16, swizzled: 2 KB per dX warp (wt < mtiles)
  static_assert(16 * 128 <= 2 * 16 * SROW * 4, "staging tiles (2 KB per 16 rows) must fit in the score buffers (2 x 16 x SROW floats)");

  if (warp == 0) { tmem_alloc(tslot, TMEM_ACC_COLS); tmem_relinquish(); }
  for (int j = 0; j < STG; j++) {
    zero_tail_rows(smem + j * XTb, V, Vp, NTB + 32);
    zero_tail_rows(smem + STG * XTb + j * BT, h, HP, NTB + 32);
  }
  if (threadIdx.x == 0) {
    for (int i = 0; i < STG; i++) { mbar_init(bar0 + 8 * i, 1); mbar_init(ebar0 + 8 * i, NTB / 32); }
    fence_barrier_init();
  }
  fence_proxy_async();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tacc;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tacc) : "r"(tslot));
  const uint32_t tacc0 = tacc;
  // this thread's accumulator cells: lane = its lane in the warp's TMEM quarter, 4 columns per chunk, the two warps of a quarter
  // (wt and wt + 4) side by side
  tacc += ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)(wt >> 2) * (TMEM_ACC_COLS / 2);

  const int npat = blockIdx.x < BL ? (BL - 1 - blockIdx.x) / gridDim.x + 1 : 0;
  const int per = 2 * nch, total = npat * per;
  auto issue = [&](int n) {             // producer lane
    const int pi = n / per, i = n - pi * per, c = i < nch ? i : per - 1 - i, st = n % STG;
    const int bl = blockIdx.x + pi * gridDim.x;
    const uint32_t bar = bar0 + 8 * st;
    mbar_expect_tx(bar, (V + h) * TB * 2 + (i >= nch ? UT : 0));
    tma_load_2d(sX + st * XTb, &tmX, bar, c * TB, bl * V);
    tma_load_2d(sB + st * BT, &tmG, bar, c * TB, bl * h);
    if (i >= nch) tma_load_2d(sB + st * BT + UT, &tmU, bar, c * TB, 0);
  };
  // Producer warp: refills a stage as soon as all 16 consumer warps have released it (empty[st]); the consumers never
  // synchronise with each other inside a pass, so warps drift apart and the per-step CTA barrier is gone.
  if (warp == NTB / 32) {
    if (lane == 0)
      for (int n = 0; n < total; n++) {
        if (n >= STG) mbar_wait(ebar0 + 8 * (n % STG), ((n / STG) + 1) & 1);
        issue(n);
      }
    return;
  }

  for (int pi = 0; pi < npat; pi++) {
    const int bl = blockIdx.x + pi * gridDim.x, n0 = pi * per;
    float acc[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
    consumer_sync();                    // previous patch finished with the score / staging buffers
    for (int i = threadIdx.x; i < Vp * HP; i += NTB) {
      int v = i / HP, a = i - v * HP;
      sAl[v * SROW + a] = (v < V && a < h) ? alpha[((size_t)bl * h + a) * V + v] : 0.f;
    }
    // ---- pass 1: dalpha[v, a] = X_v . dXbar[a, :]   (k half wh of every chunk)
    for (int i = 0; i < nch; i++) {
      const int n = n0 + i, st = n % STG;
      mbar_wait(bar0 + 8 * st, (n / STG) & 1);
      if (wt < mtiles) {
        const uint32_t xc = sX + st * XTb, bc = sB + st * BT;
#pragma unroll
        for (int ks = 0; ks < TB / 32; ks++) {
          uint32_t a[4], b[4];
          Tl<TB>::ldA(xc, wt * 16, (wh * (TB / 32) + ks) * 16, a);
          Tl<TB>::ldB_kmajor(bc, 0, (wh * (TB / 32) + ks) * 16, b);
          mma16816(acc[0], a, b[0], b[1]);
          mma16816(acc[1], a, b[2], b[3]);
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(ebar0 + 8 * st);
    }
    if (wt < mtiles && wh == 0) {
#pragma unroll
      for (int nt = 0; nt < 2; nt++) {
        int r = wt * 16 + g, c = nt * 8 + 2 * t;
        sS[r * SROW + c] = acc[nt][0]; sS[r * SROW + c + 1] = acc[nt][1];
        sS[(r + 8) * SROW + c] = acc[nt][2]; sS[(r + 8) * SROW + c + 1] = acc[nt][3];
      }
    }
    consumer_sync();
    if (wt < mtiles && wh == 1) {
#pragma unroll
      for (int nt = 0; nt < 2; nt++) {
        int r = wt * 16 + g, c = nt * 8 + 2 * t;
        sS[r * SROW + c] += acc[nt][0]; sS[r * SROW + c + 1] += acc[nt][1];
        sS[(r + 8) * SROW + c] += acc[nt][2]; sS[(r + 8) * SROW + c + 1] += acc[nt][3];
      }
    }
    consumer_sync();
    // ---- ds[v, a] = alpha (dalpha - sum_w alpha_w dalpha_w); A operands (alpha | ds) and ds^T in bf16
    for (int a = warp; a < HP; a += NTB / 32) {
      float dot = 0.f;
      for (int v = lane; v < V; v += 32) dot += sAl[v * SROW + a] * sS[v * SROW + a];
      dot = warp_sum(dot);
      for (int v = lane; v < Vp; v += 32) {
        float al = sAl[v * SROW + a];
        float ds = al * (sS[v * SROW + a] - dot);
        sAD[v * ADROW + a] = __float2bfloat16_rn(al);
        sAD[v * ADROW + HP + a] = __float2bfloat16_rn(ds);
        sDT[a * DTROW + v] = __float2bfloat16_rn(ds);
      }
    }
    consumer_sync();
    uint32_t adf[2][4];                 // this warp's 16 rows of (alpha | ds): K = 32 -> 2 k-steps
    if (wh == 0 && wt < mtiles) {
      ldA_plain(sADu, ADROW * 2, wt * 16, 0, adf[0]);
      ldA_plain(sADu, ADROW * 2, wt * 16, 16, adf[1]);
    }
    // ---- pass 2: dX chunk = (alpha | ds) [dXbar ; Ut] chunk;  dUt^T chunk += ds^T X chunk
    for (int i = nch; i < 2 * nch; i++) {
      const int n = n0 + i, st = n % STG;
      mbar_wait(bar0 + 8 * st, (n / STG) & 1);
      const uint32_t xc = sX + st * XTb, bc = sB + st * BT;
      const int c0 = (per - 1 - i) * TB;   // pass 2 runs from the last chunk back: most recently read lines first (L2)
      if (wh == 0) {
        if (wt < mtiles) {
#pragma unroll
          for (int np = 0; np < TB / 16; np++) {
            float o[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
#pragma unroll
            for (int ks = 0; ks < 2; ks++) {
              uint32_t b[4];
              Tl<TB>::ldB_nmajor(bc, ks * 16, np * 16, b);
              mma16816(o[0], adf[ks], b[0], b[1]);
              mma16816(o[1], adf[ks], b[2], b[3]);
            }
#pragma unroll
            for (int nt = 0; nt < 2; nt++) {
              const int ch = np * 2 + nt;                 // 16-byte chunk of the 128-byte staging row
              *reinterpret_cast<uint32_t*>(sO + g * 128 + ((ch ^ g) << 4) + t * 4) = pack_bf16(o[nt][0], o[nt][1]);
              *reinterpret_cast<uint32_t*>(sO + (g + 8) * 128 + ((ch ^ g) << 4) + t * 4) = pack_bf16(o[nt][2], o[nt][3]);
            }
          }
          __syncwarp();
#pragma unroll
          for (int q = 0; q < 4; q++) {
            const int row = q * 4 + (lane >> 3), ch = lane & 7, r = wt * 16 + row;
            if (r < V)
              __stcs(reinterpret_cast<uint4*>(dtok + ((size_t)bl * V + r) * D + c0 + ch * 8),   // streaming: keep X in L2
                     *reinterpret_cast<const uint4*>(sO + row * 128 + ((ch ^ (row & 7)) << 4)));
          }
        }
      } else {
        // dUt^T[a, c0 + 8 wt ...] += sum_v ds[v, a] X[v, ...]
        float o[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int ks = 0; ks < VP_MAX / 16; ks++) {
          if (ks < mtiles) {
            uint32_t a[4], b[2];
            ldA_plain(sDTu, DTROW * 2, 0, ks * 16, a);
            Tl<TB>::ldB_nmajor8(xc, ks * 16, wt * 8, b);
            mma16816(o, a, b[0], b[1]);
          }
        }
        // o[0..3] = (head g, columns d, d + 1), (head g + 8, d, d + 1) with d = c0 + 8 wt + 2 t: added to this thread's 4 TMEM cells of the chunk
        const uint32_t cell = tacc + (uint32_t)(c0 / TB) * 4;
        uint32_t av[4];
        if (pi == 0) {
#pragma unroll
          for (int q = 0; q < 4; q++) av[q] = __float_as_uint(o[q]);
        } else {
          tmem_st_wait();                // this thread's store to the cell (previous patch) has completed
          tmem_ld_32x4(cell, av);
          tmem_ld_wait();
#pragma unroll
          for (int q = 0; q < 4; q++) av[q] = __float_as_uint(__uint_as_float(av[q]) + o[q]);
        }
        tmem_st_32x4(cell, av);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(ebar0 + 8 * st);
    }
  }
  if (wh == 1 && npat > 0) {            // flush this thread's cells: one pass over the chunks
    tmem_st_wait();
    for (int c = 0; c < nch; c++) {
      uint32_t av[4];
      tmem_ld_32x4(tacc + (uint32_t)c * 4, av);
      tmem_ld_wait();
      const int d = c * TB + wt * 8 + 2 * t;
      if (g < h) {
        atomicAdd(dUt_acc + (size_t)d * h + g, __uint_as_float(av[0]));
        atomicAdd(dUt_acc + (size_t)(d + 1) * h + g, __uint_as_float(av[1]));
      }
      if (g + 8 < h) {
        atomicAdd(dUt_acc + (size_t)d * h + g + 8, __uint_as_float(av[2]));
        atomicAdd(dUt_acc + (size_t)(d + 1) * h + g + 8, __uint_as_float(av[3]));
      }
    }
  }
  tc_fence_before();
  consumer_sync();
  if (warp == 0) { tc_fence_after(); tmem_dealloc(tacc0, TMEM_ACC_COLS); }
}

// ============================================ forward on tcgen05 ============================================
// ncu of the mma.sync forward above (config 3): no unit is busy (DRAM 60 %, L2 54 %, issue slots 31 %); the 16 consumer warps
// spend ~3/4 of their time in the ldmatrix -> HMMA -> store chains of a step (short-scoreboard / fixed-latency stalls) and only
// 22 % waiting for data: a latency-bound consumer loop, ~1000 cycles per 128-column step.  (A variant that kept a patch's tile
// resident across a 4- or 8-CTA cluster, exchanging the partial scores through distributed shared memory, read X once but was
// 2.6x / 6.6x slower: 1.5k cycles per release-arrive on a peer's mbarrier, 5k per round of remote loads, per patch.)
// Here the two products run on the 5th-generation tensor cores straight from the TMA tiles, issued by one thread:
//   pass 1: S[v, a]   (TMEM, 128 lanes x 16 columns)  = sum over the chunks of  X[128 x 64] (A, K-major) . Ut[16 x 64]^T (B, K-major)
//   pass 2: Xbar[a, d] (TMEM, lanes 0..15 of 128 x 128 columns, double buffered) = alpha^T[128 x V] (A, K-major, rows >= 16 zero) . X[V x 128 d] (B, MN-major: the same tiles)
//           (X^T as an MN-major A operand with N = 16 took ~128 cycles per instruction: 780 cycles per 128-column step)
// A stage is released by tcgen05.commit.  Four worker warps (one TMEM lane quarter each) read S, run the softmax over v through
// shared memory as before (16 warps, one head each), write alpha^T as a 128B-swizzled K-major operand tile, and the first
// quarter's four warps drain the pass-2 accumulators: thread = head row, 32 columns each = 64 contiguous bytes of Xbar.
constexpr int AT5 = 128 * TB * 2;             // one 64-v block of the alpha^T operand tile: 128 rows x 128 bytes
#ifndef NACC5
#define NACC5 2                              // pass-1 accumulators: one per sub-tile of a step (probe: -DNACC5=1)
#endif
constexpr int NW5 = 16;                      // worker warps: TMEM lane quarter (warp & 3) x 4 heads of the 16 ((warp - 4) >> 2)
constexpr int NT5 = 128 + NW5 * 32;          // warps 0 / 3 TMA producers, warps 1 / 2 MMA issuers (pass 1 / pass 2), warps 4..19 workers
__device__ __forceinline__ void worker_sync() { asm volatile("bar.sync 1, 512;" ::: "memory"); }
struct T5Layout { int sX, sXB, sU, sAT, sS, bars, total; };
__host__ __device__ inline T5Layout t5_fwd_layout(int Vp, int sta, int stb) {
  T5Layout L;
  L.sX = 0;                                    // ring A: X sub-tile pairs of pass 1
  L.sXB = sta * 2 * Vp * TB * 2;               // ring B: X sub-tile pairs of pass 2
  L.sU = L.sXB + stb * 2 * Vp * TB * 2;        // ring A: Ut sub-tile pairs
  L.sAT = L.sU + sta * 2 * UT;                 // multiple of 1024: Vp * 128 is a multiple of 2048
  L.sS = L.sAT + 2 * AT5;                      // (the 128-row A operand of pass 1 reads past the Vp rows of a sub-tile: into the next one / sU)
  L.bars = L.sS + VP_MAX * SROW * 4;
  L.total = L.bars + 8 * (2 * sta + 2 * stb + 9) + 16;
  return L;
}
#ifdef ORBIT_PROBE_AGG_P1ONLY   // A/B build only: pass 1 alone (no second read of X, no Xbar): wrong results
#define AGG_PROBE_PASSES 1
#else
#define AGG_PROBE_PASSES 2
#endif
// Two rings: ring A streams X (and Ut) for pass 1, ring B re-reads X for pass 2 (from L2: a patch's tile is requested again as
// soon as its pass 1 has completed, last chunk first).  With ONE ring the stream was a FIFO of [pass 1 of patch p][second read of
// p][pass 1 of p + 1]: the DRAM stream of the next patch could not start before pass 2 had drained the slots, and every patch
// paid the softmax bubble plus a DRAM latency ramp.  Each ring has its own producer thread and its own consumer (issuing) thread.
__global__ void __launch_bounds__(NT5, 1) agg_fwd_t5_kernel(const __grid_constant__ CUtensorMap tmX,
    const __grid_constant__ CUtensorMap tmU, float* __restrict__ alpha, bf16* __restrict__ Xbar, int BL, int V, int D, int h,
    int STA, int STB, int HINT) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = smem_raw + ((1024 - (s_u32(smem_raw) & 1023)) & 1023);
  const int Vp = (V + 15) & ~15, XTb = Vp * TB * 2;
  const T5Layout L = t5_fwd_layout(Vp, STA, STB);
  const uint32_t sXA = s_u32(smem) + L.sX, sXB = s_u32(smem) + L.sXB, sU = s_u32(smem) + L.sU, sAT = s_u32(smem) + L.sAT;
  float* sS = reinterpret_cast<float*>(smem + L.sS);                          // [128][SROW]
  const uint32_t fullA = s_u32(smem) + L.bars, emptyA = fullA + 8 * STA, fullB = emptyA + 8 * STA, emptyB = fullB + 8 * STB,
                 s_full0 = emptyB + 8 * STB, s_free0 = s_full0 + 16, at_full = s_free0 + 16, o_full0 = at_full + 8,
                 o_empty0 = o_full0 + 16, tslot = o_empty0 + 16;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nch = D / (2 * TB), mtiles = Vp / 16;
  const int np2 = (AGG_PROBE_PASSES - 1) * nch;              // pass-2 steps

  for (int j = 0; j < (STA + STB) * 2; j++) zero_tail_rows(smem + L.sX + j * XTb, V, Vp, NT5);     // ring B follows ring A
  if (threadIdx.x == 0) {
    for (int i = 0; i < STA; i++) { mbar_init(fullA + 8 * i, 1); mbar_init(emptyA + 8 * i, 1); }
    for (int i = 0; i < STB; i++) { mbar_init(fullB + 8 * i, 1); mbar_init(emptyB + 8 * i, 1); }
    mbar_init(at_full, 1);
    for (int i = 0; i < 2; i++) {
      mbar_init(s_full0 + 8 * i, 1); mbar_init(s_free0 + 8 * i, NW5);
      mbar_init(o_full0 + 8 * i, 1); mbar_init(o_empty0 + 8 * i, 4);
    }
    fence_barrier_init();
  }
  if (warp == 1) { tmem_alloc(tslot, 512); tmem_relinquish(); }
  for (int i = threadIdx.x; i < 2 * AT5 / 16; i += NT5) reinterpret_cast<uint4*>(smem + L.sAT)[i] = make_uint4(0, 0, 0, 0);   // rows 16..127 of alpha^T stay zero
  fence_proxy_async();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem) : "r"(tslot));
  const uint32_t tS0 = tmem, tO = tmem + 128;            // S of patch parity pb at tS0 + 32 pb (+ 16: the second accumulator)

  const int npat = blockIdx.x < BL ? (BL - 1 - blockIdx.x) / gridDim.x + 1 : 0;
  if (warp == 0) {
    if (lane == 0) {                                      // producer A: X and Ut chunks of pass 1, patch after patch
      int st = 0; uint32_t ph = 0;
      // (evict_last on all first reads: 711 vs 701 us; on the 2-8 chunks read first, which are re-read last and are the ones the L2
      // loses: 693-702 vs 689 us, DRAM bytes unchanged -- the hint does not keep them)
      const uint64_t pol = l2_policy(HINT & 1 ? 2 : 0);
      for (int pi = 0; pi < npat; pi++) {
        const int row0 = (blockIdx.x + pi * gridDim.x) * V;
        for (int c = 0; c < nch; c++) {
          const uint32_t bar = fullA + 8 * st;
          mbar_wait(emptyA + 8 * st, ph ^ 1);
          mbar_expect_tx(bar, 2 * (V * TB * 2 + UT));
#pragma unroll
          for (int j = 0; j < 2; j++) {
            tma_load_2d_hint(sXA + (st * 2 + j) * XTb, &tmX, bar, (c * 2 + j) * TB, row0, pol);
            tma_load_2d(sU + (st * 2 + j) * UT, &tmU, bar, (c * 2 + j) * TB, 0);
          }
          if (++st == STA) { st = 0; ph ^= 1; }
        }
      }
    }
  } else if (warp == 3) {
    if (lane == 0 && np2 > 0) {                           // producer B: the second read of a patch, once its pass 1 is complete
      int st = 0; uint32_t ph = 0;
      const uint64_t pol = l2_policy(HINT & 2 ? 1 : 0);     // ... and not after that
      for (int pi = 0; pi < npat; pi++) {
        const int row0 = (blockIdx.x + pi * gridDim.x) * V;
        mbar_wait(s_full0 + 8 * (pi & 1), (pi >> 1) & 1);
        for (int c = nch - 1; c >= 0; c--) {               // most recently read lines first
          const uint32_t bar = fullB + 8 * st;
          mbar_wait(emptyB + 8 * st, ph ^ 1);
          mbar_expect_tx(bar, 2 * V * TB * 2);
#pragma unroll
          for (int j = 0; j < 2; j++) tma_load_2d_hint(sXB + (st * 2 + j) * XTb, &tmX, bar, (c * 2 + j) * TB, row0, pol);
          if (++st == STB) { st = 0; ph ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // pass-1 issuer: runs up to one patch ahead of the softmax (S is double buffered by patch parity)
    if (lane == 0) {
      constexpr uint32_t idesc1 = make_idesc_bf16(128, HP, 0, 0);
      int st = 0; uint32_t ph = 0;
      for (int pi = 0; pi < npat; pi++) {
        const uint32_t pb = pi & 1, tS = tS0 + pb * 32;
        mbar_wait(s_free0 + 8 * pb, ((pi >> 1) & 1) ^ 1);
        for (int i = 0; i < nch; i++) {
          mbar_wait(fullA + 8 * st, ph);
          tc_fence_after();
#pragma unroll
          for (int j = 0; j < 2; j++)
#pragma unroll
            for (int ks = 0; ks < TB / 16; ks++)
              mma_f16_ss(NACC5 == 2 && j ? tS + 16 : tS, make_smem_desc(sXA + (st * 2 + j) * XTb + ks * 32, 16, 1024),
                         make_smem_desc(sU + (st * 2 + j) * UT + ks * 32, 16, 1024), idesc1, (NACC5 == 2 ? (i | ks) : (i | j | ks)) != 0);
          mma_commit(emptyA + 8 * st);
          if (++st == STA) { st = 0; ph ^= 1; }
        }
        mma_commit(s_full0 + 8 * pb);
      }
    }
  } else if (warp == 2) {
    // pass-2 issuer
    if (lane == 0) {
      constexpr uint32_t idesc2 = make_idesc_bf16(128, 2 * TB, 0, 1);
      int st = 0; uint32_t ph = 0, u = 0;
      for (int pi = 0; pi < npat; pi++) {
        mbar_wait(at_full, pi & 1);
        for (int i = 0; i < np2; i++, u++) {
          const uint32_t ob = u & 1;
          mbar_wait(fullB + 8 * st, ph);
          mbar_wait(o_empty0 + 8 * ob, ((u >> 1) & 1) ^ 1);
          tc_fence_after();
          for (int ks = 0; ks < mtiles; ks++)
            mma_f16_ss(tO + ob * (2 * TB), make_smem_desc(sAT + (ks >> 2) * AT5 + (ks & 3) * 32, 16, 1024),
                       make_smem_desc(sXB + (st * 2) * XTb + ks * 2048, XTb, 1024), idesc2, ks != 0);
          mma_commit(emptyB + 8 * st);
          mma_commit(o_full0 + 8 * ob);
          if (++st == STB) { st = 0; ph ^= 1; }
        }
      }
    }
  } else {
    const int w = warp - 4, quarter = warp & 3, sub = w >> 2, r = quarter * 32 + lane;
    const uint32_t lane_off = (uint32_t)(quarter * 32) << 16;
    uint8_t* at = smem + L.sAT;
    uint32_t u = 0;
    for (int pi = 0; pi < npat; pi++) {
      const int bl = blockIdx.x + pi * gridDim.x;
      const uint32_t pb = pi & 1, tS = tS0 + pb * 32;
      mbar_wait(s_full0 + 8 * pb, (pi >> 1) & 1);
      tc_fence_after();
      uint32_t sv[4], sv2[4] = {0u, 0u, 0u, 0u};
      tmem_ld_32x4(tS + sub * 4 + lane_off, sv);
      if (NACC5 == 2) tmem_ld_32x4(tS + 16 + sub * 4 + lane_off, sv2);
      tmem_ld_wait();
#pragma unroll
      for (int a = 0; a < 4; a++) sS[r * SROW + sub * 4 + a] = __uint_as_float(sv[a]) + (NACC5 == 2 ? __uint_as_float(sv2[a]) : 0.f);
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(s_free0 + 8 * pb);
      worker_sync();
      // ---- softmax over v per head (one warp each); alpha -> global (fp32), alpha^T -> the K-major operand tile (two blocks
      // of 64 v, 128B swizzle)
      {
        const int a = w;
        float m = -INFINITY, l = 0.f;
        if (a < h) {
          for (int v = lane; v < V; v += 32) m = fmaxf(m, sS[v * SROW + a]);
          m = warp_max(m);
          for (int v = lane; v < V; v += 32) l += __expf(sS[v * SROW + a] - m);
          l = warp_sum(l);
        }
        const float inv = a < h ? 1.f / l : 0.f;
        for (int v = lane; v < 2 * TB; v += 32) {
          const float p = (a < h && v < V) ? __expf(sS[v * SROW + a] - m) * inv : 0.f;
          if (a < h && v < V) alpha[((size_t)bl * h + a) * V + v] = p;
          *reinterpret_cast<bf16*>(at + (v >> 6) * AT5 + a * 128 + ((((v & 63) >> 3) ^ (a & 7)) << 4) + (v & 7) * 2) = __float2bfloat16_rn(p);
        }
      }
      fence_proxy_async();
      worker_sync();
      if (w == 0 && lane == 0) mbar_arrive(at_full);
      // ---- pass 2: drain Xbar[a, d] of each 128-column chunk (chunks come last to first)
      for (int i = 0; i < np2; i++, u++) {
        const uint32_t ob = u & 1;
        const int c = nch - 1 - i;
        if (quarter != 0) continue;                            // the 16 head rows sit in TMEM lanes 0..15: the first quarter's warps
        mbar_wait(o_full0 + 8 * ob, (u >> 1) & 1);
        tc_fence_after();
        uint32_t ov[32];
        tmem_ld_32x32(tO + ob * (2 * TB) + sub * 32, ov);      // this warp's 32 of the chunk's 128 columns
        tmem_ld_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(o_empty0 + 8 * ob);
        if (lane < h) {
          uint4* dst = reinterpret_cast<uint4*>(Xbar + ((size_t)bl * h + lane) * D + c * (2 * TB) + sub * 32);
#pragma unroll
          for (int q = 0; q < 4; q++)
            __stcs(dst + q, make_uint4(pack_bf16(__uint_as_float(ov[q * 8]), __uint_as_float(ov[q * 8 + 1])),
                                       pack_bf16(__uint_as_float(ov[q * 8 + 2]), __uint_as_float(ov[q * 8 + 3])),
                                       pack_bf16(__uint_as_float(ov[q * 8 + 4]), __uint_as_float(ov[q * 8 + 5])),
                                       pack_bf16(__uint_as_float(ov[q * 8 + 6]), __uint_as_float(ov[q * 8 + 7]))));
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) { tc_fence_after(); tmem_dealloc(tmem, 512); }
}

#ifdef ORBIT_PROBE_AGG          // A/B build only: cycles the MMA-issuing thread of CTA 0 spends in its waits / issuing, per patch
#define TPROBE_DECL long long tp_[7] = {0, 0, 0, 0, 0, 0, 0}; const long long tt0_ = clock64()
#define TPROBE(slot, stmt) do { long long t0_ = clock64(); stmt; tp_[slot] += clock64() - t0_; } while (0)
#define TPROBE_PRINT7 do { if (blockIdx.x == 0 && npat > 0) printf("agg bwd t5 probe: patches %d  per patch: total %lld  wait pass-1 data %lld  wait (alpha|ds) %lld  wait pass-2 data %lld  wait x_empty %lld  issue pass-1 %lld  issue dX %lld  issue dUt %lld\n", npat, (clock64() - tt0_) / npat, tp_[0] / npat, tp_[1] / npat, tp_[2] / npat, tp_[3] / npat, tp_[4] / npat, tp_[5] / npat, tp_[6] / npat); } while (0)
#else
#define TPROBE_PRINT7
#define TPROBE_DECL
#define TPROBE(slot, stmt) stmt
#endif
// ============================================ backward on tcgen05 ============================================
// Same structure as the forward: the TMA ring feeds one MMA-issuing thread, 16 worker warps own the TMEM lanes.
//   pass 1: dalpha[v, a] (TMEM, 16 columns) = sum over chunks of X[128 x 64] (A, K-major) . dXbar[16 x 64]^T (B, K-major)
//   workers: dalpha -> shared memory, ds = alpha (dalpha - sum_w alpha_w dalpha_w); (alpha | ds) as packed bf16 INTO TENSOR MEMORY
//            (thread = token row v: the A operand of the dX product, never in shared memory), ds^T as a K-major B tile
//   pass 2, per 64-column sub-tile:  dX[v, d] (TMEM, 64 columns, double buffered) = (alpha | ds)[128 x 32] (A, TMEM)
//                                                                               . [dXbar ; Ut][32 x 64] (B, MN-major)
//           per 128-column step:     dUt^T[d, a] (TMEM, 16 columns per step, kept for ALL patches of the CTA)
//                                      += X^T[128 d x V] (A, MN-major: the X tiles as they are) . ds^T[16 x V]^T (B, K-major)
//   workers drain dX (thread = token row, 16 columns = 32 bytes each) and, after the last patch, dUt^T (fp32 atomics).
constexpr int BT5 = 2 * UT;                  // B tile of a 64-column sub-tile: rows 0-15 dXbar, rows 16-31 Ut
constexpr int OT5 = 32 * TB * 2;             // dX staging tile of one TMEM lane quarter: 32 token rows x 64 columns, 128B swizzle
__device__ __forceinline__ void quarter_sync(int q) { asm volatile("bar.sync %0, 128;" ::"r"(2 + q) : "memory"); }
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* m, uint32_t src, int c0, int c1, int c2, uint64_t policy) {
  asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group.L2::cache_hint [%0, {%2, %3, %4}], [%1], %5;" ::"l"(m), "r"(src), "r"(c0),
               "r"(c1), "r"(c2), "l"(policy) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
struct T5BLayout { int sX, sXB, sBA, sBB, sDT, sO, sS, sAl, bars, total; };
__host__ __device__ inline T5BLayout t5_bwd_layout(int V, int sta, int stb) {
  const int Vp = (V + 15) & ~15, nq = (V + 31) / 32;
  T5BLayout L;
  L.sX = 0;                                    // ring A: X sub-tile pairs of pass 1
  L.sXB = sta * 2 * Vp * TB * 2;               // ring B: X sub-tile pairs of pass 2
  L.sBA = L.sXB + stb * 2 * Vp * TB * 2;       // ring A: dXbar sub-tile pairs [16 x 64]
  L.sBB = L.sBA + sta * 2 * UT;                // ring B: [dXbar ; Ut] sub-tile pairs [32 x 64]
  L.sDT = L.sBB + stb * 2 * BT5;
  L.sO = L.sDT + 2 * UT;                       // dX staging: two tiles per live TMEM lane quarter
  L.sS = L.sO + nq * 2 * OT5;
  L.sAl = L.sS + Vp * SROW * 4;
  L.bars = L.sAl + Vp * SROW * 4;
  L.total = L.bars + 8 * (2 * sta + 2 * stb + 12) + 16;
  return L;
}

// Two rings and two issuing threads, as in the forward: ring A streams X and dXbar for pass 1 (issuer A: dalpha, double buffered
// by patch parity so that it runs one patch ahead), ring B re-reads X with [dXbar ; Ut] for pass 2 once pass 1 of the patch is
// complete (issuer B: per 128-column step the dUt^T product first, then the two dX sub-tiles, so that the last dX commit of a
// patch covers all of its products and the workers may overwrite (alpha | ds) / ds^T for the next patch once they have drained it).
__global__ void __launch_bounds__(NT5, 1) agg_bwd_t5_kernel(const __grid_constant__ CUtensorMap tmX,
    const __grid_constant__ CUtensorMap tmG, const __grid_constant__ CUtensorMap tmU, const __grid_constant__ CUtensorMap tmD,
    const float* __restrict__ alpha, float* __restrict__ dUt_acc, int BL, int V, int D, int h, int STA, int STB, int HINT) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = smem_raw + ((1024 - (s_u32(smem_raw) & 1023)) & 1023);
  const int Vp = (V + 15) & ~15, XTb = Vp * TB * 2;
  const T5BLayout L = t5_bwd_layout(V, STA, STB);
  const uint32_t sXA = s_u32(smem) + L.sX, sXB = s_u32(smem) + L.sXB, sBA = s_u32(smem) + L.sBA, sBB = s_u32(smem) + L.sBB,
                 sDT = s_u32(smem) + L.sDT, sO = s_u32(smem) + L.sO;
  float* sS = reinterpret_cast<float*>(smem + L.sS);                          // [Vp][SROW] dalpha, then ds
  float* sAl = reinterpret_cast<float*>(smem + L.sAl);                        // [Vp][SROW] alpha
  const uint32_t fullA = s_u32(smem) + L.bars, emptyA = fullA + 8 * STA, fullB = emptyA + 8 * STA, emptyB = fullB + 8 * STB,
                 a_full0 = emptyB + 8 * STB, a_free0 = a_full0 + 16, ad_full = a_free0 + 16, x_full0 = ad_full + 8,
                 x_empty0 = x_full0 + 16, u_done = x_empty0 + 16, tslot = u_done + 8;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nch = D / (2 * TB), mtiles = Vp / 16;

  for (int j = 0; j < (STA + STB) * 2; j++) zero_tail_rows(smem + L.sX + j * XTb, V, Vp, NT5);
  for (int j = 0; j < STA * 2; j++) zero_tail_rows(smem + L.sBA + j * UT, h, HP, NT5);     // dXbar rows h..15 (the TMA box has h rows)
  for (int j = 0; j < STB * 2; j++) zero_tail_rows(smem + L.sBB + j * BT5, h, HP, NT5);
  if (threadIdx.x == 0) {
    for (int i = 0; i < STA; i++) { mbar_init(fullA + 8 * i, 1); mbar_init(emptyA + 8 * i, 1); }
    for (int i = 0; i < STB; i++) { mbar_init(fullB + 8 * i, 1); mbar_init(emptyB + 8 * i, 1); }
    mbar_init(ad_full, 1); mbar_init(u_done, 1);
    for (int i = 0; i < 2; i++) {
      mbar_init(a_full0 + 8 * i, 1); mbar_init(a_free0 + 8 * i, NW5);
      mbar_init(x_full0 + 8 * i, 1); mbar_init(x_empty0 + 8 * i, NW5);
    }
    fence_barrier_init();
  }
  if (warp == 1) { tmem_alloc(tslot, 512); tmem_relinquish(); }
  fence_proxy_async();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem) : "r"(tslot));
  // dalpha of patch parity pb at tA0 + 32 pb (+ 16: the second accumulator), (alpha | ds), dX (2 x 64), dUt^T (16 per step)
  const uint32_t tA0 = tmem, tAD = tmem + 64, tdX = tmem + 80, tdU = tmem + 80 + 2 * TB;

  const int npat = blockIdx.x < BL ? (BL - 1 - blockIdx.x) / gridDim.x + 1 : 0;
  if (warp == 0) {
    if (lane == 0) {                                      // producer A: X and dXbar chunks of pass 1
      int st = 0; uint32_t ph = 0;
      const uint64_t polA = l2_policy(HINT & 1 ? 2 : 0);
      for (int pi = 0; pi < npat; pi++) {
        const int bl = blockIdx.x + pi * gridDim.x;
        for (int c = 0; c < nch; c++) {
          const uint32_t bar = fullA + 8 * st;
          mbar_wait(emptyA + 8 * st, ph ^ 1);
          mbar_expect_tx(bar, 2 * (V + h) * TB * 2);
#pragma unroll
          for (int j = 0; j < 2; j++) {
            tma_load_2d_hint(sXA + (st * 2 + j) * XTb, &tmX, bar, (c * 2 + j) * TB, bl * V, polA);
            tma_load_2d_hint(sBA + (st * 2 + j) * UT, &tmG, bar, (c * 2 + j) * TB, bl * h, polA);
          }
          if (++st == STA) { st = 0; ph ^= 1; }
        }
      }
    }
  } else if (warp == 3) {
    if (lane == 0) {                                      // producer B: X again (from L2), dXbar and Ut, once pass 1 of the patch is done
      int st = 0; uint32_t ph = 0;
      const uint64_t pol = l2_policy(HINT & 2 ? 1 : 0);
      for (int pi = 0; pi < npat; pi++) {
        const int bl = blockIdx.x + pi * gridDim.x;
        mbar_wait(a_full0 + 8 * (pi & 1), (pi >> 1) & 1);
        for (int c = nch - 1; c >= 0; c--) {
          const uint32_t bar = fullB + 8 * st;
          mbar_wait(emptyB + 8 * st, ph ^ 1);
          mbar_expect_tx(bar, 2 * ((V + h) * TB * 2 + UT));
#pragma unroll
          for (int j = 0; j < 2; j++) {
            tma_load_2d_hint(sXB + (st * 2 + j) * XTb, &tmX, bar, (c * 2 + j) * TB, bl * V, pol);
            tma_load_2d_hint(sBB + (st * 2 + j) * BT5, &tmG, bar, (c * 2 + j) * TB, bl * h, pol);
            tma_load_2d(sBB + (st * 2 + j) * BT5 + UT, &tmU, bar, (c * 2 + j) * TB, 0);
          }
          if (++st == STB) { st = 0; ph ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {                                      // issuer A: dalpha
      constexpr uint32_t idesc1 = make_idesc_bf16(128, HP, 0, 0);
      int st = 0; uint32_t ph = 0;
      for (int pi = 0; pi < npat; pi++) {
        const uint32_t pb = pi & 1, tA = tA0 + pb * 32;
        mbar_wait(a_free0 + 8 * pb, ((pi >> 1) & 1) ^ 1);
        for (int i = 0; i < nch; i++) {
          mbar_wait(fullA + 8 * st, ph);
          tc_fence_after();
#pragma unroll
          for (int j = 0; j < 2; j++)
#pragma unroll
            for (int ks = 0; ks < TB / 16; ks++)
              mma_f16_ss(NACC5 == 2 && j ? tA + 16 : tA, make_smem_desc(sXA + (st * 2 + j) * XTb + ks * 32, 16, 1024),
                         make_smem_desc(sBA + (st * 2 + j) * UT + ks * 32, 16, 1024), idesc1, (NACC5 == 2 ? (i | ks) : (i | j | ks)) != 0);
          mma_commit(emptyA + 8 * st);
          if (++st == STA) { st = 0; ph ^= 1; }
        }
        mma_commit(a_full0 + 8 * pb);
      }
    }
  } else if (warp == 2) {
    if (lane == 0) {                                      // issuer B: dUt^T and dX
      constexpr uint32_t idesc_x = make_idesc_bf16(128, TB, 0, 1), idesc_u = make_idesc_bf16(128, HP, 1, 0);
      int st = 0; uint32_t ph = 0, u = 0;
      for (int pi = 0; pi < npat; pi++) {
        mbar_wait(ad_full, pi & 1);
        for (int i = 0; i < nch; i++) {
          const int c = nch - 1 - i;
          mbar_wait(fullB + 8 * st, ph);
          tc_fence_after();
          for (int ks = 0; ks < mtiles; ks++)
            mma_f16_ss(tdU + c * HP, make_smem_desc(sXB + (st * 2) * XTb + ks * 2048, XTb, 1024),
                       make_smem_desc(sDT + (ks >> 2) * UT + (ks & 3) * 32, 16, 1024), idesc_u, (pi | ks) != 0);
#pragma unroll
          for (int j = 0; j < 2; j++, u++) {
            const uint32_t xb = u & 1;
            mbar_wait(x_empty0 + 8 * xb, ((u >> 1) & 1) ^ 1);
            tc_fence_after();
#pragma unroll
            for (int ks = 0; ks < 2; ks++)                 // k = (alpha | ds): rows 0-15 dXbar, 16-31 Ut of the B tile
              mma_f16_ts(tdX + xb * TB, tAD + ks * 8, make_smem_desc(sBB + (st * 2 + j) * BT5 + ks * 2048, 16, 1024), idesc_x, ks != 0);
            mma_commit(x_full0 + 8 * xb);
          }
          mma_commit(emptyB + 8 * st);
          if (++st == STB) { st = 0; ph ^= 1; }
        }
      }
      mma_commit(u_done);
    }
  } else if (warp >= 4) {
    const int w = warp - 4, quarter = warp & 3, sub = w >> 2, r = quarter * 32 + lane;
    const uint32_t lane_off = (uint32_t)(quarter * 32) << 16;
    uint8_t* dt = smem + L.sDT;
    const uint64_t pol_st = l2_policy(HINT & 4 ? 1 : 0);     // dX is not read again here: it should not push the X tiles out of L2
    uint32_t u = 0;
    for (int pi = 0; pi < npat; pi++) {
      const int bl = blockIdx.x + pi * gridDim.x;
      // alpha of this patch (dead since the previous patch's (alpha | ds) went to tensor memory)
      for (int i = threadIdx.x - 128; i < 128 * HP; i += NW5 * 32) {
        const int a = i >> 7, v = i & 127;
        if (v < Vp) sAl[v * SROW + a] = (v < V && a < h) ? alpha[((size_t)bl * h + a) * V + v] : 0.f;
      }
      const uint32_t pb = pi & 1, tA = tA0 + pb * 32;
      mbar_wait(a_full0 + 8 * pb, (pi >> 1) & 1);
      tc_fence_after();
      uint32_t sv[4], sv2[4] = {0u, 0u, 0u, 0u};
      tmem_ld_32x4(tA + sub * 4 + lane_off, sv);
      if (NACC5 == 2) tmem_ld_32x4(tA + 16 + sub * 4 + lane_off, sv2);
      tmem_ld_wait();
#pragma unroll
      for (int a = 0; a < 4; a++)
        if (r < Vp) sS[r * SROW + sub * 4 + a] = __uint_as_float(sv[a]) + (NACC5 == 2 ? __uint_as_float(sv2[a]) : 0.f);   // (lanes >= Vp: not data)
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(a_free0 + 8 * pb);
      worker_sync();
      // ---- ds[v, a] = alpha (dalpha - sum_w alpha_w dalpha_w), one head per warp; ds^T -> the K-major B tile of the dUt product
      {
        const int a = w;
        float dot = 0.f;
        for (int v = lane; v < V; v += 32) dot += sAl[v * SROW + a] * sS[v * SROW + a];
        dot = warp_sum(dot);
        for (int v = lane; v < 2 * TB; v += 32) {
          const float ds = v < V ? sAl[v * SROW + a] * (sS[v * SROW + a] - dot) : 0.f;
          if (v < Vp) sS[v * SROW + a] = ds;
          *reinterpret_cast<bf16*>(dt + (v >> 6) * UT + a * 128 + ((((v & 63) >> 3) ^ (a & 7)) << 4) + (v & 7) * 2) = __float2bfloat16_rn(ds);
        }
      }
      worker_sync();
      // ---- (alpha | ds) of this thread's token row -> tensor memory: warp (quarter, sub) writes k = 8 sub .. 8 sub + 7
      {
        const float* src = (sub < 2 ? sAl : sS) + r * SROW + (sub & 1) * 8;
        uint32_t pk[4];
#pragma unroll
        for (int q = 0; q < 4; q++) pk[q] = r < Vp ? pack_bf16(src[2 * q], src[2 * q + 1]) : 0u;
        tmem_st_32x4(tAD + sub * 4 + lane_off, pk);
        tmem_st_wait();
      }
      tc_fence_before();
      fence_proxy_async();
      worker_sync();
      if (w == 0 && lane == 0) mbar_arrive(ad_full);
      // ---- pass 2: drain dX of each 64-column sub-tile: thread = token row, this warp's 16 columns
      for (int i = 0; i < nch; i++) {
        const int c = nch - 1 - i;
#pragma unroll
        for (int j = 0; j < 2; j++, u++) {
          const uint32_t xb = u & 1;
          mbar_wait(x_full0 + 8 * xb, (u >> 1) & 1);
          tc_fence_after();
          uint32_t ov[16];
          tmem_ld_32x16(tdX + xb * TB + sub * 16 + lane_off, ov);
          tmem_ld_wait();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(x_empty0 + 8 * xb);
          // the quarter's four warps fill a [32 rows x 64 columns] staging tile (this warp: 16 columns = two 16-byte chunks
          // of every row), which leaves as ONE TMA box store over dtok seen as [BL][V][D]: rows >= V are clipped by the map.
          // (Row-per-thread 32-byte stores to rows 4 KB apart made this drain the critical path: 10.8k of 48k cycles per patch.)
          if (quarter * 32 < V) {
            const uint32_t so = sO + (quarter * 2 + xb) * OT5;
            if (sub == 0 && lane == 0) bulk_wait_read<1>();          // the store issued two sub-tiles ago has left this buffer
            quarter_sync(quarter);
#pragma unroll
            for (int q = 0; q < 2; q++) {
              const uint32_t addr = so + lane * 128 + (((sub * 2 + q) ^ (lane & 7)) << 4);
              asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr),
                           "r"(pack_bf16(__uint_as_float(ov[q * 8]), __uint_as_float(ov[q * 8 + 1]))),
                           "r"(pack_bf16(__uint_as_float(ov[q * 8 + 2]), __uint_as_float(ov[q * 8 + 3]))),
                           "r"(pack_bf16(__uint_as_float(ov[q * 8 + 4]), __uint_as_float(ov[q * 8 + 5]))),
                           "r"(pack_bf16(__uint_as_float(ov[q * 8 + 6]), __uint_as_float(ov[q * 8 + 7]))) : "memory");
            }
            fence_proxy_async();
            quarter_sync(quarter);
            if (sub == 0 && lane == 0) { tma_store_3d(&tmD, so, (c * 2 + j) * TB, quarter * 32, bl, pol_st); bulk_commit(); }
          }
        }
      }
    }
    if (sub == 0 && lane == 0) bulk_wait_all();              // the staging tiles outlive the last stores
    // ---- dUt^T accumulated over all patches of this CTA: thread = column d of a 128-column step, this warp's 4 heads
    if (npat > 0) {
      mbar_wait(u_done, 0);
      tc_fence_after();
      for (int c = 0; c < nch; c++) {
        uint32_t av[4];
        tmem_ld_32x4(tdU + c * HP + sub * 4 + lane_off, av);
        tmem_ld_wait();
        const int d = c * (2 * TB) + r;
#pragma unroll
        for (int q = 0; q < 4; q++)
          if (sub * 4 + q < h) atomicAdd(dUt_acc + (size_t)d * h + sub * 4 + q, __uint_as_float(av[q]));
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) { tc_fence_after(); tmem_dealloc(tmem, 512); }
}

// Ut [D, h] fp32 -> Utb [HP, D] bf16 (rows >= h zero)
__global__ void agg_ut_to_bf16_kernel(const float* __restrict__ Ut, bf16* __restrict__ Utb, int D, int h) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= HP * D) return;
  int a = i / D, d = i - a * D;
  Utb[i] = __float2bfloat16_rn(a < h ? Ut[(size_t)d * h + a] : 0.f);
}

size_t fwd_smem(int stg) {
  return 1024 + (size_t)stg * 2 * (XT + UT) + (size_t)VP_MAX * SROW * 4 + (size_t)HP * (VP_MAX + 8) * 2 + 16 * stg;
}
size_t bwd_smem(int V, int D, int stg) {
  const size_t Vp = (V + 15) & ~15;
  (void)D;                               // the [HP][D] accumulator is in tensor memory
  return 1024 + (size_t)stg * (Vp * TB * 2 + BT) + 2 * Vp * SROW * 4 + Vp * (2 * HP + 8) * 2 +
         (size_t)HP * (VP_MAX + 8) * 2 + 64 + 16 * stg;
}
constexpr size_t SMEM_MAX = 227 * 1024;

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
// bf16 matrix [rows, D] row-major -> boxes of [box_rows x 64 columns], 128-byte swizzle
int make_map(CUtensorMap* tm, const void* base, long long rows, int D, int box_rows) {
  static std::atomic<EncodeTiledFn> enc_c{nullptr};
  EncodeTiledFn enc = enc_c.load(std::memory_order_relaxed);
  if (!enc) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess) { set_error("cuTensorMapEncodeTiled entry point not found"); return ORBIT_ERR_CUDA; }
    enc = (EncodeTiledFn)p;
    enc_c.store(enc, std::memory_order_relaxed);
  }
  cuuint64_t dims[2] = {(cuuint64_t)D, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)D * 2};
  cuuint32_t box[2] = {(cuuint32_t)TB, (cuuint32_t)box_rows};
  cuuint32_t es[2] = {1, 1};
  CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { set_error("aggregate: cuTensorMapEncodeTiled failed (%d)", (int)r); return ORBIT_ERR_CUDA; }
  return ORBIT_OK;
}
// dtok seen as [BL][V][D] bf16 -> boxes of [1][32 rows][64 columns], 128-byte swizzle: a store clips the rows >= V of a patch
int make_map_rows3(CUtensorMap* tm, const void* base, long long BL, int V, int D) {
  static std::atomic<void*> enc_c{nullptr};                 // the entry point is process-wide: looked up once
  void* p = enc_c.load(std::memory_order_relaxed);
  if (!p) {
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess) { set_error("cuTensorMapEncodeTiled entry point not found"); return ORBIT_ERR_CUDA; }
    enc_c.store(p, std::memory_order_relaxed);
  }
  cuuint64_t dims[3] = {(cuuint64_t)D, (cuuint64_t)V, (cuuint64_t)BL};
  cuuint64_t strides[2] = {(cuuint64_t)D * 2, (cuuint64_t)V * D * 2};
  cuuint32_t box[3] = {(cuuint32_t)TB, 32, 1};
  cuuint32_t es[3] = {1, 1, 1};
  CUresult r = ((EncodeTiledFn)p)(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, es,
                                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { set_error("aggregate: cuTensorMapEncodeTiled (dtok) failed (%d)", (int)r); return ORBIT_ERR_CUDA; }
  return ORBIT_OK;
}
}  // namespace

bool agg_tc_supported(int dt, int V, int D, int heads) {
  // D / 64 chunks x 4 accumulator columns x 2 warps per TMEM lane quarter <= TMEM_ACC_COLS
  return dt == ORBIT_BF16 && heads <= HP && V <= VP_MAX && D % 128 == 0 && D / TB * 8 <= TMEM_ACC_COLS && bwd_smem(V, D, 2) <= SMEM_MAX;
}
size_t agg_tc_utb_bytes(int D) { return (size_t)HP * D * sizeof(bf16); }

bool t5_enabled() {                     // ORBIT_AGG_T5=0: the mma.sync ring kernels (A/B)
  static const int v = [] { const char* e = getenv("ORBIT_AGG_T5"); return (e && e[0] == '0') ? 0 : 1; }();
  return v != 0;
}

int agg_patch_fwd_tc(const void* tok, const float* Ut, void* Utb, float* alpha, void* Xbar, int BL, int V, int D, int heads,
                     cudaStream_t s) {
  agg_ut_to_bf16_kernel<<<cdiv((long long)HP * D, 256), 256, 0, s>>>(Ut, (bf16*)Utb, D, heads);
  ORBIT_LAUNCH_CHECK();
  CUtensorMap tmX, tmU;
  ORBIT_TRY(make_map(&tmX, tok, (long long)BL * V, D, V));
  ORBIT_TRY(make_map(&tmU, Utb, HP, D, HP));
  if (t5_enabled()) {
    const int Vp = (V + 15) & ~15;
    // ring A (DRAM stream) gets the stages that ring B (L2 re-read, shorter latency) does not need
    static const int stb_env = [] { const char* e = getenv("ORBIT_AGG_STB"); return e ? atoi(e) : 0; }();
    static const int sta_env = [] { const char* e = getenv("ORBIT_AGG_STA"); return e ? atoi(e) : 0; }();
    static const int hint_env = [] { const char* e = getenv("ORBIT_AGG_HINT"); return e ? atoi(e) : 2; }();
    int stb = stb_env > 0 ? stb_env : 4, sta = sta_env > 0 ? sta_env : 12;
    while (sta > 1 && 1024 + (size_t)t5_fwd_layout(Vp, sta, stb).total > SMEM_MAX) sta--;
    while (stb > 1 && 1024 + (size_t)t5_fwd_layout(Vp, sta, stb).total > SMEM_MAX) stb--;
    const size_t smb = 1024 + (size_t)t5_fwd_layout(Vp, sta, stb).total;
    ORBIT_SMEM_ATTR(agg_fwd_t5_kernel, SMEM_MAX);
    const int grid = BL < num_sms() ? BL : num_sms();
    agg_fwd_t5_kernel<<<grid, NT5, smb, s>>>(tmX, tmU, alpha, (bf16*)Xbar, BL, V, D, heads, sta, stb, hint_env);
    ORBIT_LAUNCH_CHECK();
    return ORBIT_OK;
  }
  constexpr int STG = 5;                // 5 x 36 KB stages + 13 KB, one CTA per SM
  const size_t smb = fwd_smem(STG);
  ORBIT_SMEM_ATTR(agg_fwd_tma_kernel<STG>, smb);
  const int grid = BL < 148 ? BL : 148;
  agg_fwd_tma_kernel<STG><<<grid, NTF + 32, smb, s>>>(tmX, tmU, alpha, (bf16*)Xbar, BL, V, D, heads);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int agg_patch_bwd_tc(const void* tok, const void* Utb, const float* alpha, const void* dXbar, void* dtok, float* dUt_acc,
                     int BL, int V, int D, int heads, cudaStream_t s) {
  CUtensorMap tmX, tmG, tmU;
  ORBIT_TRY(make_map(&tmX, tok, (long long)BL * V, D, V));
  ORBIT_TRY(make_map(&tmG, dXbar, (long long)BL * heads, D, heads));
  ORBIT_TRY(make_map(&tmU, Utb, HP, D, HP));
  if (t5_enabled() && D <= 2048) {      // dUt^T of all D / 128 steps stays in tensor memory: 16 columns each beside 160 others
    static const int stb_env = [] { const char* e = getenv("ORBIT_AGG_BSTB"); return e ? atoi(e) : 0; }();
    static const int sta_env = [] { const char* e = getenv("ORBIT_AGG_BSTA"); return e ? atoi(e) : 0; }();
    // L2 hints: bit 0 evict_last on the first read, bit 1 evict_first on the second read, bit 2 evict_first on the dX stores.
    // At config 3 one patch time moves ~180 MB through the 126 MB L2 (X, X again, dX, dXbar twice), so about half of the second
    // read misses whatever the hints are: DRAM traffic is 1.35x the algorithmic bytes and the kernel runs at ~95 % of hbm_gbs of
    // actual DRAM traffic.
    static const int hint_env = [] { const char* e = getenv("ORBIT_AGG_BHINT"); return e ? atoi(e) : 6; }();
    int stb = stb_env > 0 ? stb_env : 4, sta = sta_env > 0 ? sta_env : 12;
    while (sta > 1 && 1024 + (size_t)t5_bwd_layout(V, sta, stb).total > SMEM_MAX) sta--;
    while (stb > 1 && 1024 + (size_t)t5_bwd_layout(V, sta, stb).total > SMEM_MAX) stb--;
    const size_t smb = 1024 + (size_t)t5_bwd_layout(V, sta, stb).total;
    ORBIT_SMEM_ATTR(agg_bwd_t5_kernel, SMEM_MAX);
    // (probe: with 74 CTAs the second read still misses, 5.8 GB of DRAM reads at C3; with 37 it hits, 3.8 GB: the reuse window of
    // this access pattern is ~50 MB chip-wide, i.e. ~340 KB per CTA at 148 CTAs, less than one patch tile)
    const int grid5 = BL < num_sms() ? BL : num_sms();
    CUtensorMap tmD;
    ORBIT_TRY(make_map_rows3(&tmD, dtok, BL, V, D));
    agg_bwd_t5_kernel<<<grid5, NT5, smb, s>>>(tmX, tmG, tmU, tmD, alpha, dUt_acc, BL, V, D, heads, sta, stb, hint_env);
    ORBIT_LAUNCH_CHECK();
    return ORBIT_OK;
  }
  const int grid = BL < 148 ? BL : 148;
  int stg = 12;                         // deepest ring that fits (the dUt accumulator is in tensor memory)
  while (stg > 2 && bwd_smem(V, D, stg) > SMEM_MAX) stg -= (stg > 6 ? 2 : 1);
  const size_t smb = bwd_smem(V, D, stg);
#define AB(S) do {                                                                                            \
    ORBIT_SMEM_ATTR(agg_bwd_tma_kernel<S>, smb);                                                              \
    agg_bwd_tma_kernel<S><<<grid, NTB + 32, smb, s>>>(tmX, tmG, tmU, alpha, (bf16*)dtok, dUt_acc, BL, V, D, heads); } while (0)
  if (stg == 12) AB(12); else if (stg == 10) AB(10); else if (stg == 8) AB(8); else if (stg == 6) AB(6); else if (stg == 5) AB(5);
  else if (stg == 4) AB(4); else if (stg == 3) AB(3); else AB(2);
#undef AB
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

}  // namespace orbit
