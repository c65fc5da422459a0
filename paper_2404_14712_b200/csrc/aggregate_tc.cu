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
  static EncodeTiledFn enc = nullptr;
  if (!enc) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess) { set_error("cuTensorMapEncodeTiled entry point not found"); return ORBIT_ERR_CUDA; }
    enc = (EncodeTiledFn)p;
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
}  // namespace

bool agg_tc_supported(int dt, int V, int D, int heads) {
  // D / 64 chunks x 4 accumulator columns x 2 warps per TMEM lane quarter <= TMEM_ACC_COLS
  return dt == ORBIT_BF16 && heads <= HP && V <= VP_MAX && D % 128 == 0 && D / TB * 8 <= TMEM_ACC_COLS && bwd_smem(V, D, 2) <= SMEM_MAX;
}
size_t agg_tc_utb_bytes(int D) { return (size_t)HP * D * sizeof(bf16); }

int agg_patch_fwd_tc(const void* tok, const float* Ut, void* Utb, float* alpha, void* Xbar, int BL, int V, int D, int heads,
                     cudaStream_t s) {
  agg_ut_to_bf16_kernel<<<cdiv((long long)HP * D, 256), 256, 0, s>>>(Ut, (bf16*)Utb, D, heads);
  ORBIT_LAUNCH_CHECK();
  CUtensorMap tmX, tmU;
  ORBIT_TRY(make_map(&tmX, tok, (long long)BL * V, D, V));
  ORBIT_TRY(make_map(&tmU, Utb, HP, D, HP));
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
