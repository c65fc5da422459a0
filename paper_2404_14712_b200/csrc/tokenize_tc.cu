// tokenize_tc.cu -- a1 / a1' on tensor cores (bf16 storage): "independent patch tokenization for each
// channel input".  At patch 4 the K = p^2 = 16 contraction costs 16 FMA per 2 output bytes on CUDA cores
// (ALU-bound, ~2x the HBM time); as one or two mma.sync k-steps it disappears under the token stream.
//
// fp32 pixels are split exactly into bf16 hi + lo parts (pix = hi + lo + O(2^-17)), so the contraction is
// [hi | lo] (K = 2 p^2) against [Wp ; Wp] and loses nothing against the fp32-FMA kernel.
//   forward : tok[b, l, v, c0:c0+512] for 128 patches of one (b, v) per CTA; B = [Wp[v]; Wp[v]] chunk in smem.
//   backward: dWp[v] (p^2 x D) and dbp[v] = sum over patches of pix^T dtok / dtok: CTA = (v, 512 columns, a range
//             of patches); dtok rows stream through a 4-stage cp.async ring; A fragments are built from pixels.
#include <cuda.h>
#include <string.h>
#include "frontend.cuh"
#include "ptx.cuh"

namespace orbit {
namespace {

constexpr int NT = 256;
constexpr int DCH = 512;                 // columns per CTA
constexpr int BROW = (DCH + 8) * 2;      // padded smem row of the B tiles (bytes): conflict-free ldmatrix
constexpr int OROW = (64 + 8) * 2;       // padded row of a warp's output staging tile (bytes)

__device__ __forceinline__ uint32_t s_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
// 4-byte copy, zero-filled when bytes == 0
__device__ __forceinline__ void cp_async4(uint32_t dst, const void* src, int bytes) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(dst), "l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
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
__device__ __forceinline__ void split_bf16(float x, bf16& hi, bf16& lo) {
  hi = __float2bfloat16_rn(x);
  lo = __float2bfloat16_rn(x - __bfloat162float(hi));
}
// two fp32 values -> packed bf16 (hi, hi) and packed residuals (lo, lo): a = hi_a + lo_a + O(2^-17 |a|)
__device__ __forceinline__ void split_pair(float a, float b, uint32_t& hi, uint32_t& lo) {
  hi = pack_bf16(a, b);
  lo = pack_bf16(a - __uint_as_float(hi << 16), b - __uint_as_float(hi & 0xffff0000u));
}
// B fragments of an N-major tile with padded rows: 16 k from k0, 16 n from n0
__device__ __forceinline__ void ldB(uint32_t base, int k0, int n0, uint32_t* r) {
  int lane = threadIdx.x & 31;
  ldsm4t(base + (k0 + (lane & 7) + ((lane >> 3) & 1) * 8) * BROW + (n0 + (lane >> 4) * 8) * 2, r);
}
__device__ __forceinline__ float pixel(const float* x, int V, int Hg, int Wg, int p, int bl, int L, int v, int r) {
  const int b = bl / L, l = bl - b * L, gw = Wg / p;
  const int i = l / gw, j = l - i * gw, di = r / p, dj = r - di * p;
  return x[(((size_t)b * V + v) * Hg + i * p + di) * Wg + j * p + dj];
}

__device__ __forceinline__ void stsm4(uint32_t addr, uint32_t r0, uint32_t r1, uint32_t r2, uint32_t r3) {
  asm volatile("stmatrix.sync.aligned.m8n8.x4.shared.b16 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(r0), "r"(r1), "r"(r2), "r"(r3) : "memory");
}
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* m, uint32_t src, int c0, int c1) {
  asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];" ::"l"(m), "r"(src), "r"(c0), "r"(c1) : "memory");
}

// ---------------------------------------------------------------- forward ----------------------------------
// KP = contraction length after the hi/lo split, padded to a multiple of 16 (p = 4: 32; p = 2: 16; p = 1: 16)
// TMA_OUT (D % 64 == 0): a warp's 16 x 64 output tile is written to a 128B-swizzled staging tile with four stmatrix.x4 (the
// m16n8 accumulator fragments are exactly the 8 x 8 matrices stmatrix stores) and leaves as ONE TMA box store over tok seen as a
// [B L, V D] matrix, two staging tiles per warp in flight.  The kernel is ISSUE-bound, not HBM-bound (445 M warp instructions for
// 3 GB at 47 % issue-active, profiles/r1_twocall_front.md): per 64-column group this drops 16 st.shared + 4 ld.shared + 4
// st.global and their address arithmetic.
template <int P2, int KP, bool TMA_OUT>
__global__ void __launch_bounds__(NT) tok_fwd_tc_kernel(orbit_embed_desc d, const float* __restrict__ x,
    const bf16* __restrict__ Wp, const bf16* __restrict__ bp, bf16* __restrict__ tok, int L,
    const __grid_constant__ CUtensorMap tmTok) {
  constexpr int PT = 128, AROW = (KP + 8) * 2;          // patches per CTA; padded A row (bytes)
  extern __shared__ __align__(1024) uint8_t smem[];
  // TMA_OUT: the first 32 KB are the staging tiles (8 warps x 2 x [16 rows x 128 B], 1024-byte aligned for the 128B swizzle)
  constexpr int STAGE_BYTES = TMA_OUT ? (NT / 32) * 2 * 2048 : 0;
  uint8_t* sA = smem + STAGE_BYTES;                       // [PT][KP + 8] bf16
  uint8_t* sB = sA + PT * AROW;                           // [KP][DCH + 8] bf16
  // blockIdx.x = (v, column chunk): CTAs that run together write neighbouring 1 KB pieces of the same token rows
  // ([V x D] of a patch is contiguous), instead of pieces V*D*2 bytes apart.
  const int nz = gridDim.x / d.V;
  const int v = blockIdx.x / nz, c0 = (blockIdx.x - v * nz) * DCH;
  const int BL = d.B * L, npb = (BL + PT - 1) / PT;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int ncol = min(DCH, d.D - c0);
  constexpr int P = P2 == 16 ? 4 : (P2 == 4 ? 2 : 1);
  // B: [Wp[v]; Wp[v]; 0] columns c0..c0+ncol -- ONCE per CTA: the CTA is persistent over the patch blocks blockIdx.y,
  // blockIdx.y + gridDim.y, ... of its (variable, column chunk).  One CTA per patch block spent ~2 us of its ~5.5 us in this
  // load and in the drain of its last stores with nothing else of its own in flight (3 CTAs per SM): 0.87 ms for 3 GB.
  for (int idx = threadIdx.x; idx < KP * (DCH / 8); idx += NT) {
    const int k = idx / (DCH / 8), ch = idx - k * (DCH / 8);
    uint4 val = make_uint4(0, 0, 0, 0);
    if (k < 2 * P2 && ch * 8 < ncol) val = *reinterpret_cast<const uint4*>(Wp + ((size_t)v * P2 + (k % P2)) * d.D + c0 + ch * 8);
    *reinterpret_cast<uint4*>(sB + k * BROW + ch * 16) = val;
  }
  if (2 * P2 < KP) {
    constexpr int PAD = KP - 2 * P2 > 0 ? KP - 2 * P2 : 1;
    for (int idx = threadIdx.x; idx < PT * PAD; idx += NT)
      *reinterpret_cast<bf16*>(sA + (idx / PAD) * AROW + (2 * P2 + idx % PAD) * 2) = __float2bfloat16_rn(0.f);
  }
  // A: [hi | lo | 0] of the pixels.  One thread per (patch, patch row): the (b, i, j) arithmetic is done once per p pixels and
  // the row is one vector load; the rows of the NEXT patch block are requested before the current block is computed.
  constexpr int ITEMS = PT * P / NT > 0 ? PT * P / NT : 1;     // (patch, row) items per thread (PT * P is a multiple of NT or below it)
  float px[ITEMS][P];
  const int gw = d.Wg / P;
  auto fetch = [&](int pb) {
#pragma unroll
    for (int it = 0; it < ITEMS; it++) {
      const int idx = threadIdx.x + it * NT;
#pragma unroll
      for (int dj = 0; dj < P; dj++) px[it][dj] = 0.f;
      const int pr = idx / P, di = idx % P, bl = pb * PT + pr;
      if (idx < PT * P && pb < npb && bl < BL) {
        const int b = bl / L, l = bl - b * L, i = l / gw, jj = l - i * gw;
        const float* src = x + (((size_t)b * d.V + v) * d.Hg + i * P + di) * d.Wg + jj * P;
        if (P == 4) { const float4 q = *reinterpret_cast<const float4*>(src); px[it][0] = q.x; px[it][1 % P] = q.y; px[it][2 % P] = q.z; px[it][3 % P] = q.w; }
        else if (P == 2) { const float2 q = *reinterpret_cast<const float2*>(src); px[it][0] = q.x; px[it][1 % P] = q.y; }
        else px[it][0] = *src;
      }
    }
  };
  const bf16* bias = bp + (size_t)v * d.D + c0;
  const uint32_t sBu = s_u32(sB);
  const uint32_t stg0 = s_u32(smem) + warp * 4096;
  if (TMA_OUT && (s_u32(smem) & 1023u)) __trap();            // the swizzled staging tiles need the 1024-byte aligned base requested above
  // stmatrix row address of this lane: matrix (lane >> 3) = (rows 8 (m & 1) .., n-tile 2 q + (m >> 1)), row lane & 7
  const int mrow = (lane & 7) + ((lane >> 3) & 1) * 8, mnt = lane >> 4;
  uint8_t* sO = sB + KP * BROW + warp * (16 * OROW);        // !TMA_OUT: [16][64 + 8] bf16 per warp
  int nstore = 0;                                            // TMA stores issued by this warp
  fetch(blockIdx.y);
  for (int pb = blockIdx.y; pb < npb; pb += gridDim.y) {
    const int bl0 = pb * PT;
#pragma unroll
    for (int it = 0; it < ITEMS; it++) {
      const int idx = threadIdx.x + it * NT;
      if (idx < PT * P) {
        const int pr = idx / P, di = idx % P;
#pragma unroll
        for (int dj = 0; dj < P; dj++) {
          bf16 hi, lo;
          split_bf16(px[it][dj], hi, lo);
          *reinterpret_cast<bf16*>(sA + pr * AROW + (di * P + dj) * 2) = hi;
          *reinterpret_cast<bf16*>(sA + pr * AROW + (P2 + di * P + dj) * 2) = lo;
        }
      }
    }
    __syncthreads();
    uint32_t af[KP / 16][4];
    {
      const int row = warp * 16 + (lane & 7) + ((lane >> 3) & 1) * 8;
#pragma unroll
      for (int ks = 0; ks < KP / 16; ks++) ldsm4(s_u32(sA) + row * AROW + (ks * 16 + (lane >> 4) * 8) * 2, af[ks]);
    }
    __syncthreads();                                         // sA may be rewritten for the next patch block
    fetch(pb + gridDim.y);                                   // in flight while this block is computed and stored
    const int r0 = bl0 + warp * 16;
    for (int ng = 0; ng < DCH / 64; ng++) {
      if (ng * 64 >= ncol) break;
      if (TMA_OUT) {
        const uint32_t buf = stg0 + (nstore & 1) * 2048;
        if (nstore >= 2) {                                    // the store issued from this buffer two groups ago has read it
          if (lane == 0) asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
          __syncwarp();
        }
#pragma unroll
        for (int j = 0; j < 4; j++) {
          const int np = ng * 4 + j;
          float acc[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
#pragma unroll
          for (int ks = 0; ks < KP / 16; ks++) {
            uint32_t b[4];
            ldB(sBu, ks * 16, np * 16, b);
            mma16816(acc[0], af[ks], b[0], b[1]);
            mma16816(acc[1], af[ks], b[2], b[3]);
          }
          uint32_t pk[4];                                     // (rows 0-7, n-tile 2j), (rows 8-15, 2j), (rows 0-7, 2j+1), (rows 8-15, 2j+1)
#pragma unroll
          for (int nt = 0; nt < 2; nt++) {
            const float2 bb = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(bias + ng * 64 + j * 16 + nt * 8 + 2 * t));
            pk[nt * 2] = pack_bf16(acc[nt][0] + bb.x, acc[nt][1] + bb.y);
            pk[nt * 2 + 1] = pack_bf16(acc[nt][2] + bb.x, acc[nt][3] + bb.y);
          }
          const int chunk = j * 2 + mnt;                      // 16-byte chunk (n-tile) of the 128-byte staging row
          stsm4(buf + mrow * 128 + ((chunk ^ (mrow & 7)) << 4), pk[0], pk[1], pk[2], pk[3]);
        }
        ptx::fence_proxy_async();
        __syncwarp();
        if (lane == 0) {
          tma_store_2d(&tmTok, buf, v * d.D + c0 + ng * 64, r0);    // rows >= B L are clipped by the map
          asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
        nstore++;
      } else {
        // The m16n8 accumulator layout gives a thread 4-byte pieces of 16 different rows: each warp stages 16 rows x 64 columns
        // (+ bias) in shared memory and writes them back as 16-byte pieces, 8 lanes covering 128 contiguous bytes of a token row.
#pragma unroll
        for (int j = 0; j < 4; j++) {
          const int np = ng * 4 + j;
          float acc[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
#pragma unroll
          for (int ks = 0; ks < KP / 16; ks++) {
            uint32_t b[4];
            ldB(sBu, ks * 16, np * 16, b);
            mma16816(acc[0], af[ks], b[0], b[1]);
            mma16816(acc[1], af[ks], b[2], b[3]);
          }
#pragma unroll
          for (int nt = 0; nt < 2; nt++) {
            const int cl = j * 16 + nt * 8 + 2 * t;           // column inside the 64-column group
            float2 bb = make_float2(0.f, 0.f);
            if (ng * 64 + cl < ncol) bb = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(bias + ng * 64 + cl));
            *reinterpret_cast<uint32_t*>(sO + g * OROW + cl * 2) = pack_bf16(acc[nt][0] + bb.x, acc[nt][1] + bb.y);
            *reinterpret_cast<uint32_t*>(sO + (g + 8) * OROW + cl * 2) = pack_bf16(acc[nt][2] + bb.x, acc[nt][3] + bb.y);
          }
        }
        __syncwarp();
#pragma unroll
        for (int q = 0; q < 4; q++) {
          const int row = q * 4 + (lane >> 3), ch = lane & 7;
          const int col = ng * 64 + ch * 8;
          if (r0 + row < BL && col < ncol)
            *reinterpret_cast<uint4*>(tok + ((size_t)(r0 + row) * d.V + v) * d.D + c0 + col) =
                *reinterpret_cast<const uint4*>(sO + row * OROW + ch * 16);
        }
        __syncwarp();
      }
    }
  }
  if (TMA_OUT && lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");   // the staging tiles outlive the stores
}

// ---------------------------------------------------------------- backward ---------------------------------
// accW[v, r, c] += sum_patches pix[patch, r] dtok[patch, v, c];  accB[v, c] += sum_patches dtok[patch, v, c]
// TMA_IN (D % 64 == 0): the dtok rows of a chunk arrive as eight [16 patches x 64 columns] TMA boxes (128B swizzle; warp w's 64
// columns = box w) issued by one thread, instead of four cp.async per thread with their address arithmetic (the kernel was
// issue-bound: 498 M warp instructions for 3 GB at 52 % issue-active, profiles/r1_twocall_front.md).
template <int P2, bool TMA_IN>
__global__ void __launch_bounds__(NT) tok_bwd_tc_kernel(orbit_embed_desc d, const float* __restrict__ x,
    const bf16* __restrict__ dtok, float* __restrict__ accW, float* __restrict__ accB, int L, int patches_per_cta,
    const __grid_constant__ CUtensorMap tmTok) {
  constexpr int STG = 4, KC = 16;                         // ring stages; patches per k-chunk
  constexpr int STB = TMA_IN ? KC * DCH * 2 : KC * BROW;   // bytes of a stage of dtok rows (TMA: 8 swizzled 2 KB boxes)
  extern __shared__ __align__(1024) uint8_t smem[];
  uint8_t* sB = smem;                                     // [STG] stages of dtok rows
  float* sP = reinterpret_cast<float*>(smem + STG * STB);  // [STG][KC][16] pixels (fp32)
  __shared__ __align__(8) uint64_t full_bar[STG];
  if (TMA_IN) {
    if (s_u32(smem) & 1023u) __trap();
    if (threadIdx.x == 0) {
      for (int i = 0; i < STG; i++) ptx::mbar_init(s_u32(&full_bar[i]), 1);
      ptx::fence_barrier_init();
    }
    __syncthreads();
  }
  // blockIdx.x = (v, column chunk): CTAs that run together read neighbouring 1 KB pieces of the same token rows
  const int nz = gridDim.x / d.V;
  const int v = blockIdx.x / nz, c0 = (blockIdx.x - v * nz) * DCH;
  const int BL = d.B * L;
  const int p0 = blockIdx.y * patches_per_cta, p1 = min(BL, p0 + patches_per_cta);
  const int nchunks = (p1 - p0 + KC - 1) / KC;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int ncol = min(DCH, d.D - c0);

  // patch grid position of this thread's pixel for the next chunk to be loaded (load() is called with ci = 0, 1, 2, ...)
  constexpr int P = P2 == 16 ? 4 : (P2 == 4 ? 2 : 1);
  const int gw = d.Wg / P, gh = d.Hg / P;
  int pb, pi, pj;
  {
    const int bl = p0 + (threadIdx.x >> 4);
    pb = bl / L;
    const int l = bl - pb * L;
    pi = l / gw; pj = l - pi * gw;
  }
  const int nblk = (ncol + 63) / 64;                       // 64-column boxes of this CTA's chunk
  auto load = [&](int ci) {
    const int st = ci % STG, base = p0 + ci * KC;
    if (TMA_IN) {
      if (threadIdx.x == 0) {                                // rows >= B L read as zero; the patch range of a CTA is a multiple of KC
        const uint32_t bar = s_u32(&full_bar[st]);
        ptx::mbar_expect_tx(bar, nblk * KC * 128);
        for (int bk = 0; bk < nblk; bk++)
          ptx::tma_load_2d(s_u32(sB + st * STB + bk * (KC * 128)), &tmTok, bar, v * d.D + c0 + bk * 64, base);
      }
    } else
    for (int idx = threadIdx.x; idx < KC * (DCH / 8); idx += NT) {
      const int k = idx / (DCH / 8), ch = idx - k * (DCH / 8);
      const uint32_t dst = s_u32(sB + (st * KC + k) * BROW + ch * 16);
      if (base + k < p1 && ch * 8 < ncol) cp_async16(dst, dtok + ((size_t)(base + k) * d.V + v) * d.D + c0 + ch * 8);
      else *reinterpret_cast<uint4*>(sB + (st * KC + k) * BROW + ch * 16) = make_uint4(0, 0, 0, 0);
    }
    {
      // 16 x 16 pixels per chunk, asynchronously like the dtok rows (a plain load + st.shared stalled every warp for a
      // full memory latency per chunk: the ring never ran ahead)
      const int k = threadIdx.x >> 4, r = threadIdx.x & 15;
      const bool ok = r < P2 && base + k < p1;
      const float* src = x;
      if (ok) src = x + (((size_t)pb * d.V + v) * d.Hg + pi * P + r / P) * d.Wg + pj * P + r % P;
      // this thread's patch of the next chunk: (b, i, j) advanced by KC patches without divisions
      pj += KC;
      while (pj >= gw) { pj -= gw; pi++; }
      while (pi >= gh) { pi -= gh; pb++; }
      cp_async4(s_u32(sP + (st * KC + k) * 16 + r), src, ok ? 4 : 0);
    }
    cp_commit();
  };

  float aw[8][4], ab[8][4];
#pragma unroll
  for (int i = 0; i < 8; i++) { aw[i][0] = aw[i][1] = aw[i][2] = aw[i][3] = 0.f; ab[i][0] = ab[i][1] = ab[i][2] = ab[i][3] = 0.f; }
  uint32_t ones[4];
  ones[0] = (g == 0) ? 0x3F803F80u : 0u;                   // row 0 of the A tile = 1.0 (bf16 pair), other rows 0
  ones[1] = 0u; ones[2] = ones[0]; ones[3] = 0u;

  for (int i = 0; i < STG - 1; i++) { if (i < nchunks) load(i); else cp_commit(); }
  for (int ci = 0; ci < nchunks; ci++) {
    cp_wait<STG - 2>();
    __syncthreads();
    if (ci + STG - 1 < nchunks) load(ci + STG - 1); else cp_commit();
    const int st = ci % STG;
    // A fragments (rows = pixel index r, cols = patch k) straight from the pixel tile, split hi / lo
    const float* pt = sP + st * KC * 16;
    uint32_t ah[4], al[4];
    split_pair(pt[(2 * t) * 16 + g], pt[(2 * t + 1) * 16 + g], ah[0], al[0]);
    split_pair(pt[(2 * t) * 16 + g + 8], pt[(2 * t + 1) * 16 + g + 8], ah[1], al[1]);
    split_pair(pt[(2 * t + 8) * 16 + g], pt[(2 * t + 9) * 16 + g], ah[2], al[2]);
    split_pair(pt[(2 * t + 8) * 16 + g + 8], pt[(2 * t + 9) * 16 + g + 8], ah[3], al[3]);
    const uint32_t bt = s_u32(sB + st * STB);
    if (TMA_IN) {
      if (warp >= nblk) continue;                            // this warp's box was not loaded (columns >= D): nothing to add
      ptx::mbar_wait(s_u32(&full_bar[st]), (ci / STG) & 1);
    }
#pragma unroll
    for (int np = 0; np < 4; np++) {                       // this warp's 64 columns = 4 pairs of n-tiles
      uint32_t b[4];
      if (TMA_IN) {                                          // box `warp`: [16 rows x 128 B], 16-byte chunks XOR-swizzled with (row & 7)
        const int row = (lane & 7) + ((lane >> 3) & 1) * 8, chunk = np * 2 + (lane >> 4);
        ldsm4t(bt + warp * (KC * 128) + row * 128 + ((chunk ^ (row & 7)) << 4), b);
      } else
      ldB(bt, 0, warp * 64 + np * 16, b);
      mma16816(aw[2 * np], ah, b[0], b[1]);     mma16816(aw[2 * np + 1], ah, b[2], b[3]);
      mma16816(aw[2 * np], al, b[0], b[1]);     mma16816(aw[2 * np + 1], al, b[2], b[3]);
      mma16816(ab[2 * np], ones, b[0], b[1]);   mma16816(ab[2 * np + 1], ones, b[2], b[3]);
    }
  }
#pragma unroll
  for (int nt = 0; nt < 8; nt++) {
    const int col = warp * 64 + nt * 8 + 2 * t;
    if (col < ncol) {
      if (g < P2) {
        atomicAdd(accW + ((size_t)v * P2 + g) * d.D + c0 + col, aw[nt][0]);
        atomicAdd(accW + ((size_t)v * P2 + g) * d.D + c0 + col + 1, aw[nt][1]);
      }
      if (g + 8 < P2) {
        atomicAdd(accW + ((size_t)v * P2 + g + 8) * d.D + c0 + col, aw[nt][2]);
        atomicAdd(accW + ((size_t)v * P2 + g + 8) * d.D + c0 + col + 1, aw[nt][3]);
      }
      if (g == 0) {
        atomicAdd(accB + (size_t)v * d.D + c0 + col, ab[nt][0]);
        atomicAdd(accB + (size_t)v * d.D + c0 + col + 1, ab[nt][1]);
      }
    }
  }
}
__device__ __forceinline__ void bulk_wait_read1() { asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory"); }
// ---------------------------------------------------------------- forward on tcgen05 ------------------------
// tok[patch, v, c0 .. c0 + 512) = [hi | lo | 1] (A: 128 patches x 48, K-major, built by the worker warps) . [Wp[v] ; Wp[v] ; bp[v]]
// (B: 48 x 512 columns, MN-major, resident for the CTA's life), two N = 256 halves per stage of 128 patches into the two halves of
// tensor memory; 16 worker warps (TMEM lane quarter x 64 of a half's 256 columns) drain them: fp32 -> bf16 -> a warp-private
// swizzled [32 rows x 64 columns] staging tile -> one TMA box store (rows >= B L clipped by the map), two tiles in flight per warp.
constexpr int PT5 = 128;                       // patches per stage
constexpr int WB5 = 48 * 128;                  // one 64-column block of the B operand: 48 k-rows x 128 bytes
constexpr int AT5F = PT5 * 128;                // A tile: 128 patches x 64 k (48 used) bf16, K-major
constexpr int OT5F = 32 * 128;                 // staging tile of a warp
constexpr int NW5F = 16;
constexpr int NT5F = 32 + NW5F * 32;           // warp 0 MMA issuer, warps 1..16 workers
constexpr size_t SMEM_TOKF5 = 1024 + 8 * WB5 + 2 * AT5F + NW5F * 2 * OT5F + 64;
__global__ void __launch_bounds__(NT5F, 1) tok_fwd_t5_kernel(orbit_embed_desc d, const float* __restrict__ x,
    const bf16* __restrict__ Wp, const bf16* __restrict__ bp, int L, int patches_per_cta, const __grid_constant__ CUtensorMap tmTok, int STORE_HINT) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = smem_raw + ((1024 - (s_u32(smem_raw) & 1023)) & 1023);
  uint8_t* pW = smem;                          // [8][48][128 B]
  uint8_t* pA = pW + 8 * WB5;                  // [2][128][128 B]
  const uint32_t sW = s_u32(pW), sA = s_u32(pA), sO = sA + 2 * AT5F;
  const uint32_t a_full0 = sO + NW5F * 2 * OT5F, a_empty0 = a_full0 + 16, t_full0 = a_empty0 + 16, t_empty0 = t_full0 + 16, tslot = t_empty0 + 16;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int P = d.p, P2 = P * P;
  const int nz = gridDim.x / d.V;
  const int v = blockIdx.x / nz, c0 = (blockIdx.x - v * nz) * DCH;
  const int BL = d.B * L;
  const int p0 = blockIdx.y * patches_per_cta, p1 = min(BL, p0 + patches_per_cta);
  const int nst = (p1 - p0 + PT5 - 1) / PT5;
  const int ncol = min(DCH, d.D - c0), nhalf = (ncol + 255) / 256;

  // B operand, once: k-rows 0..P2-1 and 16..16+P2-1 = Wp[v] (the hi and the lo product), row 32 = bp[v], the rest zero
  for (int idx = threadIdx.x; idx < 48 * (DCH / 8); idx += NT5F) {
    const int k = idx / (DCH / 8), ch = idx - k * (DCH / 8), col = ch * 8;
    uint4 val = make_uint4(0, 0, 0, 0);
    if (col < ncol) {
      if ((k & 15) < P2 && k < 32) val = *reinterpret_cast<const uint4*>(Wp + ((size_t)v * P2 + (k & 15)) * d.D + c0 + col);
      else if (k == 32) val = *reinterpret_cast<const uint4*>(bp + (size_t)v * d.D + c0 + col);
    }
    *reinterpret_cast<uint4*>(pW + (col >> 6) * WB5 + k * 128 + ((((col & 63) >> 3) ^ (k & 7)) << 4)) = val;
  }
  for (int i = threadIdx.x; i < 2 * AT5F / 16; i += NT5F) reinterpret_cast<uint4*>(pA)[i] = make_uint4(0, 0, 0, 0);
  if (threadIdx.x == 0) {
    for (int i = 0; i < 2; i++) {
      ptx::mbar_init(a_full0 + 8 * i, NW5F); ptx::mbar_init(a_empty0 + 8 * i, 1);
      ptx::mbar_init(t_full0 + 8 * i, 1); ptx::mbar_init(t_empty0 + 8 * i, NW5F);
    }
    ptx::fence_barrier_init();
  }
  if (warp == 0) { ptx::tmem_alloc(tslot, 512); ptx::tmem_relinquish(); }
  ptx::fence_proxy_async();
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem) : "r"(tslot));

  if (warp == 0) {
    if (lane == 0) {
      constexpr uint32_t idesc = ptx::make_idesc_bf16(128, 256, 0, 1);
      for (int ci = 0; ci < nst; ci++) {
        const uint32_t ab = ci & 1;
        ptx::mbar_wait(a_full0 + 8 * ab, (ci >> 1) & 1);
        for (int hf = 0; hf < nhalf; hf++) {
          ptx::mbar_wait(t_empty0 + 8 * hf, (ci & 1) ^ 1);
          ptx::tc_fence_after();
#pragma unroll
          for (int ks = 0; ks < 3; ks++)
            ptx::mma_f16_ss(tmem + hf * 256, ptx::make_smem_desc(sA + ab * AT5F + ks * 32, 16, 1024),
                            ptx::make_smem_desc(sW + hf * 4 * WB5 + ks * 2048, WB5, 1024), idesc, ks != 0);
          ptx::mma_commit(t_full0 + 8 * hf);
        }
        ptx::mma_commit(a_empty0 + 8 * ab);
      }
    }
  } else {
    const int w = warp - 1, tt = threadIdx.x - 32, k = tt >> 2, sub = tt & 3;       // pixel tile: thread = (patch k, quarter of its pixels)
    const int quarter = warp & 3, cb = w >> 2;                                        // drain: TMEM lane quarter, 64-column block of a half
    const uint32_t lane_off = (uint32_t)(quarter * 32) << 16;
    const int gw = d.Wg / P;
    const int RP = P2 >= 4 ? P2 / 4 : 1, r0 = sub * RP;
    float px[4] = {0.f, 0.f, 0.f, 0.f};
    bool valid = false;
    auto fetch = [&](int ci) {
      const int bl = p0 + ci * PT5 + k;
      valid = ci < nst && bl < p1;
#pragma unroll
      for (int q = 0; q < 4; q++) px[q] = 0.f;
      if (valid && r0 < P2) {
        const int b = bl / L, l = bl - b * L, pi = l / gw, pj = l - pi * gw;
        const float* base = x + (((size_t)b * d.V + v) * d.Hg + pi * P) * d.Wg + pj * P;
        if (P == 4) {
          const float4 f = __ldg(reinterpret_cast<const float4*>(base + (size_t)sub * d.Wg));
          px[0] = f.x; px[1] = f.y; px[2] = f.z; px[3] = f.w;
        } else {
          px[0] = __ldg(base + (size_t)(r0 / P) * d.Wg + r0 % P);
        }
      }
    };
    fetch(0);
    uint32_t ob = 0;                                         // this warp's staging tile in use
    const uint64_t pol = ptx::l2_policy(STORE_HINT == 2 ? 2 : 1);
    auto build = [&](int ci) {                               // A tile of stage ci from the pixels fetched for it
      const uint32_t ab = ci & 1;
      ptx::mbar_wait(a_empty0 + 8 * ab, ((ci >> 1) & 1) ^ 1);
      uint8_t* at = pA + ab * AT5F + k * 128;                // row k: [hi (k 0..15) | lo (16..31) | 1 (32)] as 16-byte chunks ^ (k & 7)
#pragma unroll
      for (int q = 0; q < 4; q++) {
        const int r = r0 + q;
        if (q < RP && r < P2) {
          const bf16 hi = __float2bfloat16_rn(px[q]);
          const bf16 lo = __float2bfloat16_rn(px[q] - __bfloat162float(hi));
          *reinterpret_cast<bf16*>(at + (((r >> 3) ^ (k & 7)) << 4) + (r & 7) * 2) = hi;
          *reinterpret_cast<bf16*>(at + ((((16 + r) >> 3) ^ (k & 7)) << 4) + (r & 7) * 2) = lo;
        }
      }
      if (sub == 0) *reinterpret_cast<bf16*>(at + ((4 ^ (k & 7)) << 4)) = __float2bfloat16_rn(valid ? 1.f : 0.f);
      ptx::fence_proxy_async();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(a_full0 + 8 * ab);
    };
    for (int ci = 0; ci < nst; ci++) {
      // (building the NEXT stage's operand before draining this one, so that its products overlap the drain, measured SLOWER:
      // 625 vs 568-592 us at C3)
      build(ci);
      fetch(ci + 1);
      for (int hf = 0; hf < nhalf; hf++) {
        ptx::mbar_wait(t_full0 + 8 * hf, ci & 1);
        ptx::tc_fence_after();
        uint32_t o[64];
        ptx::tmem_ld_32x32(tmem + hf * 256 + cb * 64 + lane_off, o);
        ptx::tmem_ld_32x32(tmem + hf * 256 + cb * 64 + 32 + lane_off, o + 32);
        ptx::tmem_ld_wait();
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(t_empty0 + 8 * hf);
        const int col = hf * 256 + cb * 64;
        if (col < ncol) {
          const uint32_t so = sO + (w * 2 + ob) * OT5F;
          if (lane == 0) bulk_wait_read1();                  // the store issued two tiles ago has left this buffer
          __syncwarp();
#pragma unroll
          for (int c = 0; c < 8; c++) {
            const uint32_t addr = so + lane * 128 + ((c ^ (lane & 7)) << 4);
            asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr),
                         "r"(pack_bf16(__uint_as_float(o[c * 8]), __uint_as_float(o[c * 8 + 1]))),
                         "r"(pack_bf16(__uint_as_float(o[c * 8 + 2]), __uint_as_float(o[c * 8 + 3]))),
                         "r"(pack_bf16(__uint_as_float(o[c * 8 + 4]), __uint_as_float(o[c * 8 + 5]))),
                         "r"(pack_bf16(__uint_as_float(o[c * 8 + 6]), __uint_as_float(o[c * 8 + 7]))) : "memory");
          }
          ptx::fence_proxy_async();
          __syncwarp();
          if (lane == 0) {
            if (STORE_HINT)
              asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group.L2::cache_hint [%0, {%2, %3}], [%1], %4;" ::"l"(&tmTok), "r"(so),
                           "r"(v * d.D + c0 + col), "r"(p0 + ci * PT5 + quarter * 32), "l"(pol) : "memory");
            else tma_store_2d(&tmTok, so, v * d.D + c0 + col, p0 + ci * PT5 + quarter * 32);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
          }
          ob ^= 1;
        }
      }
    }
    if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 0) { ptx::tc_fence_after(); ptx::tmem_dealloc(tmem, 512); }
}

// ---------------------------------------------------------------- backward on tcgen05 -----------------------
// dWp^T[d, r] = sum over patches of dtok[patch, v, d] pix[patch, r]: M = d (the dtok tiles as they arrive from TMA, an MN-major A
// operand), K = patches, N = 48 pixel-side columns (16 bf16 "hi" parts of the p^2 pixels, 16 "lo" residuals, a column of ones for
// dbp, zeros).  The mma.sync kernel above spends its warps on HMMA (6 per 16 patches x 16 columns, a third of them for the ones
// row: legacy tensor pipe 38 % busy, 65 % of hbm_gbs); here one thread issues 16 tcgen05.mma per stage of 64 patches x 512
// columns, eight warps only build the small pixel tile (hi / lo split, K-major, 128B swizzle) and the accumulators
// [128 lanes x 48 columns] per 128-column group stay in tensor memory for the CTA's whole patch range.
constexpr int KS5 = 64;                        // patches per stage
constexpr int BOX5 = KS5 * 128;                // one [64 patches x 64 columns] TMA box
constexpr int NB5 = 48;                        // columns of the pixel-side operand
constexpr int BT5B = NB5 * 128;                // its tile: [48 rows (n) x 64 patches (k)] bf16, K-major
constexpr int ST5 = 3;
constexpr int NT5B = 64 + 256;                 // warp 0 TMA producer, warp 1 MMA issuer, warps 2..9 pixel tile / epilogue
constexpr size_t SMEM_TOKB5 = 1024 + (size_t)ST5 * (8 * BOX5 + BT5B) + 64;
__global__ void __launch_bounds__(NT5B, 1) tok_bwd_t5_kernel(orbit_embed_desc d, const float* __restrict__ x,
    float* __restrict__ accW, float* __restrict__ accB, int L, int patches_per_cta, const __grid_constant__ CUtensorMap tmTok) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = smem_raw + ((1024 - (s_u32(smem_raw) & 1023)) & 1023);
  const uint32_t sA = s_u32(smem), sBt = sA + ST5 * 8 * BOX5;
  const uint32_t full0 = sBt + ST5 * BT5B, bfull0 = full0 + 8 * ST5, empty0 = bfull0 + 8 * ST5, done = empty0 + 8 * ST5, tslot = done + 8;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int P = d.p, P2 = P * P;
  const int nz = gridDim.x / d.V;
  const int v = blockIdx.x / nz, c0 = (blockIdx.x - v * nz) * DCH;
  const int BL = d.B * L;
  const int p0 = blockIdx.y * patches_per_cta, p1 = min(BL, p0 + patches_per_cta);
  const int nst = (p1 - p0 + KS5 - 1) / KS5;
  const int ncol = min(DCH, d.D - c0), nblk = ncol / 64, ncg = (ncol + 127) / 128;

  for (int i = threadIdx.x; i < ST5 * BT5B / 16; i += NT5B) reinterpret_cast<uint4*>(smem + ST5 * 8 * BOX5)[i] = make_uint4(0, 0, 0, 0);
  if (threadIdx.x == 0) {
    for (int i = 0; i < ST5; i++) { ptx::mbar_init(full0 + 8 * i, 1); ptx::mbar_init(bfull0 + 8 * i, 8); ptx::mbar_init(empty0 + 8 * i, 1); }
    ptx::mbar_init(done, 1);
    ptx::fence_barrier_init();
  }
  if (warp == 1) { ptx::tmem_alloc(tslot, 256); ptx::tmem_relinquish(); }
  ptx::fence_proxy_async();
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem) : "r"(tslot));

  if (warp == 0) {
    if (lane == 0) {
      int st = 0; uint32_t ph = 0;
      for (int ci = 0; ci < nst; ci++) {
        ptx::mbar_wait(empty0 + 8 * st, ph ^ 1);
        ptx::mbar_expect_tx(full0 + 8 * st, nblk * BOX5);
        for (int bk = 0; bk < nblk; bk++)                    // rows >= B L read as zero
          ptx::tma_load_2d(sA + (st * 8 + bk) * BOX5, &tmTok, full0 + 8 * st, v * d.D + c0 + bk * 64, p0 + ci * KS5);
        if (++st == ST5) { st = 0; ph ^= 1; }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      constexpr uint32_t idesc = ptx::make_idesc_bf16(128, NB5, 1, 0);
      int st = 0; uint32_t ph = 0;
      for (int ci = 0; ci < nst; ci++) {
        ptx::mbar_wait(full0 + 8 * st, ph);
        ptx::mbar_wait(bfull0 + 8 * st, ph);
        ptx::tc_fence_after();
        for (int cg = 0; cg < ncg; cg++)
#pragma unroll
          for (int ks = 0; ks < KS5 / 16; ks++)
            ptx::mma_f16_ss(tmem + cg * NB5, ptx::make_smem_desc(sA + (st * 8 + cg * 2) * BOX5 + ks * 2048, BOX5, 1024),
                            ptx::make_smem_desc(sBt + st * BT5B + ks * 32, 16, 1024), idesc, (ci | ks) != 0);
        ptx::mma_commit(empty0 + 8 * st);
        if (++st == ST5) { st = 0; ph ^= 1; }
      }
      ptx::mma_commit(done);
    }
  } else {
    // pixel tile of a stage: thread = (patch k of the stage, quarter of its pixels), loaded one stage ahead
    const int tt = threadIdx.x - 64, k = tt >> 2, sub = tt & 3;
    const int gw = d.Wg / P;
    const int RP = P2 >= 4 ? P2 / 4 : 1, r0 = sub * RP;                      // this thread's pixels r0 .. r0 + RP - 1 (if < P2)
    float px[4] = {0.f, 0.f, 0.f, 0.f};
    bool valid = false;
    auto fetch = [&](int ci) {
      const int bl = p0 + ci * KS5 + k;
      valid = ci < nst && bl < p1;
#pragma unroll
      for (int q = 0; q < 4; q++) px[q] = 0.f;
      if (valid && r0 < P2) {
        const int b = bl / L, l = bl - b * L, pi = l / gw, pj = l - pi * gw;
        const float* base = x + (((size_t)b * d.V + v) * d.Hg + pi * P) * d.Wg + pj * P;
        if (P == 4) {                                        // r0 = 4 sub: one pixel row of the patch, 16 aligned bytes
          const float4 f = __ldg(reinterpret_cast<const float4*>(base + (size_t)sub * d.Wg));
          px[0] = f.x; px[1] = f.y; px[2] = f.z; px[3] = f.w;
        } else {
          px[0] = __ldg(base + (size_t)(r0 / P) * d.Wg + r0 % P);
        }
      }
    };
    fetch(0);
    int st = 0; uint32_t ph = 0;
    for (int ci = 0; ci < nst; ci++) {
      ptx::mbar_wait(empty0 + 8 * st, ph ^ 1);               // the products of the stage that used this tile have completed
      uint8_t* bt = smem + ST5 * 8 * BOX5 + st * BT5B;
#pragma unroll
      for (int q = 0; q < 4; q++) {
        const int r = r0 + q;
        if (q < RP && r < P2) {
          const bf16 hi = __float2bfloat16_rn(px[q]);
          const bf16 lo = __float2bfloat16_rn(px[q] - __bfloat162float(hi));
          *reinterpret_cast<bf16*>(bt + r * 128 + (((k >> 3) ^ (r & 7)) << 4) + (k & 7) * 2) = hi;
          *reinterpret_cast<bf16*>(bt + (16 + r) * 128 + (((k >> 3) ^ ((16 + r) & 7)) << 4) + (k & 7) * 2) = lo;
        }
      }
      if (sub == 0) *reinterpret_cast<bf16*>(bt + 32 * 128 + (((k >> 3) ^ 0) << 4) + (k & 7) * 2) = __float2bfloat16_rn(valid ? 1.f : 0.f);
      ptx::fence_proxy_async();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(bfull0 + 8 * st);
      fetch(ci + 1);
      if (++st == ST5) { st = 0; ph ^= 1; }
    }
    // accumulators -> fp32 atomics: thread = column d of a 128-column group; the two warps of a TMEM lane quarter split the groups
    ptx::mbar_wait(done, 0);
    ptx::tc_fence_after();
    const int quarter = warp & 3, half = (warp - 2) >> 2;
    const uint32_t lane_off = (uint32_t)(quarter * 32) << 16;
    for (int cg = half; cg < ncg; cg += 2) {
      uint32_t a[NB5];
      ptx::tmem_ld_32x16(tmem + cg * NB5 + lane_off, a);
      ptx::tmem_ld_32x16(tmem + cg * NB5 + 16 + lane_off, a + 16);
      ptx::tmem_ld_32x16(tmem + cg * NB5 + 32 + lane_off, a + 32);
      ptx::tmem_ld_wait();
      const int col = cg * 128 + quarter * 32 + lane;
      if (col < ncol && nst > 0) {
#pragma unroll
        for (int r = 0; r < 16; r++)
          if (r < P2) atomicAdd(accW + ((size_t)v * P2 + r) * d.D + c0 + col, __uint_as_float(a[r]) + __uint_as_float(a[16 + r]));
        atomicAdd(accB + (size_t)v * d.D + c0 + col, __uint_as_float(a[32]));
      }
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 1) { ptx::tc_fence_after(); ptx::tmem_dealloc(tmem, 256); }
}
}  // namespace

bool tokenize_tc_supported(const orbit_embed_desc& d) {
  return d.dtype == ORBIT_BF16 && (d.p == 1 || d.p == 2 || d.p == 4) && d.D % 16 == 0;
}

// tok seen as a bf16 matrix [B L rows, V D columns]: boxes of 16 rows x 64 columns, 128-byte swizzle
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static int make_tok_map(CUtensorMap* tm, void* tok, long long rows, long long cols,
                        CUtensorMapL2promotion promo = CU_TENSOR_MAP_L2_PROMOTION_NONE, int box_rows = 16) {
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
  cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)cols * 2};
  cuuint32_t box[2] = {64, (cuuint32_t)box_rows};
  cuuint32_t es[2] = {1, 1};
  CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, tok, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   CU_TENSOR_MAP_SWIZZLE_128B, promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { set_error("tokenize: cuTensorMapEncodeTiled failed (%d)", (int)r); return ORBIT_ERR_CUDA; }
  return ORBIT_OK;
}

int tokenize_fwd_tc(const orbit_embed_desc& d, const float* x, const void* Wp, const void* bp, void* tok, cudaStream_t s) {
  const int L = (d.Hg / d.p) * (d.Wg / d.p), P2 = d.p * d.p;
  static const int t5_env = [] { const char* e = getenv("ORBIT_TOK_T5"); return (e && e[0] == '0') ? 0 : 1; }();
  if (t5_env && d.D % 64 == 0 && (long long)d.V * d.D < (1ll << 31) && P2 <= 16) {
    const long long BL = (long long)d.B * L;
    const int nz = cdiv(d.D, DCH);
    int splits = 1;                      // one CTA per SM: patch splits so that the grid fills whole waves of the SMs
    {
      const long long slots = num_sms(), per = (long long)d.V * nz;
      double best = 0.0;
      for (int sp = 1; sp <= 32; sp++) {
        if (cdiv(BL, sp) < 4 * PT5 && sp > 1) break;         // keep at least 4 stages per CTA
        const long long n = per * sp, waves = (n + slots - 1) / slots;
        const double eff = (double)n / (double)(waves * slots);
        if (eff > best + 1e-9) { best = eff; splits = sp; }
        if (eff >= 0.97) { splits = sp; break; }
      }
    }
    int ppc = cdiv(BL, splits);
    ppc = ((ppc + PT5 - 1) / PT5) * PT5;
    dim3 grid(d.V * nz, cdiv(BL, ppc));
    CUtensorMap tm;
    ORBIT_TRY(make_tok_map(&tm, tok, BL, (long long)d.V * d.D, CU_TENSOR_MAP_L2_PROMOTION_NONE, 32));
    ORBIT_SMEM_ATTR(tok_fwd_t5_kernel, SMEM_TOKF5);
    static const int hint_env = [] { const char* e = getenv("ORBIT_TOK_HINT"); return e ? atoi(e) : 1; }();
    tok_fwd_t5_kernel<<<grid, NT5F, SMEM_TOKF5, s>>>(d, x, (const bf16*)Wp, (const bf16*)bp, L, ppc, tm, hint_env);
    ORBIT_LAUNCH_CHECK();
    return ORBIT_OK;
  }
  // persistent over the patch blocks: grid.y CTAs per (variable, column chunk), chosen so that the grid fills whole waves
  // of 3 CTAs per SM (the shared-memory limit) as evenly as possible, 4+ patch blocks per CTA when there are enough
  const int gx = d.V * cdiv(d.D, DCH), npb = cdiv((long long)d.B * L, 128);
  int gy = 1;
  {
    const long long slots = (long long)num_sms() * 3;
    double best = -1.0;
    for (int c = 1; c <= npb && c <= 64; c++) {
      const int per = cdiv(npb, c);                          // patch blocks of the longest CTA
      const long long waves = ((long long)gx * c + slots - 1) / slots;
      const double eff = (double)gx * npb / ((double)waves * slots * per);      // useful / available block slots
      if (per < (npb < 4 ? npb : 4)) break;                  // keep at least 4 patch blocks per CTA (the point of the loop)
      if (eff > best + 1e-9) { best = eff; gy = c; }
    }
  }
  dim3 grid(gx, gy);
  const bool tma_out = d.D % 64 == 0 && (long long)d.V * d.D < (1ll << 31);
  CUtensorMap tm;
  memset(&tm, 0, sizeof(tm));
  if (tma_out) ORBIT_TRY(make_tok_map(&tm, tok, (long long)d.B * L, (long long)d.V * d.D));
#define TF(P, K) do {                                                                                         \
    if (tma_out) {                                                                                            \
      const size_t smb = (size_t)(NT / 32) * 4096 + (size_t)128 * (K + 8) * 2 + (size_t)K * BROW;              \
      ORBIT_SMEM_ATTR((tok_fwd_tc_kernel<P, K, true>), smb);                                                  \
      tok_fwd_tc_kernel<P, K, true><<<grid, NT, smb, s>>>(d, x, (const bf16*)Wp, (const bf16*)bp, (bf16*)tok, L, tm); \
    } else {                                                                                                  \
      const size_t smb = (size_t)128 * (K + 8) * 2 + (size_t)K * BROW + (size_t)(NT / 32) * 16 * OROW;         \
      ORBIT_SMEM_ATTR((tok_fwd_tc_kernel<P, K, false>), smb);                                                 \
      tok_fwd_tc_kernel<P, K, false><<<grid, NT, smb, s>>>(d, x, (const bf16*)Wp, (const bf16*)bp, (bf16*)tok, L, tm); \
    } } while (0)
  if (P2 == 16) TF(16, 32);
  else if (P2 == 4) TF(4, 16);
  else TF(1, 16);
#undef TF
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int tokenize_bwd_acc_tc(const orbit_embed_desc& d, const float* x, const void* dtok, float* accW, float* accB, cudaStream_t s) {
  const int L = (d.Hg / d.p) * (d.Wg / d.p), P2 = d.p * d.p;
  const long long BL = (long long)d.B * L;
  const int nz = cdiv(d.D, DCH);
  static const int t5_env = [] { const char* e = getenv("ORBIT_TOK_T5"); return (e && e[0] == '0') ? 0 : 1; }();
  if (t5_env && d.D % 64 == 0 && (long long)d.V * d.D < (1ll << 31) && P2 <= 16) {
    // one CTA per SM (192 KB of stages): patch splits so that the grid fills whole waves of the SMs
    int splits = 1;
    {
      const long long slots = num_sms(), per = (long long)d.V * nz;
      double best = 0.0;
      for (int sp = 1; sp <= 32; sp++) {
        if (cdiv(BL, sp) < 4 * KS5 && sp > 1) break;         // keep at least 4 stages per CTA
        const long long n = per * sp, waves = (n + slots - 1) / slots;
        const double eff = (double)n / (double)(waves * slots);
        if (eff > best + 1e-9) { best = eff; splits = sp; }
        if (eff >= 0.97) { splits = sp; break; }
      }
    }
    int ppc = cdiv(BL, splits);
    ppc = ((ppc + KS5 - 1) / KS5) * KS5;
    dim3 grid(d.V * nz, cdiv(BL, ppc));
    CUtensorMap tm;
    ORBIT_TRY(make_tok_map(&tm, const_cast<void*>(dtok), BL, (long long)d.V * d.D, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, KS5));
    ORBIT_SMEM_ATTR(tok_bwd_t5_kernel, SMEM_TOKB5);
    tok_bwd_t5_kernel<<<grid, NT5B, SMEM_TOKB5, s>>>(d, x, accW, accB, L, ppc, tm);
    ORBIT_LAUNCH_CHECK();
    return ORBIT_OK;
  }
  // patch splits: the first count whose grid fills whole waves of 2 CTAs per SM to >= 95 % (else the fullest)
  int splits = 1;
  {
    const long long slots = 148 * 2, per = (long long)d.V * nz;
    double best = 0.0;
    for (int sp = 1; sp <= 16; sp++) {
      const long long n = per * sp, waves = (n + slots - 1) / slots;
      const double eff = (double)n / (double)(waves * slots);
      if (eff > best + 1e-9) { best = eff; splits = sp; }
      if (n >= slots * 2 && eff >= 0.95) { splits = sp; break; }
    }
  }
  int ppc = cdiv(BL, splits);
  ppc = ((ppc + 15) / 16) * 16;
  if (ppc < 64) ppc = 64;
  dim3 grid(d.V * nz, cdiv(BL, ppc));
  const bool tma_in = d.D % 64 == 0 && (long long)d.V * d.D < (1ll << 31);
  CUtensorMap tm;
  memset(&tm, 0, sizeof(tm));
  if (tma_in) ORBIT_TRY(make_tok_map(&tm, const_cast<void*>(dtok), BL, (long long)d.V * d.D, CU_TENSOR_MAP_L2_PROMOTION_L2_256B));
  const size_t smb = (size_t)4 * (tma_in ? 16 * DCH * 2 : 16 * BROW) + (size_t)4 * 16 * 16 * sizeof(float);
#define TB(P) do {                                                                                            \
    if (tma_in) {                                                                                             \
      ORBIT_SMEM_ATTR((tok_bwd_tc_kernel<P, true>), smb);                                                     \
      tok_bwd_tc_kernel<P, true><<<grid, NT, smb, s>>>(d, x, (const bf16*)dtok, accW, accB, L, ppc, tm);      \
    } else {                                                                                                  \
      ORBIT_SMEM_ATTR((tok_bwd_tc_kernel<P, false>), smb);                                                    \
      tok_bwd_tc_kernel<P, false><<<grid, NT, smb, s>>>(d, x, (const bf16*)dtok, accW, accB, L, ppc, tm);     \
    } } while (0)
  if (P2 == 16) TB(16);
  else if (P2 == 4) TB(4);
  else TB(1);
#undef TB
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

}  // namespace orbit
