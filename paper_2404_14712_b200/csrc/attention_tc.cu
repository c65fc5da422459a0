// attention_tc.cu -- bf16 tensor-core flash attention, forward and backward (PAPER.md:88 softmax(QK^T)V,
// :114 scaled dot product; readings R8, R19).  No N x N matrix is stored: forward keeps one logsumexp per row,
// backward recomputes the probabilities tile by tile.
//
// Three kernels with one skeleton -- a CTA owns 64 rows (4 warps x 16), sweeps the other index in tiles of 64
// through a cp.async double buffer in XOR-swizzled shared memory, and contracts with mma.sync.m16n8k16 (bf16 in,
// fp32 accumulate, operands via ldmatrix):
//   fwd : rows = queries.  S = Q K^T, online softmax, O += P V.
//   dQ  : rows = queries.  S = Q K^T, dP = dO V^T, dS = P o (dP - delta), dQ += dS K.
//   dKV : rows = keys.     S^T = K Q^T, dP^T = V dO^T, dV += P^T dO, dK += dS^T Q.
// The backward is split in two so that no atomics and no shared-memory transposes are needed (deterministic);
// it costs 7 instead of 5 tile products.  delta = rowsum(dO o O) comes from a small pre-pass.
#include "common.cuh"

namespace orbit {
namespace {

constexpr int BR = 64;       // rows per CTA
constexpr int BC = 64;       // loop-tile rows
constexpr int NT = 128;      // threads

__device__ __forceinline__ uint32_t s_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, int bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(bytes) : "memory");
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

// A [64 x DH] bf16 tile in shared memory, rows of DH*2 bytes, 16-byte chunks XOR-swizzled with (row & 7)
template <int DH>
struct Tile {
  static constexpr int CH = DH / 8;
  static constexpr int BYTES = 64 * DH * 2;
  __device__ static __forceinline__ uint32_t addr(uint32_t base, int row, int chunk) {
    return base + row * (DH * 2) + ((chunk ^ (row & 7)) << 4);
  }
  // rows [row0, row0+64) of a [*, ld] bf16 matrix (column offset col0); rows >= nrows are zero-filled
  __device__ static __forceinline__ void load_async(uint32_t base, const bf16* g, long long ld, int row0, int nrows,
                                                     int col0) {
#pragma unroll
    for (int i = 0; i < 64 * CH / NT; i++) {
      int idx = threadIdx.x + i * NT;
      int r = idx / CH, c = idx - r * CH;
      int gr = row0 + r;
      bool ok = gr < nrows;
      const bf16* src = g + (size_t)(ok ? gr : 0) * ld + col0 + c * 8;
      cp_async16(addr(base, r, c), src, ok ? 16 : 0);
    }
  }
  // A fragments (16 rows starting at r0, 16 k starting at k0) of a row-major tile
  __device__ static __forceinline__ void ldA(uint32_t base, int r0, int k0, uint32_t* a) {
    int lane = threadIdx.x & 31;
    int row = r0 + (lane & 7) + ((lane >> 3) & 1) * 8;
    int chunk = (k0 >> 3) + (lane >> 4);
    ldsm4(addr(base, row, chunk), a);
  }
  // B fragments for C += A * Tile^T : B(k, n) = Tile[n][k]; 16 n starting at n0, 16 k starting at k0
  // r[0], r[1] = (b0, b1) of n-tile n0 ; r[2], r[3] = (b0, b1) of n-tile n0 + 8
  __device__ static __forceinline__ void ldB_kmajor(uint32_t base, int n0, int k0, uint32_t* r) {
    int lane = threadIdx.x & 31;
    int row = n0 + (lane & 7) + (lane >> 4) * 8;
    int chunk = (k0 >> 3) + ((lane >> 3) & 1);
    ldsm4(addr(base, row, chunk), r);
  }
  // B fragments for C += A * Tile : B(k, n) = Tile[k][n]; 16 k starting at k0, 16 n starting at n0
  __device__ static __forceinline__ void ldB_nmajor(uint32_t base, int k0, int n0, uint32_t* r) {
    int lane = threadIdx.x & 31;
    int row = k0 + (lane & 7) + ((lane >> 3) & 1) * 8;
    int chunk = (n0 >> 3) + (lane >> 4);
    ldsm4t(addr(base, row, chunk), r);
  }
};

// C[16 x 64] = A(16 x DH, rows r0.. of tile sa) * (tile sb [64 x DH])^T
template <int DH>
__device__ __forceinline__ void mma_abt(float (*c)[4], uint32_t sa, int r0, uint32_t sb) {
#pragma unroll
  for (int ks = 0; ks < DH / 16; ks++) {
    uint32_t a[4];
    Tile<DH>::ldA(sa, r0, ks * 16, a);
#pragma unroll
    for (int np = 0; np < 4; np++) {
      uint32_t b[4];
      Tile<DH>::ldB_kmajor(sb, np * 16, ks * 16, b);
      mma16816(c[2 * np], a, b[0], b[1]);
      mma16816(c[2 * np + 1], a, b[2], b[3]);
    }
  }
}
// C[16 x DH] += P(16 x 64, register A fragments pf[4][4]) * tile sb [64 x DH]
template <int DH>
__device__ __forceinline__ void mma_pb(float (*c)[4], const uint32_t (*pf)[4], uint32_t sb) {
#pragma unroll
  for (int ks = 0; ks < 4; ks++) {
#pragma unroll
    for (int dp = 0; dp < DH / 16; dp++) {
      uint32_t b[4];
      Tile<DH>::ldB_nmajor(sb, ks * 16, dp * 16, b);
      mma16816(c[2 * dp], pf[ks], b[0], b[1]);
      mma16816(c[2 * dp + 1], pf[ks], b[2], b[3]);
    }
  }
}
// C-fragment layout [8 n-tiles][4] of a 16 x 64 product -> A fragments [4 k-steps][4] (bf16)
__device__ __forceinline__ void c_to_a(const float (*c)[4], uint32_t (*pf)[4]) {
#pragma unroll
  for (int j = 0; j < 4; j++) {
    pf[j][0] = pack_bf16(c[2 * j][0], c[2 * j][1]);
    pf[j][1] = pack_bf16(c[2 * j][2], c[2 * j][3]);
    pf[j][2] = pack_bf16(c[2 * j + 1][0], c[2 * j + 1][1]);
    pf[j][3] = pack_bf16(c[2 * j + 1][2], c[2 * j + 1][3]);
  }
}
// write a warp's 16 x DH fp32 accumulator (scaled) as bf16 into tile `st` rows r0.., then the CTA stores the tile
template <int DH>
__device__ __forceinline__ void stage_rows(uint32_t st, int r0, const float (*c)[4], float s_lo, float s_hi) {
  int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
#pragma unroll
  for (int nt = 0; nt < DH / 8; nt++) {
    uint32_t lo = pack_bf16(c[nt][0] * s_lo, c[nt][1] * s_lo);
    uint32_t hi = pack_bf16(c[nt][2] * s_hi, c[nt][3] * s_hi);
    asm volatile("st.shared.b32 [%0], %1;" ::"r"(Tile<DH>::addr(st, r0 + g, nt) + t * 4), "r"(lo));
    asm volatile("st.shared.b32 [%0], %1;" ::"r"(Tile<DH>::addr(st, r0 + g + 8, nt) + t * 4), "r"(hi));
  }
}
template <int DH>
__device__ __forceinline__ void store_tile(uint32_t st, bf16* g, long long ld, int row0, int nrows, int col0) {
#pragma unroll
  for (int i = 0; i < 64 * Tile<DH>::CH / NT; i++) {
    int idx = threadIdx.x + i * NT;
    int r = idx / Tile<DH>::CH, c = idx - r * Tile<DH>::CH;
    if (row0 + r < nrows) {
      uint4 v;
      asm volatile("ld.shared.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(Tile<DH>::addr(st, r, c)));
      *reinterpret_cast<uint4*>(g + (size_t)(row0 + r) * ld + col0 + c * 8) = v;
    }
  }
}

constexpr float LOG2E = 1.4426950408889634f;
constexpr float LN2 = 0.6931471805599453f;

// ============================== forward ==============================
template <int DH>
__global__ void __launch_bounds__(NT) attn_fwd_tc_kernel(AttnArgs a, float sl2 /* scale * log2(e) */) {
  extern __shared__ __align__(128) uint8_t smem[];
  const uint32_t sQ = s_u32(smem), sK = sQ + Tile<DH>::BYTES, sV = sK + 2 * Tile<DH>::BYTES;
  const int bh = blockIdx.y, b = bh / a.heads, h = bh - b * a.heads, N = a.N;
  const int q0 = blockIdx.x * BR;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const bf16* base = (const bf16*)a.qkv + (size_t)b * N * a.ld;
  const int qc = a.q_off + h * DH, kc = a.k_off + h * DH, vc = a.v_off + h * DH;
  const int ntiles = (N + BC - 1) / BC;

  Tile<DH>::load_async(sQ, base, a.ld, q0, N, qc);
  Tile<DH>::load_async(sK, base, a.ld, 0, N, kc);
  Tile<DH>::load_async(sV, base, a.ld, 0, N, vc);
  cp_commit();

  float o[DH / 8][4];
#pragma unroll
  for (int i = 0; i < DH / 8; i++) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f;
  float m_lo = -INFINITY, m_hi = -INFINITY, l_lo = 0.f, l_hi = 0.f;

  for (int j = 0; j < ntiles; j++) {
    cp_wait<0>();
    __syncthreads();
    if (j + 1 < ntiles) {
      Tile<DH>::load_async(sK + ((j + 1) & 1) * Tile<DH>::BYTES, base, a.ld, (j + 1) * BC, N, kc);
      Tile<DH>::load_async(sV + ((j + 1) & 1) * Tile<DH>::BYTES, base, a.ld, (j + 1) * BC, N, vc);
      cp_commit();
    }
    const uint32_t k_t = sK + (j & 1) * Tile<DH>::BYTES, v_t = sV + (j & 1) * Tile<DH>::BYTES;
    float s[8][4];
#pragma unroll
    for (int i = 0; i < 8; i++) s[i][0] = s[i][1] = s[i][2] = s[i][3] = 0.f;
    mma_abt<DH>(s, sQ, warp * 16, k_t);
    // scale to the base-2 domain, mask keys >= N
    float mx_lo = -INFINITY, mx_hi = -INFINITY;
#pragma unroll
    for (int nt = 0; nt < 8; nt++) {
      int col = j * BC + nt * 8 + 2 * t;
#pragma unroll
      for (int e = 0; e < 4; e++) {
        float v = s[nt][e] * sl2;
        if (col + (e & 1) >= N) v = -INFINITY;
        s[nt][e] = v;
      }
      mx_lo = fmaxf(mx_lo, fmaxf(s[nt][0], s[nt][1]));
      mx_hi = fmaxf(mx_hi, fmaxf(s[nt][2], s[nt][3]));
    }
    mx_lo = fmaxf(mx_lo, __shfl_xor_sync(0xffffffffu, mx_lo, 1));
    mx_lo = fmaxf(mx_lo, __shfl_xor_sync(0xffffffffu, mx_lo, 2));
    mx_hi = fmaxf(mx_hi, __shfl_xor_sync(0xffffffffu, mx_hi, 1));
    mx_hi = fmaxf(mx_hi, __shfl_xor_sync(0xffffffffu, mx_hi, 2));
    const float mn_lo = fmaxf(m_lo, mx_lo), mn_hi = fmaxf(m_hi, mx_hi);
    const float c_lo = exp2f(m_lo - mn_lo), c_hi = exp2f(m_hi - mn_hi);
    m_lo = mn_lo; m_hi = mn_hi;
    float sum_lo = 0.f, sum_hi = 0.f;
#pragma unroll
    for (int nt = 0; nt < 8; nt++) {
      s[nt][0] = exp2f(s[nt][0] - mn_lo); s[nt][1] = exp2f(s[nt][1] - mn_lo);
      s[nt][2] = exp2f(s[nt][2] - mn_hi); s[nt][3] = exp2f(s[nt][3] - mn_hi);
      sum_lo += s[nt][0] + s[nt][1];
      sum_hi += s[nt][2] + s[nt][3];
    }
    l_lo = l_lo * c_lo + sum_lo;
    l_hi = l_hi * c_hi + sum_hi;
#pragma unroll
    for (int i = 0; i < DH / 8; i++) { o[i][0] *= c_lo; o[i][1] *= c_lo; o[i][2] *= c_hi; o[i][3] *= c_hi; }
    uint32_t pf[4][4];
    c_to_a(s, pf);
    mma_pb<DH>(o, pf, v_t);
  }
  l_lo += __shfl_xor_sync(0xffffffffu, l_lo, 1); l_lo += __shfl_xor_sync(0xffffffffu, l_lo, 2);
  l_hi += __shfl_xor_sync(0xffffffffu, l_hi, 1); l_hi += __shfl_xor_sync(0xffffffffu, l_hi, 2);
  __syncthreads();                                   // everyone is done reading sQ
  stage_rows<DH>(sQ, warp * 16, o, 1.f / l_lo, 1.f / l_hi);
  if (t == 0) {
    int r = q0 + warp * 16 + g;
    if (r < N) a.lse[(size_t)bh * N + r] = (m_lo + log2f(l_lo)) * LN2;
    if (r + 8 < N) a.lse[(size_t)bh * N + r + 8] = (m_hi + log2f(l_hi)) * LN2;
  }
  __syncthreads();
  store_tile<DH>(sQ, (bf16*)a.O + (size_t)b * N * a.ldo, a.ldo, q0, N, h * DH);
}

// delta[b,h,i] = sum_d dO[i, h*dh+d] * O[i, h*dh+d]
__global__ void attn_delta_tc_kernel(AttnArgs a) {
  const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  const int total = a.B * a.heads * a.N;
  if (w >= total) return;
  const int bh = w / a.N, i = w - bh * a.N, b = bh / a.heads, h = bh - b * a.heads;
  const size_t row = (size_t)b * a.N + i;
  const bf16* po = (const bf16*)a.O + row * a.ldo + h * a.dh;
  const bf16* pd = (const bf16*)a.dO + row * a.lddo + h * a.dh;
  float s = 0.f;
  for (int d = lane * 2; d < a.dh; d += 64) {
    float2 x = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(po + d));
    float2 y = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(pd + d));
    s += x.x * y.x + x.y * y.y;
  }
  s = warp_sum(s);
  if (lane == 0) a.delta[w] = s;
}

// ============================== backward: dQ ==============================
template <int DH>
__global__ void __launch_bounds__(NT) attn_bwd_dq_tc_kernel(AttnArgs a, float scale, float sl2) {
  extern __shared__ __align__(128) uint8_t smem[];
  const uint32_t sQ = s_u32(smem), sdO = sQ + Tile<DH>::BYTES, sK = sdO + Tile<DH>::BYTES, sV = sK + 2 * Tile<DH>::BYTES;
  const int bh = blockIdx.y, b = bh / a.heads, h = bh - b * a.heads, N = a.N;
  const int q0 = blockIdx.x * BR;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const bf16* base = (const bf16*)a.qkv + (size_t)b * N * a.ld;
  const bf16* dObase = (const bf16*)a.dO + (size_t)b * N * a.lddo;
  const int qc = a.q_off + h * DH, kc = a.k_off + h * DH, vc = a.v_off + h * DH;
  const int ntiles = (N + BC - 1) / BC;

  Tile<DH>::load_async(sQ, base, a.ld, q0, N, qc);
  Tile<DH>::load_async(sdO, dObase, a.lddo, q0, N, h * DH);
  Tile<DH>::load_async(sK, base, a.ld, 0, N, kc);
  Tile<DH>::load_async(sV, base, a.ld, 0, N, vc);
  cp_commit();
  const int r_lo = q0 + warp * 16 + g, r_hi = r_lo + 8;
  const float lse_lo = r_lo < N ? a.lse[(size_t)bh * N + r_lo] * LOG2E : 0.f;
  const float lse_hi = r_hi < N ? a.lse[(size_t)bh * N + r_hi] * LOG2E : 0.f;
  const float dl_lo = r_lo < N ? a.delta[(size_t)bh * N + r_lo] : 0.f;
  const float dl_hi = r_hi < N ? a.delta[(size_t)bh * N + r_hi] : 0.f;

  float dq[DH / 8][4];
#pragma unroll
  for (int i = 0; i < DH / 8; i++) dq[i][0] = dq[i][1] = dq[i][2] = dq[i][3] = 0.f;

  for (int j = 0; j < ntiles; j++) {
    cp_wait<0>();
    __syncthreads();
    if (j + 1 < ntiles) {
      Tile<DH>::load_async(sK + ((j + 1) & 1) * Tile<DH>::BYTES, base, a.ld, (j + 1) * BC, N, kc);
      Tile<DH>::load_async(sV + ((j + 1) & 1) * Tile<DH>::BYTES, base, a.ld, (j + 1) * BC, N, vc);
      cp_commit();
    }
    const uint32_t k_t = sK + (j & 1) * Tile<DH>::BYTES, v_t = sV + (j & 1) * Tile<DH>::BYTES;
    float s[8][4], dp[8][4];
#pragma unroll
    for (int i = 0; i < 8; i++) { s[i][0] = s[i][1] = s[i][2] = s[i][3] = 0.f; dp[i][0] = dp[i][1] = dp[i][2] = dp[i][3] = 0.f; }
    mma_abt<DH>(s, sQ, warp * 16, k_t);
    mma_abt<DH>(dp, sdO, warp * 16, v_t);
#pragma unroll
    for (int nt = 0; nt < 8; nt++) {
      int col = j * BC + nt * 8 + 2 * t;
#pragma unroll
      for (int e = 0; e < 4; e++) {
        float lse = (e < 2) ? lse_lo : lse_hi, dl = (e < 2) ? dl_lo : dl_hi;
        float p = (col + (e & 1) < N) ? exp2f(s[nt][e] * sl2 - lse) : 0.f;
        s[nt][e] = p * (dp[nt][e] - dl);
      }
    }
    uint32_t pf[4][4];
    c_to_a(s, pf);
    mma_pb<DH>(dq, pf, k_t);
  }
  __syncthreads();
  stage_rows<DH>(sQ, warp * 16, dq, scale, scale);
  __syncthreads();
  store_tile<DH>(sQ, (bf16*)a.dqkv + (size_t)b * N * a.ld, a.ld, q0, N, qc);
}

// ============================== backward: dK, dV ==============================
template <int DH>
__global__ void __launch_bounds__(NT) attn_bwd_dkv_tc_kernel(AttnArgs a, float scale, float sl2) {
  extern __shared__ __align__(128) uint8_t smem[];
  const uint32_t sK = s_u32(smem), sV = sK + Tile<DH>::BYTES, sQ = sV + Tile<DH>::BYTES, sdO = sQ + 2 * Tile<DH>::BYTES;
  float* s_lse = reinterpret_cast<float*>(smem + 6 * Tile<DH>::BYTES);   // [2][64]
  float* s_dl = s_lse + 2 * BC;                                          // [2][64]
  const int bh = blockIdx.y, b = bh / a.heads, h = bh - b * a.heads, N = a.N;
  const int k0 = blockIdx.x * BR;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, t = lane & 3;
  const bf16* base = (const bf16*)a.qkv + (size_t)b * N * a.ld;
  const bf16* dObase = (const bf16*)a.dO + (size_t)b * N * a.lddo;
  const int qc = a.q_off + h * DH, kc = a.k_off + h * DH, vc = a.v_off + h * DH;
  const int ntiles = (N + BC - 1) / BC;

  auto load_q_tile = [&](int j) {
    const int buf = j & 1;
    Tile<DH>::load_async(sQ + buf * Tile<DH>::BYTES, base, a.ld, j * BC, N, qc);
    Tile<DH>::load_async(sdO + buf * Tile<DH>::BYTES, dObase, a.lddo, j * BC, N, h * DH);
    if (threadIdx.x < BC) {
      int r = j * BC + threadIdx.x;
      s_lse[buf * BC + threadIdx.x] = r < N ? a.lse[(size_t)bh * N + r] * LOG2E : 0.f;
      s_dl[buf * BC + threadIdx.x] = r < N ? a.delta[(size_t)bh * N + r] : 0.f;
    }
  };
  Tile<DH>::load_async(sK, base, a.ld, k0, N, kc);
  Tile<DH>::load_async(sV, base, a.ld, k0, N, vc);
  load_q_tile(0);
  cp_commit();

  float dk[DH / 8][4], dv[DH / 8][4];
#pragma unroll
  for (int i = 0; i < DH / 8; i++) { dk[i][0] = dk[i][1] = dk[i][2] = dk[i][3] = 0.f; dv[i][0] = dv[i][1] = dv[i][2] = dv[i][3] = 0.f; }

  for (int j = 0; j < ntiles; j++) {
    cp_wait<0>();
    __syncthreads();
    if (j + 1 < ntiles) { load_q_tile(j + 1); cp_commit(); }
    const int buf = j & 1;
    const uint32_t q_t = sQ + buf * Tile<DH>::BYTES, do_t = sdO + buf * Tile<DH>::BYTES;
    float s[8][4], dp[8][4];
#pragma unroll
    for (int i = 0; i < 8; i++) { s[i][0] = s[i][1] = s[i][2] = s[i][3] = 0.f; dp[i][0] = dp[i][1] = dp[i][2] = dp[i][3] = 0.f; }
    mma_abt<DH>(s, sK, warp * 16, q_t);       // S^T[key, query]
    mma_abt<DH>(dp, sV, warp * 16, do_t);     // dP^T[key, query]
#pragma unroll
    for (int nt = 0; nt < 8; nt++) {
#pragma unroll
      for (int e = 0; e < 4; e++) {
        int c = nt * 8 + 2 * t + (e & 1);
        s[nt][e] = (j * BC + c < N) ? exp2f(s[nt][e] * sl2 - s_lse[buf * BC + c]) : 0.f;   // P^T
      }
    }
    uint32_t pf[4][4];
    c_to_a(s, pf);
    mma_pb<DH>(dv, pf, do_t);                 // dV += P^T dO
#pragma unroll
    for (int nt = 0; nt < 8; nt++) {
#pragma unroll
      for (int e = 0; e < 4; e++) {
        int c = nt * 8 + 2 * t + (e & 1);
        s[nt][e] *= dp[nt][e] - s_dl[buf * BC + c];                                         // dS^T
      }
    }
    c_to_a(s, pf);
    mma_pb<DH>(dk, pf, q_t);                  // dK += dS^T Q
  }
  __syncthreads();
  bf16* out = (bf16*)a.dqkv + (size_t)b * N * a.ld;
  stage_rows<DH>(sQ, warp * 16, dk, scale, scale);
  stage_rows<DH>(sdO, warp * 16, dv, 1.f, 1.f);
  __syncthreads();
  store_tile<DH>(sQ, out, a.ld, k0, N, kc);
  store_tile<DH>(sdO, out, a.ld, k0, N, vc);
}

template <int DH> size_t fwd_smem() { return 5 * Tile<DH>::BYTES; }
template <int DH> size_t dq_smem() { return 6 * Tile<DH>::BYTES; }
template <int DH> size_t dkv_smem() { return 6 * Tile<DH>::BYTES + 4 * BC * sizeof(float); }

template <int DH>
int launch_fwd(const AttnArgs& a, cudaStream_t s) {
  ORBIT_SMEM_ATTR(attn_fwd_tc_kernel<DH>, fwd_smem<DH>());
  dim3 grid(cdiv(a.N, BR), a.B * a.heads);
  attn_fwd_tc_kernel<DH><<<grid, NT, fwd_smem<DH>(), s>>>(a, LOG2E / sqrtf((float)DH));
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}
template <int DH>
int launch_bwd(const AttnArgs& a, cudaStream_t s) {
  ORBIT_SMEM_ATTR(attn_bwd_dq_tc_kernel<DH>, dq_smem<DH>());
  ORBIT_SMEM_ATTR(attn_bwd_dkv_tc_kernel<DH>, dkv_smem<DH>());
  const int total_w = a.B * a.heads * a.N;
  attn_delta_tc_kernel<<<cdiv((long long)total_w * 32, 256), 256, 0, s>>>(a);
  ORBIT_LAUNCH_CHECK();
  dim3 grid(cdiv(a.N, BR), a.B * a.heads);
  const float scale = 1.0f / sqrtf((float)DH);
  attn_bwd_dq_tc_kernel<DH><<<grid, NT, dq_smem<DH>(), s>>>(a, scale, scale * LOG2E);
  ORBIT_LAUNCH_CHECK();
  attn_bwd_dkv_tc_kernel<DH><<<grid, NT, dkv_smem<DH>(), s>>>(a, scale, scale * LOG2E);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}
}  // namespace

bool attention_tc_supported(const AttnArgs& a) {
  if (a.dtype != ORBIT_BF16) return false;
  if (a.dh != 64 && a.dh != 128) return false;
  auto al16 = [](const void* p) { return (((uintptr_t)p) & 15) == 0; };
  if (a.ld % 8 || a.ldo % 8 || a.q_off % 8 || a.k_off % 8 || a.v_off % 8) return false;
  if (!al16(a.qkv) || !al16(a.O)) return false;
  if (a.dO && (!al16(a.dO) || a.lddo % 8 || !al16(a.dqkv))) return false;
  return true;
}
int attention_fwd_tc(const AttnArgs& a, cudaStream_t s) {
  return a.dh == 64 ? launch_fwd<64>(a, s) : launch_fwd<128>(a, s);
}
int attention_bwd_tc(const AttnArgs& a, cudaStream_t s) {
  return a.dh == 64 ? launch_bwd<64>(a, s) : launch_bwd<128>(a, s);
}

}  // namespace orbit
