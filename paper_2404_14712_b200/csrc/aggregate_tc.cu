// aggregate_tc.cu -- tensor-core versions of the per-patch aggregation kernels (a2 / a2'; collapsed
// form of DESIGN.md §4).  bf16 storage, heads <= 16, V <= 128, D % 64 == 0.
//
// A CTA streams one patch's token tile X [V x D] through shared memory in D-chunks (cp.async double buffer,
// XOR-swizzled 16-byte chunks) and runs the small products on mma.sync.m16n8k16 (bf16 in, fp32 accumulate):
//   forward : S = X Ut^T  (scores, [V x h])  -> warp softmax over V -> Xbar = alpha^T X  ([h x D])
//   backward: dA = X dXbar^T ([V x h]) -> ds -> dX = [alpha | ds] [dXbar ; Ut]  ([V x D]),  dUt^T += ds^T X
// X is read twice per direction (second pass mostly from L2); everything else is tiny.  This makes the kernels
// HBM/L2-bound instead of fp32-ALU-bound (2*heads .. 4*heads FMA per token element on CUDA cores).
#include "frontend.cuh"

namespace orbit {
namespace {

constexpr int NT = 256;            // 8 warps
constexpr int VP_MAX = 128;
constexpr int HP = 16;             // heads padded to 16

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

// bf16 tile with rows of DC elements (DC*2 bytes, a multiple of 128), 16-byte chunks XOR-swizzled with (row & 7)
template <int DC>
struct Tl {
  static constexpr int CH = DC / 8;
  static constexpr int ROWB = DC * 2;
  __device__ static __forceinline__ uint32_t addr(uint32_t base, int row, int chunk) {
    return base + row * ROWB + ((chunk ^ (row & 7)) << 4);
  }
  // rows [0, nrows_tile) <- g[(row) * ld + col0 ...]; rows >= nvalid zero-filled
  __device__ static __forceinline__ void load_async(uint32_t base, const bf16* g, long long ld, int nrows_tile, int nvalid,
                                                     int col0) {
    for (int idx = threadIdx.x; idx < nrows_tile * CH; idx += NT) {
      int r = idx / CH, c = idx - r * CH;
      bool ok = r < nvalid;
      cp_async16(addr(base, r, c), g + (size_t)(ok ? r : 0) * ld + col0 + c * 8, ok ? 16 : 0);
    }
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

// ============================================ forward ============================================
template <int DC>
__global__ void __launch_bounds__(NT) agg_fwd_tc_kernel(const bf16* __restrict__ tok, const bf16* __restrict__ Utb /* [HP, D] */,
    float* __restrict__ alpha, bf16* __restrict__ Xbar, int BL, int V, int D, int h) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const int Vp = (V + 15) & ~15;
  const int XB = VP_MAX * Tl<DC>::ROWB, UB = HP * Tl<DC>::ROWB;
  const uint32_t sX = s_u32(smem), sU = sX + 2 * XB;
  float* sS = reinterpret_cast<float*>(smem + 2 * XB + 2 * UB);            // [VP_MAX][SROW]
  bf16* sAT = reinterpret_cast<bf16*>(sS + VP_MAX * SROW);                  // alpha^T [HP][ATROW]
  constexpr int ATROW = VP_MAX + 8;
  const uint32_t sATu = s_u32(sAT);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int nch = D / DC, mtiles = Vp / 16;

  for (int bl = blockIdx.x; bl < BL; bl += gridDim.x) {
    const bf16* X = tok + (size_t)bl * V * D;
    auto load = [&](int i) {            // i in [0, 2*nch): pass 1 (scores) then pass 2 (Xbar)
      const int c = i % nch, buf = i & 1;
      Tl<DC>::load_async(sX + buf * XB, X, D, Vp, V, c * DC);
      if (i < nch) Tl<DC>::load_async(sU + buf * UB, Utb, D, HP, HP, c * DC);
      cp_commit();
    };
    float acc[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
    __syncthreads();                    // previous patch finished with every buffer
    load(0);
    // ---- pass 1: S[v, a] = X_v . Ut[a, :]
    for (int i = 0; i < nch; i++) {
      cp_wait<0>();
      __syncthreads();
      load(i + 1);                      // i + 1 == nch starts pass 2's first chunk
      if (warp < mtiles) chunk_scores<DC>(acc, sX + (i & 1) * XB, warp * 16, sU + (i & 1) * UB);
    }
    if (warp < mtiles) {
#pragma unroll
      for (int nt = 0; nt < 2; nt++) {
        int r = warp * 16 + g, c = nt * 8 + 2 * t;
        sS[r * SROW + c] = acc[nt][0]; sS[r * SROW + c + 1] = acc[nt][1];
        sS[(r + 8) * SROW + c] = acc[nt][2]; sS[(r + 8) * SROW + c + 1] = acc[nt][3];
      }
    }
    __syncthreads();
    // ---- softmax over v per head; alpha -> global (fp32) and alpha^T (bf16) -> smem
    for (int a = warp; a < HP; a += NT / 32) {
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
    __syncthreads();
    // ---- pass 2: Xbar[a, d] = sum_v alpha[v, a] X[v, d]; warp w owns DC/8 columns of the chunk
    uint32_t af[VP_MAX / 16][4];
#pragma unroll
    for (int ks = 0; ks < VP_MAX / 16; ks++)
      if (ks < mtiles) ldA_plain(sATu, ATROW * 2, 0, ks * 16, af[ks]);
    constexpr int WN = DC / 8;          // columns per warp per chunk (16 for DC = 128, 8 for DC = 64)
    for (int i = nch; i < 2 * nch; i++) {
      cp_wait<0>();
      __syncthreads();
      if (i + 1 < 2 * nch) load(i + 1);
      const uint32_t xc = sX + (i & 1) * XB;
      float o[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
      const int n0 = (warp * WN) & ~15;  // 16-column group holding this warp's columns
#pragma unroll
      for (int ks = 0; ks < VP_MAX / 16; ks++) {
        if (ks < mtiles) {
          uint32_t b[4];
          Tl<DC>::ldB_nmajor(xc, ks * 16, n0, b);
          if (WN == 16) { mma16816(o[0], af[ks], b[0], b[1]); mma16816(o[1], af[ks], b[2], b[3]); }
          else { if (warp & 1) mma16816(o[0], af[ks], b[2], b[3]); else mma16816(o[0], af[ks], b[0], b[1]); }
        }
      }
      const int c = (i - nch) * DC + warp * WN;
#pragma unroll
      for (int nt = 0; nt < WN / 8; nt++) {
        const int d = c + nt * 8 + 2 * t;
        if (g < h) *reinterpret_cast<uint32_t*>(Xbar + ((size_t)bl * h + g) * D + d) = pack_bf16(o[nt][0], o[nt][1]);
        if (g + 8 < h) *reinterpret_cast<uint32_t*>(Xbar + ((size_t)bl * h + g + 8) * D + d) = pack_bf16(o[nt][2], o[nt][3]);
      }
    }
  }
}

// ============================================ backward ============================================
template <int DC>
__global__ void __launch_bounds__(NT) agg_bwd_tc_kernel(const bf16* __restrict__ tok, const bf16* __restrict__ Utb,
    const float* __restrict__ alpha, const bf16* __restrict__ dXbar, bf16* __restrict__ dtok, float* __restrict__ dUt_acc,
    int BL, int V, int D, int h) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const int Vp = (V + 15) & ~15;
  const int XB = VP_MAX * Tl<DC>::ROWB, BB = 2 * HP * Tl<DC>::ROWB;          // B tile: rows 0-15 dXbar chunk, 16-31 Ut chunk
  const uint32_t sX = s_u32(smem), sB = sX + 2 * XB;
  float* sS = reinterpret_cast<float*>(smem + 2 * XB + 2 * BB);              // [VP_MAX][SROW] dalpha
  float* sAl = sS + VP_MAX * SROW;                                            // [VP_MAX][SROW] alpha
  bf16* sAD = reinterpret_cast<bf16*>(sAl + VP_MAX * SROW);                  // [VP_MAX][ADROW]  (alpha | ds)
  constexpr int ADROW = 2 * HP + 8;
  bf16* sDT = sAD + VP_MAX * ADROW;                                          // ds^T [HP][DTROW]
  constexpr int DTROW = VP_MAX + 8;
  float* sAcc = reinterpret_cast<float*>(sDT + HP * DTROW);                  // [HP][D] block-private dUt^T accumulator
  const uint32_t sADu = s_u32(sAD), sDTu = s_u32(sDT);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int nch = D / DC, mtiles = Vp / 16;

  for (int i = threadIdx.x; i < HP * D; i += NT) sAcc[i] = 0.f;

  for (int bl = blockIdx.x; bl < BL; bl += gridDim.x) {
    const bf16* X = tok + (size_t)bl * V * D;
    const bf16* dXb = dXbar + (size_t)bl * h * D;
    auto load = [&](int i) {
      const int c = i % nch, buf = i & 1;
      Tl<DC>::load_async(sX + buf * XB, X, D, Vp, V, c * DC);
      Tl<DC>::load_async(sB + buf * BB, dXb, D, HP, h, c * DC);
      if (i >= nch) Tl<DC>::load_async(sB + buf * BB + HP * Tl<DC>::ROWB, Utb, D, HP, HP, c * DC);
      cp_commit();
    };
    float acc[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
    __syncthreads();
    load(0);
    for (int i = threadIdx.x; i < Vp * HP; i += NT) {
      int v = i / HP, a = i - v * HP;
      sAl[v * SROW + a] = (v < V && a < h) ? alpha[((size_t)bl * h + a) * V + v] : 0.f;
    }
    // ---- pass 1: dalpha[v, a] = X_v . dXbar[a, :]
    for (int i = 0; i < nch; i++) {
      cp_wait<0>();
      __syncthreads();
      load(i + 1);
      if (warp < mtiles) chunk_scores<DC>(acc, sX + (i & 1) * XB, warp * 16, sB + (i & 1) * BB);
    }
    if (warp < mtiles) {
#pragma unroll
      for (int nt = 0; nt < 2; nt++) {
        int r = warp * 16 + g, c = nt * 8 + 2 * t;
        sS[r * SROW + c] = acc[nt][0]; sS[r * SROW + c + 1] = acc[nt][1];
        sS[(r + 8) * SROW + c] = acc[nt][2]; sS[(r + 8) * SROW + c + 1] = acc[nt][3];
      }
    }
    __syncthreads();
    // ---- ds[v, a] = alpha (dalpha - sum_w alpha_w dalpha_w); A operands (alpha | ds) and ds^T in bf16
    for (int a = warp; a < HP; a += NT / 32) {
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
    __syncthreads();
    uint32_t adf[2][4];                 // this warp's 16 rows of (alpha | ds): K = 32 -> 2 k-steps
    if (warp < mtiles) {
      ldA_plain(sADu, ADROW * 2, warp * 16, 0, adf[0]);
      ldA_plain(sADu, ADROW * 2, warp * 16, 16, adf[1]);
    }
    // ---- pass 2: dX chunk = (alpha | ds) [dXbar ; Ut] chunk;  dUt^T chunk += ds^T X chunk
    for (int i = nch; i < 2 * nch; i++) {
      cp_wait<0>();
      __syncthreads();
      if (i + 1 < 2 * nch) load(i + 1);
      const uint32_t xc = sX + (i & 1) * XB, bc = sB + (i & 1) * BB;
      const int c0 = (i - nch) * DC;
      if (warp < mtiles) {
#pragma unroll
        for (int np = 0; np < DC / 16; np++) {
          float o[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
#pragma unroll
          for (int ks = 0; ks < 2; ks++) {
            uint32_t b[4];
            Tl<DC>::ldB_nmajor(bc, ks * 16, np * 16, b);
            mma16816(o[0], adf[ks], b[0], b[1]);
            mma16816(o[1], adf[ks], b[2], b[3]);
          }
          const int r = warp * 16 + g;
#pragma unroll
          for (int nt = 0; nt < 2; nt++) {
            const int d = c0 + np * 16 + nt * 8 + 2 * t;
            if (r < V) *reinterpret_cast<uint32_t*>(dtok + ((size_t)bl * V + r) * D + d) = pack_bf16(o[nt][0], o[nt][1]);
            if (r + 8 < V) *reinterpret_cast<uint32_t*>(dtok + ((size_t)bl * V + r + 8) * D + d) = pack_bf16(o[nt][2], o[nt][3]);
          }
        }
      }
      // dUt^T[a, c0 + ...] += sum_v ds[v, a] X[v, ...]: 16-column groups over the warps
      for (int np = (warp + 4) & 7; np < DC / 16; np += NT / 32) {   // warps 4..7 (the dX warps are 0..mtiles-1)
        float o[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
#pragma unroll
        for (int ks = 0; ks < VP_MAX / 16; ks++) {
          if (ks < mtiles) {
            uint32_t a[4], b[4];
            ldA_plain(sDTu, DTROW * 2, 0, ks * 16, a);
            Tl<DC>::ldB_nmajor(xc, ks * 16, np * 16, b);
            mma16816(o[0], a, b[0], b[1]);
            mma16816(o[1], a, b[2], b[3]);
          }
        }
#pragma unroll
        for (int nt = 0; nt < 2; nt++) {
          const int d = c0 + np * 16 + nt * 8 + 2 * t;
          sAcc[g * D + d] += o[nt][0]; sAcc[g * D + d + 1] += o[nt][1];
          sAcc[(g + 8) * D + d] += o[nt][2]; sAcc[(g + 8) * D + d + 1] += o[nt][3];
        }
      }
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < h * D; i += NT) {
    int a = i / D, d = i - a * D;
    atomicAdd(dUt_acc + (size_t)d * h + a, sAcc[i]);
  }
}

// Ut [D, h] fp32 -> Utb [HP, D] bf16 (rows >= h zero)
__global__ void agg_ut_to_bf16_kernel(const float* __restrict__ Ut, bf16* __restrict__ Utb, int D, int h) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= HP * D) return;
  int a = i / D, d = i - a * D;
  Utb[i] = __float2bfloat16_rn(a < h ? Ut[(size_t)d * h + a] : 0.f);
}

template <int DC> size_t fwd_smem() {
  return 2 * (size_t)VP_MAX * Tl<DC>::ROWB + 2 * (size_t)HP * Tl<DC>::ROWB + (size_t)VP_MAX * SROW * 4 + (size_t)HP * (VP_MAX + 8) * 2;
}
template <int DC> size_t bwd_smem(int D) {
  return 2 * (size_t)VP_MAX * Tl<DC>::ROWB + 2 * (size_t)2 * HP * Tl<DC>::ROWB + 2 * (size_t)VP_MAX * SROW * 4 +
         (size_t)VP_MAX * (2 * HP + 8) * 2 + (size_t)HP * (VP_MAX + 8) * 2 + (size_t)HP * D * 4;
}
}  // namespace

bool agg_tc_supported(int dt, int V, int D, int heads) {
  return dt == ORBIT_BF16 && heads <= HP && V <= VP_MAX && D % 128 == 0 && bwd_smem<64>(D) <= 225 * 1024;
}
size_t agg_tc_utb_bytes(int D) { return (size_t)HP * D * sizeof(bf16); }

int agg_patch_fwd_tc(const void* tok, const float* Ut, void* Utb, float* alpha, void* Xbar, int BL, int V, int D, int heads,
                     cudaStream_t s) {
  agg_ut_to_bf16_kernel<<<cdiv((long long)HP * D, 256), 256, 0, s>>>(Ut, (bf16*)Utb, D, heads);
  ORBIT_LAUNCH_CHECK();
  constexpr int DC = 128;
  static bool set = false;
  if (!set) { ORBIT_CUDA_CHECK(cudaFuncSetAttribute((const void*)agg_fwd_tc_kernel<DC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fwd_smem<DC>())); set = true; }
  int grid = BL < 148 * 2 ? BL : 148 * 2;
  agg_fwd_tc_kernel<DC><<<grid, NT, fwd_smem<DC>(), s>>>((const bf16*)tok, (const bf16*)Utb, alpha, (bf16*)Xbar, BL, V, D, heads);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int agg_patch_bwd_tc(const void* tok, const void* Utb, const float* alpha, const void* dXbar, void* dtok, float* dUt_acc,
                     int BL, int V, int D, int heads, cudaStream_t s) {
  constexpr int DC = 64;
  const size_t smb = bwd_smem<DC>(D);
  ORBIT_CUDA_CHECK(cudaFuncSetAttribute((const void*)agg_bwd_tc_kernel<DC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smb));
  int grid = BL < 148 ? BL : 148;
  agg_bwd_tc_kernel<DC><<<grid, NT, smb, s>>>((const bf16*)tok, (const bf16*)Utb, alpha, (const bf16*)dXbar, (bf16*)dtok, dUt_acc,
                                              BL, V, D, heads);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

}  // namespace orbit
