// front_fused.cu -- kernels of the fused pixel-space front end (a1 + a2 and a2' + a1' with
// the [B, L, V, D] token tensor never materialised).
//
// Tokenisation is affine in the pixels ("independent patch tokenization for each channel input") and
// nothing non-linear sits between it and the K/V projections of the aggregation cross-attention (PAPER.md:46
// "aggregated together across different channels using cross-attention"), so with
//     pixext[v, r] = pix(b, v, l, r) for r < p^2,  1 for r = p^2            (R = p^2 + 1 entries per variable)
//     Wpb[(r, v), :] = Wp[v, r, :] for r < p^2,    bp[v, :] for r = p^2     (the tokeniser as one [R*V, D] matrix)
// the collapsed aggregation of DESIGN.md §4 becomes, exactly (real arithmetic):
//     s[v, a]  = X_v . Ut[:, a]              = sum_r pixext[v, r] G[(r, v), a],        G = Wpb Ut        [R*V, heads]
//     o[:, a]  = (sum_v alpha[v, a] X_v) Wv[:, a] + bv[a]
//              = sum_{r, v} (alpha[v, a] pixext[v, r]) H[(r, v), a-columns] + bv[a],   H = Wpb Wv        [R*V, D]
// i.e. per head a GEMM  o_a = A_a H_a  with  A_a[bl, (r, v)] = alpha[bl, v, a] pixext[bl, v, r]  (K = R*V, 1547 at
// C3) instead of V token rows of D elements per patch.  The k index is (r, v) with v fastest and V padded to Vp
// (a multiple of 8) so that a warp's lanes (= variables) write and read A / dA contiguously.
//
// Kernels here (the GEMMs are the library's tcgen05 / SIMT GEMM, strided-batched over the heads):
//   fe_pack_wpb      Wpb  <- (Wp, bp)
//   fe_make_g        G    <- Wpb Ut                     (fp32, [R][Vp][HP])
//   fe_patch_fwd     per patch (one warp): scores, softmax over V, alpha, A
//   fe_patch_bwd     per patch (one warp): dalpha = <dA, pixext>, ds -> dsT [Vp][BL][HP]
//   fe_dg            dG[(r, v), a] = sum_bl pixext ds           (score path, reduction over patches)
//   fe_dut           dUt = Wpb^T dG                              (feeds agg_param_bwd: dWk, dbq, dWq, dq)
//   fe_finish_dwp    dWp, dbp <- dH Wv^T (fp32 from the GEMM) + dG Ut^T
#include "front_fused.cuh"

namespace orbit {
namespace {

constexpr int HP = FE_HP;
constexpr int HG = 8;     // heads per pass of fe_patch_fwd

template <typename T> struct Pair;
template <> struct Pair<float> {
  typedef float2 type;
  static __device__ __forceinline__ float2 make(float a, float b) { return make_float2(a, b); }
  static __device__ __forceinline__ float2 unpack(float2 v) { return v; }
};
template <> struct Pair<bf16> {
  typedef __nv_bfloat162 type;
  static __device__ __forceinline__ __nv_bfloat162 make(float a, float b) { return __floats2bfloat162_rn(a, b); }
  static __device__ __forceinline__ float2 unpack(__nv_bfloat162 v) { return __bfloat1622float2(v); }
};

// pixels of patch (b, i, j) of variable v: out[di*P + dj] = x[b, v, i*P + di, j*P + dj]
template <int P>
__device__ __forceinline__ void load_pix(const float* __restrict__ x, int V, int Hg, int Wg, int b, int v, int i, int j,
                                         float* out) {
  const float* base = x + (((size_t)b * V + v) * Hg + (size_t)i * P) * Wg + (size_t)j * P;
#pragma unroll
  for (int di = 0; di < P; di++) {
    if (P == 4) {
      const float4 q = *reinterpret_cast<const float4*>(base + (size_t)di * Wg);
      out[di * 4 + 0] = q.x; out[di * 4 + 1] = q.y; out[di * 4 + 2] = q.z; out[di * 4 + 3] = q.w;
    } else if (P == 2) {
      const float2 q = *reinterpret_cast<const float2*>(base + (size_t)di * Wg);
      out[di * 2 + 0] = q.x; out[di * 2 + 1] = q.y;
    } else {
#pragma unroll
      for (int dj = 0; dj < P; dj++) out[di * P + dj] = base[(size_t)di * Wg + dj];
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
template <typename T>
__global__ void fe_pack_wpb_kernel(const T* __restrict__ Wp, const T* __restrict__ bp, T* __restrict__ Wpb, int V, int Vp,
                                   int P2, int D) {
  const size_t n = (size_t)(P2 + 1) * Vp * D;
  for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += (size_t)gridDim.x * blockDim.x) {
    const int d = (int)(idx % D);
    const int k = (int)(idx / D), r = k / Vp, v = k - r * Vp;
    T val = from_f<T>(0.f);
    if (v < V) val = r < P2 ? Wp[((size_t)v * P2 + r) * D + d] : bp[(size_t)v * D + d];
    Wpb[idx] = val;
  }
}

// G[r][a][v] = sum_d Wpb[(r, v), d] Ut[d, a]  (fp32 [R][HP][Vp], v fastest); one warp per k = (r, v) row, lanes stride over d
template <typename T>
__global__ void fe_make_g_kernel(const T* __restrict__ Wpb, const float* __restrict__ Ut, float* __restrict__ G, int KVp,
                                 int Vp, int D, int h) {
  const int k = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (k >= KVp) return;
  float acc[HP];
#pragma unroll
  for (int a = 0; a < HP; a++) acc[a] = 0.f;
  if (h == HP) {                       // rows of Ut are 64 bytes: four 16-byte loads
    for (int d = lane; d < D; d += 32) {
      const float w = to_f<T>(Wpb[(size_t)k * D + d]);
      const float4* u4 = reinterpret_cast<const float4*>(Ut + (size_t)d * HP);
#pragma unroll
      for (int q = 0; q < HP / 4; q++) {
        const float4 u = __ldg(u4 + q);
        acc[4 * q] = fmaf(w, u.x, acc[4 * q]); acc[4 * q + 1] = fmaf(w, u.y, acc[4 * q + 1]);
        acc[4 * q + 2] = fmaf(w, u.z, acc[4 * q + 2]); acc[4 * q + 3] = fmaf(w, u.w, acc[4 * q + 3]);
      }
    }
  } else {
    for (int d = lane; d < D; d += 32) {
      const float w = to_f<T>(Wpb[(size_t)k * D + d]);
#pragma unroll
      for (int a = 0; a < HP; a++)
        if (a < h) acc[a] = fmaf(w, Ut[(size_t)d * h + a], acc[a]);
    }
  }
#pragma unroll
  for (int a = 0; a < HP; a++) acc[a] = warp_sum(acc[a]);
  if (lane == 0) {
    const int r = k / Vp, v = k - r * Vp;
#pragma unroll
    for (int a = 0; a < HP; a++) G[((size_t)r * HP + a) * Vp + v] = acc[a];
  }
}

// ---------------------------------------------------------------------------------------------------------
// forward, one warp per patch; lane owns the variable pairs (64 n + 2 lane, +1), n < NV
template <typename T, int P, int NV>
__global__ void __launch_bounds__(256, NV == 2 ? 1 : 2) fe_patch_fwd_kernel(const float* __restrict__ x, const float* __restrict__ G,
    float* __restrict__ alpha, T* __restrict__ A, int V, int Vp, int Hg, int Wg, int h, int BL) {
  constexpr int P2 = P * P, R = P2 + 1, E = 2 * NV;
  typedef typename Pair<T>::type pair_t;
  const int lane = threadIdx.x & 31;
  const int warp0 = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
  const int gw = Wg / P, L = (Hg / P) * gw, KVp = R * Vp;
  for (int bl = warp0; bl < BL; bl += nwarps) {
    const int b = bl / L, l = bl - b * L, i = l / gw, j = l - i * gw;
    float pix[E][P2];
#pragma unroll
    for (int e = 0; e < E; e++) {
      const int v = 64 * (e >> 1) + 2 * lane + (e & 1);
      if (v < V) load_pix<P>(x, V, Hg, Wg, b, v, i, j, pix[e]);
      else {
#pragma unroll
        for (int r = 0; r < P2; r++) pix[e][r] = 0.f;
      }
    }
    // heads in groups of HG = 8: 16 score accumulators per variable pair at a time keep the kernel at ~128 registers
    // (all 16 heads at once needed 255 registers and left 12 % occupancy on a purely HBM-bound kernel)
#pragma unroll 1
    for (int a0 = 0; a0 < h; a0 += HG) {
      float s[E][HG];
      // G is stored [r][head][v] (v fastest): the lanes of a warp (consecutive variable pairs) read 256 contiguous bytes
      // per (r, head).  With the [(r, v)][head] layout every 16-byte load of a warp touched 32 different lines.
#pragma unroll
      for (int n = 0; n < NV; n++) {
        const int v0 = 64 * n + 2 * lane;
        if (v0 < Vp) {
#pragma unroll
          for (int aa = 0; aa < HG; aa++) {
            const float2 g = __ldg(reinterpret_cast<const float2*>(G + ((size_t)P2 * HP + a0 + aa) * Vp + v0));
            s[2 * n][aa] = g.x; s[2 * n + 1][aa] = g.y;
          }
#pragma unroll
          for (int r = 0; r < P2; r++) {
            float2 g[HG];
#pragma unroll
            for (int aa = 0; aa < HG; aa++) g[aa] = __ldg(reinterpret_cast<const float2*>(G + ((size_t)r * HP + a0 + aa) * Vp + v0));
#pragma unroll
            for (int aa = 0; aa < HG; aa++) {
              s[2 * n][aa] = fmaf(pix[2 * n][r], g[aa].x, s[2 * n][aa]);
              s[2 * n + 1][aa] = fmaf(pix[2 * n + 1][r], g[aa].y, s[2 * n + 1][aa]);
            }
          }
        }
#pragma unroll
        for (int q = 0; q < 2; q++) {
          if (v0 + q >= V) {
#pragma unroll
            for (int aa = 0; aa < HG; aa++) s[2 * n + q][aa] = -INFINITY;
          }
        }
      }
      // softmax over the variables, per head (R3): alpha replaces s
#pragma unroll
      for (int aa = 0; aa < HG; aa++) {
        if (a0 + aa < h) {
          float m = s[0][aa];
#pragma unroll
          for (int e = 1; e < E; e++) m = fmaxf(m, s[e][aa]);
          m = warp_max(m);
          float sum = 0.f;
#pragma unroll
          for (int e = 0; e < E; e++) { s[e][aa] = __expf(s[e][aa] - m); sum += s[e][aa]; }
          sum = warp_sum(sum);
          const float inv = 1.f / sum;
#pragma unroll
          for (int e = 0; e < E; e++) s[e][aa] *= inv;
        }
      }
      // alpha [BL, h, Vp] fp32 and A [BL, h, R*Vp] (k = r*Vp + v); padded variables get exact zeros
#pragma unroll
      for (int aa = 0; aa < HG; aa++) {
        if (a0 + aa < h) {
          const int a = a0 + aa;
#pragma unroll
          for (int n = 0; n < NV; n++) {
            const int v0 = 64 * n + 2 * lane;
            if (v0 < Vp) {
              const float w0 = s[2 * n][aa], w1 = s[2 * n + 1][aa];
              *reinterpret_cast<float2*>(alpha + ((size_t)bl * h + a) * Vp + v0) = make_float2(w0, w1);
              T* row = A + ((size_t)bl * h + a) * KVp + v0;
#pragma unroll
              for (int r = 0; r < P2; r++)
                *reinterpret_cast<pair_t*>(row + (size_t)r * Vp) = Pair<T>::make(w0 * pix[2 * n][r], w1 * pix[2 * n + 1][r]);
              *reinterpret_cast<pair_t*>(row + (size_t)P2 * Vp) = Pair<T>::make(w0, w1);
            }
          }
        }
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// backward, one warp per patch: dalpha[v, a] = sum_r dA[bl, a, (r, v)] pixext[v, r];
// ds = alpha (dalpha - sum_w alpha_w dalpha_w) -> dsT[v][bl][a]
template <typename T, int P, int NV>
__global__ void __launch_bounds__(256, 2) fe_patch_bwd_kernel(const float* __restrict__ x, const float* __restrict__ alpha,
    const T* __restrict__ dA, float* __restrict__ dsT, int V, int Vp, int Hg, int Wg, int h, int BL) {
  constexpr int P2 = P * P, R = P2 + 1, E = 2 * NV;
  typedef typename Pair<T>::type pair_t;
  const int lane = threadIdx.x & 31;
  const int warp0 = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
  const int gw = Wg / P, L = (Hg / P) * gw, KVp = R * Vp;
  for (int bl = warp0; bl < BL; bl += nwarps) {
    const int b = bl / L, l = bl - b * L, i = l / gw, j = l - i * gw;
    float pix[E][P2], ds[E][HP];
#pragma unroll
    for (int e = 0; e < E; e++) {
      const int v = 64 * (e >> 1) + 2 * lane + (e & 1);
      if (v < V) load_pix<P>(x, V, Hg, Wg, b, v, i, j, pix[e]);
      else {
#pragma unroll
        for (int r = 0; r < P2; r++) pix[e][r] = 0.f;
      }
    }
#pragma unroll
    for (int a = 0; a < HP; a++) {
      if (a < h) {
        float al[E], da[E];
        float dot = 0.f;
#pragma unroll
        for (int n = 0; n < NV; n++) {
          const int v0 = 64 * n + 2 * lane;
          al[2 * n] = al[2 * n + 1] = 0.f; da[2 * n] = da[2 * n + 1] = 0.f;
          if (v0 < Vp) {
            const float2 aa = *reinterpret_cast<const float2*>(alpha + ((size_t)bl * h + a) * Vp + v0);
            al[2 * n] = aa.x; al[2 * n + 1] = aa.y;
            const T* row = dA + ((size_t)bl * h + a) * KVp + v0;
            float2 acc = Pair<T>::unpack(*reinterpret_cast<const pair_t*>(row + (size_t)P2 * Vp));
#pragma unroll
            for (int r = 0; r < P2; r++) {
              const float2 g = Pair<T>::unpack(*reinterpret_cast<const pair_t*>(row + (size_t)r * Vp));
              acc.x = fmaf(g.x, pix[2 * n][r], acc.x);
              acc.y = fmaf(g.y, pix[2 * n + 1][r], acc.y);
            }
            da[2 * n] = acc.x; da[2 * n + 1] = acc.y;
            dot += aa.x * acc.x + aa.y * acc.y;     // padded variables have alpha == 0
          }
        }
        dot = warp_sum(dot);
#pragma unroll
        for (int e = 0; e < E; e++) ds[e][a] = al[e] * (da[e] - dot);
      } else {
#pragma unroll
        for (int e = 0; e < E; e++) ds[e][a] = 0.f;
      }
    }
#pragma unroll
    for (int e = 0; e < E; e++) {
      const int v = 64 * (e >> 1) + 2 * lane + (e & 1);
      if (v < V) {
        float4* o = reinterpret_cast<float4*>(dsT + ((size_t)v * BL + bl) * HP);
#pragma unroll
        for (int q = 0; q < HP / 4; q++) o[q] = make_float4(ds[e][4 * q], ds[e][4 * q + 1], ds[e][4 * q + 2], ds[e][4 * q + 3]);
      }
    }
  }
}

// dG[(r, v), a] += sum_{bl in this split} pixext[bl, v, r] dsT[v][bl][a]; block = (v, a range of patch rows),
// thread = (r, a).  A patch row (b, i) is gw consecutive patches: its pixels for (v, r) are x[row + j*P] and its
// ds values dsT[v][bl0 + j][a], so the inner loop has no index arithmetic beyond two strides.
template <int P>
__global__ void fe_dg_kernel(const float* __restrict__ x, const float* __restrict__ dsT, float* __restrict__ dG, int V, int Vp,
                             int Hg, int Wg, int B, int rows_per_split) {
  constexpr int P2 = P * P, R = P2 + 1;
  const int v = blockIdx.x, t = threadIdx.x;
  if (t >= R * HP) return;
  const int r = t / HP, a = t - r * HP;
  const int gh = Hg / P, gw = Wg / P, BL = B * gh * gw;
  const int di = r / P, dj = r - di * P;
  const int pr0 = blockIdx.y * rows_per_split, pr1 = min(B * gh, pr0 + rows_per_split);
  float acc = 0.f;
  const float* dsv = dsT + (size_t)v * BL * HP + a;
  for (int pr = pr0; pr < pr1; pr++) {
    const int b = pr / gh, i = pr - b * gh;
    const float* ds = dsv + (size_t)pr * gw * HP;
    if (r < P2) {
      const float* px = x + (((size_t)b * V + v) * Hg + (size_t)i * P + di) * Wg + dj;
#pragma unroll 8
      for (int j = 0; j < gw; j++) acc = fmaf(__ldg(px + j * P), ds[(size_t)j * HP], acc);
    } else {
#pragma unroll 8
      for (int j = 0; j < gw; j++) acc += ds[(size_t)j * HP];
    }
  }
  atomicAdd(dG + ((size_t)r * Vp + v) * HP + a, acc);
}

// dUt[d, a] += sum_{k in split} Wpb[k, d] dG[k, a]; block = 32 d x 16 a (thread t <-> (d, a), a fastest: the
// atomics of a warp cover consecutive floats of dUt [D, h] when h == HP), blockIdx.y = k split
template <typename T>
__global__ void __launch_bounds__(512) fe_dut_kernel(const T* __restrict__ Wpb, const float* __restrict__ dG,
                                                     float* __restrict__ dUt, int KVp, int D, int h, int per_split) {
  const int a = threadIdx.x & (HP - 1), d = blockIdx.x * 32 + (threadIdx.x >> 4);
  if (d >= D) return;
  const int k0 = blockIdx.y * per_split, k1 = min(KVp, k0 + per_split);
  float acc = 0.f;
#pragma unroll 4
  for (int k = k0; k < k1; k++) acc = fmaf(to_f<T>(Wpb[(size_t)k * D + d]), __ldg(dG + (size_t)k * HP + a), acc);
  if (a < h) atomicAdd(dUt + (size_t)d * h + a, acc);
}

// dWp[v, r, d] / dbp[v, d] = accW[(r, v), d] + sum_a dG[(r, v), a] Ut[d, a]; blockIdx.y = (r, v), threads over d
template <typename T>
__global__ void fe_finish_dwp_kernel(const float* __restrict__ accW, const float* __restrict__ dG, const float* __restrict__ Ut,
                                     T* __restrict__ dWp, T* __restrict__ dbp, int V, int Vp, int P2, int D, int h) {
  const int rv = blockIdx.y, r = rv / V, v = rv - r * V;
  const size_t k = (size_t)r * Vp + v;
  float g[HP];
#pragma unroll
  for (int a = 0; a < HP; a++) g[a] = a < h ? dG[k * HP + a] : 0.f;
  T* out = r < P2 ? dWp + ((size_t)v * P2 + r) * D : dbp + (size_t)v * D;
  for (int d = blockIdx.x * blockDim.x + threadIdx.x; d < D; d += gridDim.x * blockDim.x) {
    float val = accW[k * D + d];
    if (h == HP) {
      const float4* u4 = reinterpret_cast<const float4*>(Ut + (size_t)d * HP);
#pragma unroll
      for (int q = 0; q < HP / 4; q++) {
        const float4 u = __ldg(u4 + q);
        val = fmaf(g[4 * q], u.x, val); val = fmaf(g[4 * q + 1], u.y, val);
        val = fmaf(g[4 * q + 2], u.z, val); val = fmaf(g[4 * q + 3], u.w, val);
      }
    } else {
#pragma unroll
      for (int a = 0; a < HP; a++)
        if (a < h) val = fmaf(g[a], Ut[(size_t)d * h + a], val);
    }
    out[d] = from_f<T>(val);
  }
}

int grid_for(size_t n, int block) {
  size_t g = (n + block - 1) / block;
  return (int)(g > 148 * 16 ? 148 * 16 : (g ? g : 1));
}
}  // namespace

bool fe_supported(int V, int p, int heads) { return V <= 64 * 2 && (p == 1 || p == 2 || p == 4) && heads <= HP; }

int fe_pack_wpb(const void* Wp, const void* bp, int dt, void* Wpb, int V, int Vp, int P2, int D, cudaStream_t s) {
  const size_t n = (size_t)(P2 + 1) * Vp * D;
  if (dt == ORBIT_BF16) fe_pack_wpb_kernel<bf16><<<grid_for(n, 256), 256, 0, s>>>((const bf16*)Wp, (const bf16*)bp, (bf16*)Wpb, V, Vp, P2, D);
  else fe_pack_wpb_kernel<float><<<grid_for(n, 256), 256, 0, s>>>((const float*)Wp, (const float*)bp, (float*)Wpb, V, Vp, P2, D);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int fe_make_g(const void* Wpb, int dt, const float* Ut, float* G, int KVp, int Vp, int D, int h, cudaStream_t s) {
  const int grid = cdiv((long long)KVp * 32, 256);
  if (dt == ORBIT_BF16) fe_make_g_kernel<bf16><<<grid, 256, 0, s>>>((const bf16*)Wpb, Ut, G, KVp, Vp, D, h);
  else fe_make_g_kernel<float><<<grid, 256, 0, s>>>((const float*)Wpb, Ut, G, KVp, Vp, D, h);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int fe_patch_fwd(const float* x, const float* G, float* alpha, void* A, int dt, int V, int Vp, int Hg, int Wg, int p, int h,
                 int BL, cudaStream_t s) {
#define ARGS_F(TT) x, G, alpha, (TT*)A, V, Vp, Hg, Wg, h, BL
  const int nv = V <= 64 ? 1 : 2;
  const int grid = cdiv(BL, 8) < 148 * 8 ? cdiv(BL, 8) : 148 * 8;
#define LF(TT, PP, NN) fe_patch_fwd_kernel<TT, PP, NN><<<grid, 256, 0, s>>>(ARGS_F(TT))
  if (dt == ORBIT_BF16) {
    if (p == 4) { if (nv == 1) LF(bf16, 4, 1); else LF(bf16, 4, 2); }
    else if (p == 2) { if (nv == 1) LF(bf16, 2, 1); else LF(bf16, 2, 2); }
    else { if (nv == 1) LF(bf16, 1, 1); else LF(bf16, 1, 2); }
  } else {
    if (p == 4) { if (nv == 1) LF(float, 4, 1); else LF(float, 4, 2); }
    else if (p == 2) { if (nv == 1) LF(float, 2, 1); else LF(float, 2, 2); }
    else { if (nv == 1) LF(float, 1, 1); else LF(float, 1, 2); }
  }
#undef LF
#undef ARGS_F
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int fe_patch_bwd(const float* x, const float* alpha, const void* dA, int dt, float* dsT, int V, int Vp, int Hg, int Wg, int p,
                 int h, int BL, cudaStream_t s) {
#define ARGS_B(TT) x, alpha, (const TT*)dA, dsT, V, Vp, Hg, Wg, h, BL
  const int nv = V <= 64 ? 1 : 2;
  const int grid = cdiv(BL, 8) < 148 * 8 ? cdiv(BL, 8) : 148 * 8;
#define LB(TT, PP, NN) fe_patch_bwd_kernel<TT, PP, NN><<<grid, 256, 0, s>>>(ARGS_B(TT))
  if (dt == ORBIT_BF16) {
    if (p == 4) { if (nv == 1) LB(bf16, 4, 1); else LB(bf16, 4, 2); }
    else if (p == 2) { if (nv == 1) LB(bf16, 2, 1); else LB(bf16, 2, 2); }
    else { if (nv == 1) LB(bf16, 1, 1); else LB(bf16, 1, 2); }
  } else {
    if (p == 4) { if (nv == 1) LB(float, 4, 1); else LB(float, 4, 2); }
    else if (p == 2) { if (nv == 1) LB(float, 2, 1); else LB(float, 2, 2); }
    else { if (nv == 1) LB(float, 1, 1); else LB(float, 1, 2); }
  }
#undef LB
#undef ARGS_B
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int fe_dg(const float* x, const float* dsT, float* dG, int B, int V, int Vp, int Hg, int Wg, int p, cudaStream_t s) {
  const int P2 = p * p, R = P2 + 1, prows = B * (Hg / p);
  int splits = cdiv(148 * 32, V);     // 4x more, shorter serial loops than one wave of CTAs: 152 -> 99 us at C3
  if (splits > prows) splits = prows;
  const int per = cdiv(prows, splits);
  dim3 grid(V, cdiv(prows, per));
  const int nt = ((R * HP + 31) / 32) * 32;
  if (p == 4) fe_dg_kernel<4><<<grid, nt, 0, s>>>(x, dsT, dG, V, Vp, Hg, Wg, B, per);
  else if (p == 2) fe_dg_kernel<2><<<grid, nt, 0, s>>>(x, dsT, dG, V, Vp, Hg, Wg, B, per);
  else fe_dg_kernel<1><<<grid, nt, 0, s>>>(x, dsT, dG, V, Vp, Hg, Wg, B, per);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int fe_dut(const void* Wpb, int dt, const float* dG, float* dUt, int KVp, int D, int h, cudaStream_t s) {
  const int gx = cdiv(D, 32);
  int splits = cdiv(148 * 4, gx);
  if (splits > cdiv(KVp, 16)) splits = cdiv(KVp, 16);
  const int per = cdiv(KVp, splits);
  dim3 grid(gx, cdiv(KVp, per));
  if (dt == ORBIT_BF16) fe_dut_kernel<bf16><<<grid, 512, 0, s>>>((const bf16*)Wpb, dG, dUt, KVp, D, h, per);
  else fe_dut_kernel<float><<<grid, 512, 0, s>>>((const float*)Wpb, dG, dUt, KVp, D, h, per);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int fe_finish_dwp(const float* accW, const float* dG, const float* Ut, void* dWp, void* dbp, int dt, int V, int Vp, int P2,
                  int D, int h, cudaStream_t s) {
  dim3 grid(cdiv(D, 256), (P2 + 1) * V);
  if (dt == ORBIT_BF16) fe_finish_dwp_kernel<bf16><<<grid, 256, 0, s>>>(accW, dG, Ut, (bf16*)dWp, (bf16*)dbp, V, Vp, P2, D, h);
  else fe_finish_dwp_kernel<float><<<grid, 256, 0, s>>>(accW, dG, Ut, (float*)dWp, (float*)dbp, V, Vp, P2, D, h);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

}  // namespace orbit
