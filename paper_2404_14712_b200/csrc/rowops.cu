// rowops.cu -- HBM-bound row-wise kernels: LayerNorm fwd/bwd, column sums (bias grads), casts, combines.
// All are one pass over their inputs with 16-byte vector accesses; statistics and sums in fp32.
#include "common.cuh"
#include "vec8.cuh"
#include <stdlib.h>

namespace orbit {

namespace {

__device__ __forceinline__ float2 block_sum2(float2 v, float2* sh) {
  int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  v.x = warp_sum(v.x); v.y = warp_sum(v.y);
  __syncthreads();
  if (lane == 0) sh[w] = v;
  __syncthreads();
  float2 r = lane < nw ? sh[lane] : make_float2(0.f, 0.f);
  r.x = warp_sum(r.x); r.y = warp_sum(r.y);
  return r;
}

// ---- LayerNorm forward: one block per row (persistent over rows), row cached in registers ------------
template <int MAXCH>
__global__ void __launch_bounds__(1024) ln_fwd_kernel(const void* __restrict__ x, int x_dt,
    const void* __restrict__ gamma, const void* __restrict__ beta, int p_dt, void* __restrict__ out, int out_dt,
    float* __restrict__ mean, float* __restrict__ rstd, int M, int D, float eps, void* __restrict__ x_copy) {
  __shared__ float2 sh[32];
  const int nch = D >> 3;
  for (int row = blockIdx.x; row < M; row += gridDim.x) {
    float v[MAXCH][8];
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < MAXCH; c++) {
      int ch = threadIdx.x + c * blockDim.x;
      if (ch < nch) {
        ld8(x, (size_t)row * D + (size_t)ch * 8, x_dt, v[c]);
        if (x_copy) st8(x_copy, (size_t)row * D + (size_t)ch * 8, x_dt, v[c]);
#pragma unroll
        for (int j = 0; j < 8; j++) s += v[c][j];
      }
    }
    float2 r = block_sum2(make_float2(s, 0.f), sh);
    const float mu = r.x / D;
    float q = 0.f;
#pragma unroll
    for (int c = 0; c < MAXCH; c++) {
      int ch = threadIdx.x + c * blockDim.x;
      if (ch < nch) {
#pragma unroll
        for (int j = 0; j < 8; j++) { float d = v[c][j] - mu; q += d * d; }
      }
    }
    r = block_sum2(make_float2(q, 0.f), sh);
    const float rs = rsqrtf(r.x / D + eps);
    if (threadIdx.x == 0) { mean[row] = mu; rstd[row] = rs; }
#pragma unroll
    for (int c = 0; c < MAXCH; c++) {
      int ch = threadIdx.x + c * blockDim.x;
      if (ch < nch) {
        float g[8], b[8], o[8];
        ld8(gamma, (size_t)ch * 8, p_dt, g);
        ld8(beta, (size_t)ch * 8, p_dt, b);
#pragma unroll
        for (int j = 0; j < 8; j++) o[j] = (v[c][j] - mu) * rs * g[j] + b[j];
        st8(out, (size_t)row * D + (size_t)ch * 8, out_dt, o);
      }
    }
  }
}

// ---- LayerNorm backward ------------------------------------------------------------------------------
// One block per row (persistent over rows); a thread owns MAXCH 8-column chunks and keeps their dgamma / dbeta
// sums in registers across rows.  With MAXCH == 1 the next row's x / dout / add chunks are requested before
// the block-wide reduction of the current row (software prefetch: the two barriers of the reduction otherwise
// expose a full HBM round trip per row).
template <int MAXCH, int TMAX>
__global__ void __launch_bounds__(TMAX) ln_bwd_kernel(const void* __restrict__ dout, int dout_dt,
    const void* __restrict__ x, int x_dt, const float* __restrict__ mean, const float* __restrict__ rstd,
    const void* __restrict__ gamma, int p_dt, const void* __restrict__ add, int add_dt,
    float* __restrict__ dx_f32, void* __restrict__ dx_out, int out_dt,
    float* __restrict__ dgamma_acc, float* __restrict__ dbeta_acc, int M, int D) {
  __shared__ float2 sh[32];
  const int nch = D >> 3;
  float dg[MAXCH][8], db[MAXCH][8], gm[MAXCH][8];
#pragma unroll
  for (int c = 0; c < MAXCH; c++) {
    int ch = threadIdx.x + c * blockDim.x;
#pragma unroll
    for (int j = 0; j < 8; j++) { dg[c][j] = 0.f; db[c][j] = 0.f; gm[c][j] = 0.f; }
    if (ch < nch) ld8(gamma, (size_t)ch * 8, p_dt, gm[c]);
  }
  if (MAXCH == 1) {
    const int ch = threadIdx.x;
    const bool act = ch < nch;
    float xn[8], dn[8], an[8];
#pragma unroll
    for (int j = 0; j < 8; j++) { xn[j] = 0.f; dn[j] = 0.f; an[j] = 0.f; }
    int row = blockIdx.x;
    if (row < M && act) {
      const size_t off = (size_t)row * D + (size_t)ch * 8;
      ld8(x, off, x_dt, xn); ld8(dout, off, dout_dt, dn);
      if (add) ld8(add, off, add_dt, an);
    }
    for (; row < M; row += gridDim.x) {
      const float mu = mean[row], rs = rstd[row];
      float zh[8], gh[8], av[8];
      float s1 = 0.f, s2 = 0.f;
#pragma unroll
      for (int j = 0; j < 8; j++) {
        const float z = (xn[j] - mu) * rs;
        zh[j] = z; av[j] = an[j];
        dg[0][j] += dn[j] * z;
        db[0][j] += dn[j];
        const float g = dn[j] * gm[0][j];
        gh[j] = g;
        s1 += g; s2 += g * z;
      }
      const int nrow = row + gridDim.x;
      if (nrow < M && act) {                       // prefetch the next row before the reduction barriers
        const size_t off = (size_t)nrow * D + (size_t)ch * 8;
        ld8(x, off, x_dt, xn); ld8(dout, off, dout_dt, dn);
        if (add) ld8(add, off, add_dt, an);
      }
      const float2 r = block_sum2(make_float2(s1, s2), sh);
      const float m1 = r.x / D, m2 = r.y / D;
      if (act) {
        float o[8];
        const size_t off = (size_t)row * D + (size_t)ch * 8;
#pragma unroll
        for (int j = 0; j < 8; j++) o[j] = av[j] + (gh[j] - m1 - zh[j] * m2) * rs;
        if (dx_f32) st8(dx_f32, off, ORBIT_F32, o);
        if (dx_out) st8(dx_out, off, out_dt, o);
      }
    }
  } else {
    for (int row = blockIdx.x; row < M; row += gridDim.x) {
      const float mu = mean[row], rs = rstd[row];
      float zh[MAXCH][8], gh[MAXCH][8];
      float s1 = 0.f, s2 = 0.f;
#pragma unroll
      for (int c = 0; c < MAXCH; c++) {
        int ch = threadIdx.x + c * blockDim.x;
        if (ch < nch) {
          float xv[8], dv[8];
          ld8(x, (size_t)row * D + (size_t)ch * 8, x_dt, xv);
          ld8(dout, (size_t)row * D + (size_t)ch * 8, dout_dt, dv);
#pragma unroll
          for (int j = 0; j < 8; j++) {
            float z = (xv[j] - mu) * rs;
            zh[c][j] = z;
            dg[c][j] += dv[j] * z;
            db[c][j] += dv[j];
            float g = dv[j] * gm[c][j];
            gh[c][j] = g;
            s1 += g; s2 += g * z;
          }
        }
      }
      float2 r = block_sum2(make_float2(s1, s2), sh);
      const float m1 = r.x / D, m2 = r.y / D;
#pragma unroll
      for (int c = 0; c < MAXCH; c++) {
        int ch = threadIdx.x + c * blockDim.x;
        if (ch < nch) {
          float o[8];
          size_t off = (size_t)row * D + (size_t)ch * 8;
          if (add) ld8(add, off, add_dt, o);
          else {
#pragma unroll
            for (int j = 0; j < 8; j++) o[j] = 0.f;
          }
#pragma unroll
          for (int j = 0; j < 8; j++) o[j] += (gh[c][j] - m1 - zh[c][j] * m2) * rs;
          if (dx_f32) st8(dx_f32, off, ORBIT_F32, o);
          if (dx_out) st8(dx_out, off, out_dt, o);
        }
      }
    }
  }
  // dgamma / dbeta: a thread's 8 consecutive columns are transposed through a per-warp shared-memory strip so that
  // every atomic instruction of a warp covers 32 consecutive floats (one 128-byte line instead of eight)
  __shared__ float tr[TMAX / 32][256];
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
  for (int c = 0; c < MAXCH; c++) {
    const int col0 = (w * 32 + c * blockDim.x) * 8;          // first column of this warp's 256-column strip
#pragma unroll
    for (int which = 0; which < 2; which++) {
#pragma unroll
      for (int j = 0; j < 8; j++) tr[w][lane * 8 + j] = which ? db[c][j] : dg[c][j];
      __syncwarp();
      float* acc = which ? dbeta_acc : dgamma_acc;
#pragma unroll
      for (int i = 0; i < 8; i++) {
        const int col = col0 + i * 32 + lane;
        if (col < D) atomicAdd(acc + col, tr[w][i * 32 + lane]);
      }
      __syncwarp();
    }
  }
}

// ---- column sums (+ optional dtype-converting copy) ---------------------------------------------------
__global__ void __launch_bounds__(256) colsum_kernel(const void* __restrict__ in, int in_dt, long long ld, int M,
    int N, float* __restrict__ acc, void* __restrict__ copy_out, int copy_dt, long long ld_copy,
    int rows_per_block) {
  pdl_wait();
  pdl_trigger();
  __shared__ float sh[8][32][9];
  const int cx = threadIdx.x & 31, ry = threadIdx.x >> 5;
  const int col = (blockIdx.x * 32 + cx) * 8;
  const int r0 = blockIdx.y * rows_per_block;
  const int r1 = min(M, r0 + rows_per_block);
  float s[8];
#pragma unroll
  for (int j = 0; j < 8; j++) s[j] = 0.f;
  if (col < N) {
    int r = r0 + ry;
    // four rows requested before the first add (one load in flight per thread left the kernel latency-bound at ~3.7 TB/s on cold data)
    for (; r + 24 < r1; r += 32) {
      float v[4][8];
      if (in_dt == ORBIT_BF16) {
        uint4 raw[4];
#pragma unroll
        for (int u = 0; u < 4; u++) raw[u] = *reinterpret_cast<const uint4*>((const bf16*)in + (size_t)(r + 8 * u) * ld + col);
#pragma unroll
        for (int u = 0; u < 4; u++) {
          const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&raw[u]);
#pragma unroll
          for (int j = 0; j < 4; j++) { const float2 f = __bfloat1622float2(h[j]); v[u][2 * j] = f.x; v[u][2 * j + 1] = f.y; }
        }
      } else {
        float4 raw[8];
#pragma unroll
        for (int u = 0; u < 4; u++) {
          const float4* q = reinterpret_cast<const float4*>((const float*)in + (size_t)(r + 8 * u) * ld + col);
          raw[2 * u] = q[0]; raw[2 * u + 1] = q[1];
        }
#pragma unroll
        for (int u = 0; u < 4; u++) {
          v[u][0] = raw[2 * u].x; v[u][1] = raw[2 * u].y; v[u][2] = raw[2 * u].z; v[u][3] = raw[2 * u].w;
          v[u][4] = raw[2 * u + 1].x; v[u][5] = raw[2 * u + 1].y; v[u][6] = raw[2 * u + 1].z; v[u][7] = raw[2 * u + 1].w;
        }
      }
#pragma unroll
      for (int u = 0; u < 4; u++) {
#pragma unroll
        for (int j = 0; j < 8; j++) s[j] += v[u][j];
        if (copy_out) st8(copy_out, (size_t)(r + 8 * u) * ld_copy + col, copy_dt, v[u]);
      }
    }
    for (; r < r1; r += 8) {
      float v[8];
      ld8(in, (size_t)r * ld + col, in_dt, v);
#pragma unroll
      for (int j = 0; j < 8; j++) s[j] += v[j];
      if (copy_out) st8(copy_out, (size_t)r * ld_copy + col, copy_dt, v);
    }
  }
#pragma unroll
  for (int j = 0; j < 8; j++) sh[ry][cx][j] = s[j];
  __syncthreads();
  {  // thread t <-> column t of the block's 256: a warp's atomics cover 32 consecutive floats (one line)
    const int t = threadIdx.x, c2 = t >> 3, j = t & 7;
    const int colt = blockIdx.x * 256 + t;
    if (colt < N) {
      float tot = 0.f;
#pragma unroll
      for (int y = 0; y < 8; y++) tot += sh[y][c2][j];
      atomicAdd(acc + colt, tot);
    }
  }
}

__global__ void cast_kernel(const void* __restrict__ in, int in_dt, void* __restrict__ out, int out_dt, size_t n) {
  size_t stride = (size_t)gridDim.x * blockDim.x;
  size_t nv = n >> 3;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nv; i += stride) {
    float v[8];
    ld8(in, i * 8, in_dt, v);
    st8(out, i * 8, out_dt, v);
  }
  for (size_t i = (nv << 3) + (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
    stf(out, i, ldf(in, i, in_dt), out_dt);
}

// column sums of several matrices + casts of their and of other accumulators: see block_tail() in common.cuh
__global__ void __launch_bounds__(256) block_tail_kernel(TailSegs sums, CastSegs casts, int out_dt, unsigned int* tickets) {
  pdl_wait();
  pdl_trigger();
  __shared__ float sh[8][32][9];
  __shared__ unsigned int last;
  // accumulators that were complete before this launch: every block takes a slice
  for (int c = 0; c < casts.count; c++) {
    const CastSeg cs = casts.s[c];
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < cs.n; i += (size_t)gridDim.x * 256) stf(cs.dst, i, cs.src[i], out_dt);
  }
  int si = 0;
#pragma unroll 1
  while (si + 1 < sums.count && (int)blockIdx.x >= sums.s[si + 1].first_block) si++;
  const TailSeg sg = sums.s[si];
  const int b = blockIdx.x - sg.first_block, bx = b % sg.gx, by = b / sg.gx;
  const int cx = threadIdx.x & 31, ry = threadIdx.x >> 5;
  const int col = (bx * 32 + cx) * 8;
  const int r0 = by * sg.rows_per_block;
  const int r1 = min(sg.M, r0 + sg.rows_per_block);
  float s[8];
#pragma unroll
  for (int j = 0; j < 8; j++) s[j] = 0.f;
  // the dtype branch sits outside the row loop and four rows are requested before the first add: one load in flight per thread
  // (the form colsum_kernel has) moved 3.7 TB/s here, where the matrices are cold by the end of the block backward
  if (col < sg.N) {
    int r = r0 + ry;
    if (sg.in_dt == ORBIT_BF16) {
      const bf16* in = (const bf16*)sg.in + col;
      for (; r + 24 < r1; r += 32) {
        uint4 raw[4];
#pragma unroll
        for (int u = 0; u < 4; u++) raw[u] = __ldcs(reinterpret_cast<const uint4*>(in + (size_t)(r + 8 * u) * sg.ld));
#pragma unroll
        for (int u = 0; u < 4; u++) {
          const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&raw[u]);
#pragma unroll
          for (int j = 0; j < 4; j++) { const float2 f = __bfloat1622float2(h[j]); s[2 * j] += f.x; s[2 * j + 1] += f.y; }
        }
      }
    } else {
      const float* in = (const float*)sg.in + col;
      for (; r + 24 < r1; r += 32) {
        float4 raw[8];
#pragma unroll
        for (int u = 0; u < 4; u++) {
          const float4* q = reinterpret_cast<const float4*>(in + (size_t)(r + 8 * u) * sg.ld);
          raw[2 * u] = __ldcs(q); raw[2 * u + 1] = __ldcs(q + 1);
        }
#pragma unroll
        for (int u = 0; u < 4; u++) {
          s[0] += raw[2 * u].x; s[1] += raw[2 * u].y; s[2] += raw[2 * u].z; s[3] += raw[2 * u].w;
          s[4] += raw[2 * u + 1].x; s[5] += raw[2 * u + 1].y; s[6] += raw[2 * u + 1].z; s[7] += raw[2 * u + 1].w;
        }
      }
    }
    for (; r < r1; r += 8) {
      float v[8];
      ld8(sg.in, (size_t)r * sg.ld + col, sg.in_dt, v);
#pragma unroll
      for (int j = 0; j < 8; j++) s[j] += v[j];
    }
  }
#pragma unroll
  for (int j = 0; j < 8; j++) sh[ry][cx][j] = s[j];
  __syncthreads();
  const int t = threadIdx.x, colt = bx * 256 + t;
  if (colt < sg.N) {
    const int c2 = t >> 3, j = t & 7;
    float tot = 0.f;
#pragma unroll
    for (int y = 0; y < 8; y++) tot += sh[y][c2][j];
    atomicAdd(sg.acc + colt, tot);
  }
  __threadfence();                       // this block's atomics are performed before its ticket
  __syncthreads();
  unsigned int* ticket = tickets + sg.first_group + bx;
  if (threadIdx.x == 0) last = atomicAdd(ticket, 1u) == (unsigned int)sg.gy - 1;
  __syncthreads();
  if (!last) return;
  __threadfence();
  if (colt < sg.N) stf(sg.out, colt, __ldcg(sg.acc + colt), out_dt);
  if (threadIdx.x == 0) *ticket = 0u;
}

// several fp32 -> out_dt casts in one launch (the small parameter-gradient accumulators of a block backward)
__global__ void cast_multi_kernel(CastSegs segs, int out_dt) {
  pdl_wait();
  pdl_trigger();
  const CastSeg sg = segs.s[blockIdx.y];
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < sg.n; i += (size_t)gridDim.x * blockDim.x)
    stf(sg.dst, i, sg.src[i], out_dt);
}

__global__ void add_partial_kernel(const void* __restrict__ a, int a_dt, const float* __restrict__ part,
    const void* __restrict__ bias, int p_dt, void* __restrict__ out, int out_dt, size_t n8, int D8) {
  pdl_wait();
  pdl_trigger();
  size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n8; i += stride) {
    float va[8], vp[8], vb[8], o[8];
    ld8(a, i * 8, a_dt, va);
    ld8(part, i * 8, ORBIT_F32, vp);
    ld8(bias, (i % D8) * 8, p_dt, vb);
#pragma unroll
    for (int j = 0; j < 8; j++) o[j] = va[j] + vp[j] + vb[j];
    st8(out, i * 8, out_dt, o);
  }
}

// dy = 2 (y - t) / n ; loss += sum (y - t)^2 / n      (harness loss, BASELINE.json config 1: MSE)
__global__ void mse_kernel(const void* __restrict__ y, const void* __restrict__ t, int dt, void* __restrict__ dy,
                           float* __restrict__ loss, size_t n) {
  __shared__ float sh[32];
  size_t stride = (size_t)gridDim.x * blockDim.x;
  float acc = 0.f;
  const float inv = 1.0f / (float)n;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    float d = ldf(y, i, dt) - ldf(t, i, dt);
    acc += d * d;
    stf(dy, i, 2.f * d * inv, dt);
  }
  acc = block_sum(acc, sh);
  if (threadIdx.x == 0) atomicAdd(loss, acc * inv);
}

// TMA-staged kernels (layernorm_tma.cu) unless the row does not fit two stages or ORBIT_LN_ONEBLOCK=1 (A/B timing)
bool ln_use_tma(int D, int x_dt, int dout_dt, int add_dt, bool has_add) {
  static int forced = -1;
  if (forced < 0) { const char* e = getenv("ORBIT_LN_ONEBLOCK"); forced = (e && e[0] == '1') ? 1 : 0; }
  return !forced && layernorm_tma_supported(D, x_dt, dout_dt, add_dt, has_add);
}
int ln_threads(int D) {
  int nch = D / 8;
  int t = ((nch + 31) / 32) * 32;
  return t > 1024 ? 1024 : t;
}
}  // namespace

int layernorm_fwd(const void* x, int x_dt, const void* gamma, const void* beta, int p_dt, void* out, int out_dt,
                  float* mean, float* rstd, int M, int D, float eps, void* x_copy, cudaStream_t s) {
  // algorithmic bytes: read x, write out (+ the copy of x the backward needs)
  ProfScope prof(PROF_LN, (double)M * D * (dsize(x_dt) + dsize(out_dt) + (x_copy ? dsize(x_dt) : 0)), s);
  if (ln_use_tma(D, x_dt, -1, 0, false)) return layernorm_fwd_tma(x, x_dt, gamma, beta, p_dt, out, out_dt, mean, rstd, M, D, eps, x_copy, s);
  int thr = ln_threads(D);
  int maxch = cdiv(D / 8, thr);
  int grid = M < 148 * 4 ? M : 148 * 4;
  if (maxch <= 1) ln_fwd_kernel<1><<<grid, thr, 0, s>>>(x, x_dt, gamma, beta, p_dt, out, out_dt, mean, rstd, M, D, eps, x_copy);
  else if (maxch <= 2) ln_fwd_kernel<2><<<grid, thr, 0, s>>>(x, x_dt, gamma, beta, p_dt, out, out_dt, mean, rstd, M, D, eps, x_copy);
  else if (maxch <= 4) ln_fwd_kernel<4><<<grid, thr, 0, s>>>(x, x_dt, gamma, beta, p_dt, out, out_dt, mean, rstd, M, D, eps, x_copy);
  else if (maxch <= 8) ln_fwd_kernel<8><<<grid, thr, 0, s>>>(x, x_dt, gamma, beta, p_dt, out, out_dt, mean, rstd, M, D, eps, x_copy);
  else { set_error("layernorm: D=%d too large", D); return ORBIT_ERR_SHAPE; }
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int layernorm_bwd(const void* dout, int dout_dt, const void* x, int x_dt, const float* mean, const float* rstd,
                  const void* gamma, int p_dt, const void* add, int add_dt, float* dx_f32, void* dx_out,
                  int out_dt, float* dgamma_acc, float* dbeta_acc, int M, int D, cudaStream_t s) {
  // algorithmic bytes: read dout, x (+ add), write dx in the requested forms
  ProfScope prof(PROF_LN, (double)M * D * (dsize(dout_dt) + dsize(x_dt) + (add ? dsize(add_dt) : 0) + (dx_f32 ? 4 : 0) +
                                           (dx_out ? dsize(out_dt) : 0)), s);
  if (ln_use_tma(D, x_dt, dout_dt, add_dt, add != nullptr))
    return layernorm_bwd_tma(dout, dout_dt, x, x_dt, mean, rstd, gamma, p_dt, add, add_dt, dx_f32, dx_out, out_dt, dgamma_acc,
                            dbeta_acc, M, D, s);
  // <= 512 threads once a thread owns more than one 8-column chunk: the per-column dgamma/dbeta accumulators
  // (16 registers per chunk) then fit without spills
  const int nch = D / 8;
  int thr = ln_threads(D);
  int maxch = cdiv(nch, thr);
  if (maxch > 1) {
    maxch = cdiv(nch, 512);
    thr = ((cdiv(nch, maxch) + 31) / 32) * 32;
  }
  int grid = M < 148 * 4 ? M : 148 * 4;
#define LNB(C, T) ln_bwd_kernel<C, T><<<grid, thr, 0, s>>>(dout, dout_dt, x, x_dt, mean, rstd, gamma, p_dt, add, add_dt, \
                                                           dx_f32, dx_out, out_dt, dgamma_acc, dbeta_acc, M, D)
  if (maxch <= 1) {                      // register budget follows the block size (no spills up to 512 threads)
    if (thr <= 256) LNB(1, 256);
    else if (thr <= 512) LNB(1, 512);
    else LNB(1, 1024);
  }
  else if (maxch <= 2) LNB(2, 512);
  else if (maxch <= 3) LNB(3, 512);
  else if (maxch <= 4) LNB(4, 512);
  else { set_error("layernorm_bwd: D=%d too large", D); return ORBIT_ERR_SHAPE; }
#undef LNB
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int colsum(const void* in, int in_dt, long long ld, int M, int N, float* acc, void* copy_out, int copy_dt,
           long long ld_copy, cudaStream_t s) {
  int gx = cdiv(N, 256);
  int want_y = cdiv(148 * 4, gx);
  int rows_per_block = cdiv(M, want_y);
  rows_per_block = ((rows_per_block + 7) / 8) * 8;
  if (rows_per_block < 8) rows_per_block = 8;
  dim3 grid(gx, cdiv(M, rows_per_block));
  ORBIT_CUDA_CHECK(launch_pdl(colsum_kernel, grid, dim3(256), 0, s, in, in_dt, ld, M, N, acc, copy_out, copy_dt, ld_copy, rows_per_block));
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int cast_copy(const void* in, int in_dt, void* out, int out_dt, size_t n, cudaStream_t s) {
  if (n == 0) return ORBIT_OK;
  size_t blocks = (n / 8 + 255) / 256;
  if (blocks < 1) blocks = 1;
  if (blocks > 148 * 8) blocks = 148 * 8;
  cast_kernel<<<(int)blocks, 256, 0, s>>>(in, in_dt, out, out_dt, n);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int block_tail(TailSegs& sums, const CastSegs& casts, int out_dt, unsigned int* tickets, cudaStream_t s) {
  int total = 0, groups = 0, all_gx = 0;
  for (int i = 0; i < sums.count; i++) all_gx += cdiv(sums.s[i].N, 256);
  for (int i = 0; i < sums.count; i++) {
    TailSeg& t = sums.s[i];
    t.gx = cdiv(t.N, 256);
    int want_y = cdiv(num_sms() * 8, all_gx > 0 ? all_gx : 1);      // ~8 blocks per SM over all segments
    if (want_y < 1) want_y = 1;
    int rpb = cdiv(t.M, want_y);
    rpb = ((rpb + 7) / 8) * 8;
    if (rpb < 8) rpb = 8;
    t.rows_per_block = rpb;
    t.gy = cdiv(t.M, rpb);
    t.first_block = total; t.first_group = groups;
    total += t.gx * t.gy; groups += t.gx;
  }
  if (total == 0) return cast_multi(casts, out_dt, s);
  ORBIT_CUDA_CHECK(launch_pdl(block_tail_kernel, dim3(total), dim3(256), 0, s, sums, casts, out_dt, tickets));
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int cast_multi(const CastSegs& segs, int out_dt, cudaStream_t s) {
  if (segs.count <= 0) return ORBIT_OK;
  size_t mx = 0;
  for (int i = 0; i < segs.count; i++) mx = segs.s[i].n > mx ? segs.s[i].n : mx;
  int gx = (int)((mx + 255) / 256);
  if (gx > 148) gx = 148;
  if (gx < 1) gx = 1;
  ORBIT_CUDA_CHECK(launch_pdl(cast_multi_kernel, dim3(gx, segs.count), dim3(256), 0, s, segs, out_dt));
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int fill_zero(void* p, size_t bytes, cudaStream_t s) {
  if (bytes == 0) return ORBIT_OK;
  ORBIT_CUDA_CHECK(cudaMemsetAsync(p, 0, bytes, s));
  return ORBIT_OK;
}

int mse_loss_grad(const void* y, const void* t, int dt, void* dy, float* loss, size_t n, cudaStream_t s) {
  ORBIT_CUDA_CHECK(cudaMemsetAsync(loss, 0, sizeof(float), s));
  size_t blocks = (n + 255) / 256;
  if (blocks > 148 * 8) blocks = 148 * 8;
  mse_kernel<<<(int)blocks, 256, 0, s>>>(y, t, dt, dy, loss, n);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int add_partial(const void* a, int a_dt, const float* part, const void* bias, int p_dt, void* out, int out_dt,
                int M, int D, cudaStream_t s) {
  size_t n8 = (size_t)M * D / 8;
  size_t blocks = (n8 + 255) / 256;
  if (blocks > 148 * 8) blocks = 148 * 8;
  ORBIT_CUDA_CHECK(launch_pdl(add_partial_kernel, dim3((int)blocks), dim3(256), 0, s, a, a_dt, part, bias, p_dt, out, out_dt, n8, D / 8));
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

}  // namespace orbit
