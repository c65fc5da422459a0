// layernorm_tma.cu -- LayerNorm forward / backward (PAPER.md:88 pre-LN sub-layers, readings R5/R6) as HBM-streaming
// kernels whose loads are staged through shared memory by the TMA engine.
//
// One CTA per row, persistent over rows.  The rows of a CTA stream through a ring of NS shared-memory stages filled
// by 1-D bulk copies (cp.async.bulk, completion on an mbarrier), issued by one thread NS rows ahead: the bytes in
// flight per SM are (CTAs per SM) x NS x (row bytes) -- 100-200 KB -- and cost no registers, where the register-
// staged kernels of rowops.cu had one row per CTA in flight (16-24 KB per SM: 1.2-3.2 TB/s of 6.5).
// Row statistics take ONE exchange per row: warp partials into shared-memory slots (double buffered by row parity),
// one __syncthreads, every warp re-reduces the <= 32 slots.
// Algorithmic bytes: forward read M*D + write M*D (+ copy of x); backward read 3*M*D, write <= 2*M*D.
#include <cuda_runtime.h>
#include "common.cuh"
#include "ptx.cuh"
#include "vec8.cuh"

namespace orbit {
namespace {

constexpr int SLOTS = 32;          // warps per CTA

__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
// 8 consecutive elements of a staged row (shared memory, generic pointer)
__device__ __forceinline__ void lds8(const uint8_t* stage, int ch, int dt, float* v) {
  if (dt == ORBIT_BF16) ld8(stage, (size_t)ch * 8, ORBIT_BF16, v);
  else ld8(stage, (size_t)ch * 8, ORBIT_F32, v);
}

// ------------------------------------------------------------------------------------------------------
// forward: out = (x - mu) * rstd * gamma + beta ; mean / rstd saved ; optional copy of x (the block's saved input)
// Statistics: exact two-pass inside a warp (warp mean, then squared deviations from it), pooled over the warps with
//   mu = sum n_w m_w / D ,  var = (sum Q_w + sum n_w (m_w - mu)^2) / D      (no E[x^2] - mu^2 cancellation)
// ------------------------------------------------------------------------------------------------------
template <int MAXCH>
__global__ void __launch_bounds__(512, MAXCH >= 3 ? 2 : 1) ln_fwd_tma_kernel(const void* __restrict__ x, int x_dt, const void* __restrict__ gamma,
    const void* __restrict__ beta, int p_dt, void* __restrict__ out, int out_dt, float* __restrict__ mean,
    float* __restrict__ rstd, int M, int D, float eps, void* __restrict__ x_copy, int NS) {
  pdl_wait();          // PDL (common.cuh): nothing above touches global memory
  pdl_trigger();
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ float slots[2][3 * SLOTS];
  __shared__ __align__(8) uint64_t full_bar[8];
  const int nch = D >> 3;
  const uint32_t row_bytes = (uint32_t)D * (x_dt == ORBIT_BF16 ? 2u : 4u);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const int nrows = blockIdx.x < M ? (M - 1 - blockIdx.x) / gridDim.x + 1 : 0;     // rows blockIdx.x + i * gridDim.x
  if (threadIdx.x == 0) {
    for (int i = 0; i < NS; i++) ptx::mbar_init(ptx::smem_u32(&full_bar[i]), 1);
    ptx::fence_barrier_init();
  }
  __syncthreads();
  auto issue = [&](int i) {                       // thread 0: row i of this CTA into stage i % NS
    const int st = i % NS;
    const uint32_t bar = ptx::smem_u32(&full_bar[st]);
    ptx::mbar_expect_tx(bar, row_bytes);
    const size_t row = (size_t)blockIdx.x + (size_t)i * gridDim.x;
    bulk_load(ptx::smem_u32(smem + (size_t)st * row_bytes), (const uint8_t*)x + row * row_bytes, row_bytes, bar);
  };
  if (threadIdx.x == 0)
    for (int i = 0; i < NS && i < nrows; i++) issue(i);
  // this warp's element count is the same for every row
  int wcnt = 0;
#pragma unroll
  for (int c = 0; c < MAXCH; c++) wcnt += max(0, min(32, nch - (c * (int)blockDim.x + w * 32)));
  const float wn = 8.f * (float)wcnt;
  const float inv_wn = wcnt > 0 ? 1.f / wn : 0.f;
  const float invD = 1.f / (float)D;
  for (int i = 0; i < nrows; i++) {
    const int st = i % NS, par = i & 1;
    const size_t row = (size_t)blockIdx.x + (size_t)i * gridDim.x;
    ptx::mbar_wait(ptx::smem_u32(&full_bar[st]), (i / NS) & 1);
    const uint8_t* stage = smem + (size_t)st * row_bytes;
    float v[MAXCH][8];
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < MAXCH; c++) {
      const int ch = threadIdx.x + c * blockDim.x;
      if (ch < nch) {
        lds8(stage, ch, x_dt, v[c]);
#pragma unroll
        for (int j = 0; j < 8; j++) s += v[c][j];
      }
    }
    const float wm = warp_sum(s) * inv_wn;
    float q = 0.f;
#pragma unroll
    for (int c = 0; c < MAXCH; c++) {
      const int ch = threadIdx.x + c * blockDim.x;
      if (ch < nch) {
#pragma unroll
        for (int j = 0; j < 8; j++) { const float d = v[c][j] - wm; q += d * d; }
      }
    }
    q = warp_sum(q);
    if (lane == 0) { slots[par][w] = wn; slots[par][SLOTS + w] = wm; slots[par][2 * SLOTS + w] = q; }
    __syncthreads();                               // every thread has its chunks in registers: the stage is free
    if (threadIdx.x == 0 && i + NS < nrows) issue(i + NS);
    const float sn = lane < nw ? slots[par][lane] : 0.f, sm = lane < nw ? slots[par][SLOTS + lane] : 0.f;
    const float sq = lane < nw ? slots[par][2 * SLOTS + lane] : 0.f;
    const float mu = warp_sum(sn * sm) * invD;
    const float dm = sm - mu;
    const float rs = rsqrtf(warp_sum(sq + sn * dm * dm) * invD + eps);
    if (threadIdx.x == 0) { mean[row] = mu; rstd[row] = rs; }
#pragma unroll
    for (int c = 0; c < MAXCH; c++) {
      const int ch = threadIdx.x + c * blockDim.x;
      if (ch < nch) {
        const size_t off = row * D + (size_t)ch * 8;
        if (x_copy) st8(x_copy, off, x_dt, v[c]);
        float g[8], b[8], o[8];
        ld8(gamma, (size_t)ch * 8, p_dt, g);
        ld8(beta, (size_t)ch * 8, p_dt, b);
#pragma unroll
        for (int j = 0; j < 8; j++) o[j] = (v[c][j] - mu) * rs * g[j] + b[j];
        st8(out, off, out_dt, o);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------------
// backward (SURVEY.md 8(c) BLK'): zh = (x - mu) rstd, gh = dout * gamma,
//   dz = (gh - mean(gh) - zh * mean(gh * zh)) * rstd ;  dx = add + dz ;  dgamma += dout * zh ;  dbeta += dout
// A stage holds the row's x | dout | add slices.  Pass 1 (row sums, dgamma / dbeta) and pass 2 (dx) both read the
// stage, so nothing but the column sums lives in registers across the exchange; the stage of row i-1 is refilled
// after the barrier of row i.  dgamma / dbeta stay in registers over the rows of the CTA and are flushed once with
// fp32 atomics, transposed through shared memory so that one atomic instruction covers one 128-byte line.
// ------------------------------------------------------------------------------------------------------
template <int MAXCH>
__global__ void __launch_bounds__(512) ln_bwd_tma_kernel(const void* __restrict__ dout, int dout_dt,
    const void* __restrict__ x, int x_dt, const float* __restrict__ mean, const float* __restrict__ rstd,
    const void* __restrict__ gamma, int p_dt, const void* __restrict__ add, int add_dt,
    float* __restrict__ dx_f32, void* __restrict__ dx_out, int out_dt,
    float* __restrict__ dgamma_acc, float* __restrict__ dbeta_acc, int M, int D, int NS, int add_direct) {
  pdl_wait();          // PDL (common.cuh): nothing above touches global memory
  pdl_trigger();
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ float slots[2][2 * SLOTS];
  __shared__ __align__(8) uint64_t full_bar[8];
  const int nch = D >> 3;
  const uint32_t xb = (uint32_t)D * (x_dt == ORBIT_BF16 ? 2u : 4u), db_ = (uint32_t)D * (dout_dt == ORBIT_BF16 ? 2u : 4u);
  // add_direct: `add` is not staged (the three slices of a row would not fit twice) but read from global memory in pass 2
  const uint32_t ab = (add && !add_direct) ? (uint32_t)D * (add_dt == ORBIT_BF16 ? 2u : 4u) : 0u;
  const uint32_t stage_bytes = xb + db_ + ab;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const int nrows = blockIdx.x < M ? (M - 1 - blockIdx.x) / gridDim.x + 1 : 0;
  if (threadIdx.x == 0) {
    for (int i = 0; i < NS; i++) ptx::mbar_init(ptx::smem_u32(&full_bar[i]), 1);
    ptx::fence_barrier_init();
  }
  __syncthreads();
  auto issue = [&](int i) {
    const int st = i % NS;
    const uint32_t bar = ptx::smem_u32(&full_bar[st]);
    ptx::mbar_expect_tx(bar, stage_bytes);
    const size_t row = (size_t)blockIdx.x + (size_t)i * gridDim.x;
    const uint32_t s0 = ptx::smem_u32(smem + (size_t)st * stage_bytes);
    bulk_load(s0, (const uint8_t*)x + row * xb, xb, bar);
    bulk_load(s0 + xb, (const uint8_t*)dout + row * db_, db_, bar);
    if (ab) bulk_load(s0 + xb + db_, (const uint8_t*)add + row * ab, ab, bar);
  };
  if (threadIdx.x == 0)
    for (int i = 0; i < NS && i < nrows; i++) issue(i);
  float dg[MAXCH][8], db[MAXCH][8], gm[MAXCH][8];
#pragma unroll
  for (int c = 0; c < MAXCH; c++) {
    const int ch = threadIdx.x + c * blockDim.x;
#pragma unroll
    for (int j = 0; j < 8; j++) { dg[c][j] = 0.f; db[c][j] = 0.f; gm[c][j] = 0.f; }
    if (ch < nch) ld8(gamma, (size_t)ch * 8, p_dt, gm[c]);
  }
  const float invD = 1.f / (float)D;
  float mun = 0.f, rsn = 0.f;
  if (nrows > 0) { mun = mean[blockIdx.x]; rsn = rstd[blockIdx.x]; }
  for (int i = 0; i < nrows; i++) {
    const int st = i % NS, par = i & 1;
    const size_t row = (size_t)blockIdx.x + (size_t)i * gridDim.x;
    const float mu = mun, rs = rsn;
    if (i + 1 < nrows) { mun = mean[row + gridDim.x]; rsn = rstd[row + gridDim.x]; }
    ptx::mbar_wait(ptx::smem_u32(&full_bar[st]), (i / NS) & 1);
    const uint8_t* sx = smem + (size_t)st * stage_bytes;
    const uint8_t* sd = sx + xb;
    const uint8_t* sa = sd + db_;
    float s1 = 0.f, s2 = 0.f;
#pragma unroll
    for (int c = 0; c < MAXCH; c++) {
      const int ch = threadIdx.x + c * blockDim.x;
      if (ch < nch) {
        float xv[8], dv[8];
        lds8(sx, ch, x_dt, xv); lds8(sd, ch, dout_dt, dv);
#pragma unroll
        for (int j = 0; j < 8; j++) {
          const float z = (xv[j] - mu) * rs;
          dg[c][j] += dv[j] * z;
          db[c][j] += dv[j];
          const float g = dv[j] * gm[c][j];
          s1 += g; s2 += g * z;
        }
      }
    }
    s1 = warp_sum(s1); s2 = warp_sum(s2);
    if (lane == 0) { slots[par][w] = s1; slots[par][SLOTS + w] = s2; }
    __syncthreads();                               // also: every thread has finished pass 2 of row i-1
    if (threadIdx.x == 0 && i >= 1 && i - 1 + NS < nrows) issue(i - 1 + NS);
    const float m1 = warp_sum(lane < nw ? slots[par][lane] : 0.f) * invD;
    const float m2 = warp_sum(lane < nw ? slots[par][SLOTS + lane] : 0.f) * invD;
#pragma unroll
    for (int c = 0; c < MAXCH; c++) {
      const int ch = threadIdx.x + c * blockDim.x;
      if (ch < nch) {
        float xv[8], dv[8], o[8];
        lds8(sx, ch, x_dt, xv); lds8(sd, ch, dout_dt, dv);
        if (ab) lds8(sa, ch, add_dt, o);
        else if (add) ld8(add, row * D + (size_t)ch * 8, add_dt, o);
        else {
#pragma unroll
          for (int j = 0; j < 8; j++) o[j] = 0.f;
        }
#pragma unroll
        for (int j = 0; j < 8; j++) {
          const float z = (xv[j] - mu) * rs;
          o[j] += (dv[j] * gm[c][j] - m1 - z * m2) * rs;
        }
        const size_t off = row * D + (size_t)ch * 8;
        if (dx_f32) st8(dx_f32, off, ORBIT_F32, o);
        if (dx_out) st8(dx_out, off, out_dt, o);
      }
    }
  }
  // dgamma / dbeta flush through the (now idle) staging memory: [warp][256] floats
  __syncthreads();
  float* tr = reinterpret_cast<float*>(smem) + w * 256;
#pragma unroll
  for (int c = 0; c < MAXCH; c++) {
    const int col0 = (w * 32 + c * blockDim.x) * 8;
#pragma unroll
    for (int which = 0; which < 2; which++) {
#pragma unroll
      for (int j = 0; j < 8; j++) tr[lane * 8 + j] = which ? db[c][j] : dg[c][j];
      __syncwarp();
      float* acc = which ? dbeta_acc : dgamma_acc;
#pragma unroll
      for (int k = 0; k < 8; k++) {
        const int col = col0 + k * 32 + lane;
        if (col < D) atomicAdd(acc + col, tr[k * 32 + lane]);
      }
      __syncwarp();
    }
  }
}

// ------------------------------------------------------------------------------------------------------
// Short rows (D <= 4096: one chunk per thread): R consecutive rows (contiguous in memory: ONE bulk copy) per stage and
// per exchange.  A row's dependent chain (shuffle reductions, barrier, second reduction) is ~1.5-2 us whatever its
// length, so with one 4-8 KB row per exchange and 4 CTAs per SM the kernels stalled at 2.5 TB/s; R rows per exchange
// put R times the bytes behind every chain.
// ------------------------------------------------------------------------------------------------------
template <int R>
__global__ void __launch_bounds__(512) ln_fwd_tma_rows_kernel(const void* __restrict__ x, int x_dt,
    const void* __restrict__ gamma, const void* __restrict__ beta, int p_dt, void* __restrict__ out, int out_dt,
    float* __restrict__ mean, float* __restrict__ rstd, int M, int D, float eps, void* __restrict__ x_copy, int NS) {
  pdl_wait();          // PDL (common.cuh): nothing above touches global memory
  pdl_trigger();
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ float slots[2][R][3 * SLOTS];
  __shared__ __align__(8) uint64_t full_bar[8];
  const int nch = D >> 3;
  const uint32_t row_bytes = (uint32_t)D * (x_dt == ORBIT_BF16 ? 2u : 4u), stage_bytes = R * row_bytes;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const int ngroups = (M + R - 1) / R;
  const int ngr = blockIdx.x < ngroups ? (ngroups - 1 - blockIdx.x) / gridDim.x + 1 : 0;
  if (threadIdx.x == 0) {
    for (int i = 0; i < NS; i++) ptx::mbar_init(ptx::smem_u32(&full_bar[i]), 1);
    ptx::fence_barrier_init();
  }
  __syncthreads();
  auto issue = [&](int i) {
    const int st = i % NS;
    const uint32_t bar = ptx::smem_u32(&full_bar[st]);
    const size_t row0 = ((size_t)blockIdx.x + (size_t)i * gridDim.x) * R;
    const uint32_t bytes = (uint32_t)min((size_t)R, (size_t)M - row0) * row_bytes;
    ptx::mbar_expect_tx(bar, bytes);
    bulk_load(ptx::smem_u32(smem + (size_t)st * stage_bytes), (const uint8_t*)x + row0 * row_bytes, bytes, bar);
  };
  if (threadIdx.x == 0)
    for (int i = 0; i < NS && i < ngr; i++) issue(i);
  const int ch = threadIdx.x;
  const bool act = ch < nch;
  const float wn = 8.f * (float)max(0, min(32, nch - w * 32));
  const float inv_wn = wn > 0.f ? 1.f / wn : 0.f;
  const float invD = 1.f / (float)D;
  float g[8], b[8];
#pragma unroll
  for (int j = 0; j < 8; j++) { g[j] = 0.f; b[j] = 0.f; }
  if (act) { ld8(gamma, (size_t)ch * 8, p_dt, g); ld8(beta, (size_t)ch * 8, p_dt, b); }
  for (int i = 0; i < ngr; i++) {
    const int st = i % NS, par = i & 1;
    const size_t row0 = ((size_t)blockIdx.x + (size_t)i * gridDim.x) * R;
    const int cnt = (int)min((size_t)R, (size_t)M - row0);
    ptx::mbar_wait(ptx::smem_u32(&full_bar[st]), (i / NS) & 1);
    const uint8_t* stage = smem + (size_t)st * stage_bytes;
    float v[R][8], s[R], q[R];
#pragma unroll
    for (int r = 0; r < R; r++) {
      s[r] = 0.f;
#pragma unroll
      for (int j = 0; j < 8; j++) v[r][j] = 0.f;
      if (act && r < cnt) {
        lds8(stage + (size_t)r * row_bytes, ch, x_dt, v[r]);
#pragma unroll
        for (int j = 0; j < 8; j++) s[r] += v[r][j];
      }
    }
#pragma unroll
    for (int r = 0; r < R; r++) s[r] = warp_sum(s[r]) * inv_wn;
#pragma unroll
    for (int r = 0; r < R; r++) {
      q[r] = 0.f;
      if (act) {
#pragma unroll
        for (int j = 0; j < 8; j++) { const float d = v[r][j] - s[r]; q[r] += d * d; }
      }
    }
#pragma unroll
    for (int r = 0; r < R; r++) q[r] = warp_sum(q[r]);
    if (lane == 0) {
#pragma unroll
      for (int r = 0; r < R; r++) { slots[par][r][w] = wn; slots[par][r][SLOTS + w] = s[r]; slots[par][r][2 * SLOTS + w] = q[r]; }
    }
    __syncthreads();                               // every thread has its chunks in registers: the stage is free
    if (threadIdx.x == 0 && i + NS < ngr) issue(i + NS);
    float mu[R], rs[R];
#pragma unroll
    for (int r = 0; r < R; r++) {
      const float sn = lane < nw ? slots[par][r][lane] : 0.f, sm = lane < nw ? slots[par][r][SLOTS + lane] : 0.f;
      mu[r] = warp_sum(sn * sm) * invD;
    }
#pragma unroll
    for (int r = 0; r < R; r++) {
      const float sn = lane < nw ? slots[par][r][lane] : 0.f, sm = lane < nw ? slots[par][r][SLOTS + lane] : 0.f;
      const float sq = lane < nw ? slots[par][r][2 * SLOTS + lane] : 0.f;
      const float dm = sm - mu[r];
      rs[r] = rsqrtf(warp_sum(sq + sn * dm * dm) * invD + eps);
    }
    if (threadIdx.x < cnt) {
#pragma unroll
      for (int r = 0; r < R; r++)
        if (threadIdx.x == r) { mean[row0 + r] = mu[r]; rstd[row0 + r] = rs[r]; }
    }
    if (act) {
#pragma unroll
      for (int r = 0; r < R; r++) {
        if (r < cnt) {
          const size_t off = (row0 + r) * D + (size_t)ch * 8;
          if (x_copy) st8(x_copy, off, x_dt, v[r]);
          float o[8];
#pragma unroll
          for (int j = 0; j < 8; j++) o[j] = (v[r][j] - mu[r]) * rs[r] * g[j] + b[j];
          st8(out, off, out_dt, o);
        }
      }
    }
  }
}

template <int R>
__global__ void __launch_bounds__(512) ln_bwd_tma_rows_kernel(const void* __restrict__ dout, int dout_dt,
    const void* __restrict__ x, int x_dt, const float* __restrict__ mean, const float* __restrict__ rstd,
    const void* __restrict__ gamma, int p_dt, const void* __restrict__ add, int add_dt,
    float* __restrict__ dx_f32, void* __restrict__ dx_out, int out_dt,
    float* __restrict__ dgamma_acc, float* __restrict__ dbeta_acc, int M, int D, int NS) {
  pdl_wait();          // PDL (common.cuh): nothing above touches global memory
  pdl_trigger();
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ float slots[2][R][2 * SLOTS];
  __shared__ __align__(8) uint64_t full_bar[8];
  const int nch = D >> 3;
  const uint32_t xb = (uint32_t)D * (x_dt == ORBIT_BF16 ? 2u : 4u), db_ = (uint32_t)D * (dout_dt == ORBIT_BF16 ? 2u : 4u);
  const uint32_t ab = add ? (uint32_t)D * (add_dt == ORBIT_BF16 ? 2u : 4u) : 0u;
  const uint32_t stage_bytes = R * (xb + db_ + ab);          // [R rows of x | R rows of dout | R rows of add]
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const int ngroups = (M + R - 1) / R;
  const int ngr = blockIdx.x < ngroups ? (ngroups - 1 - blockIdx.x) / gridDim.x + 1 : 0;
  if (threadIdx.x == 0) {
    for (int i = 0; i < NS; i++) ptx::mbar_init(ptx::smem_u32(&full_bar[i]), 1);
    ptx::fence_barrier_init();
  }
  __syncthreads();
  auto issue = [&](int i) {
    const int st = i % NS;
    const uint32_t bar = ptx::smem_u32(&full_bar[st]);
    const size_t row0 = ((size_t)blockIdx.x + (size_t)i * gridDim.x) * R;
    const uint32_t cnt = (uint32_t)min((size_t)R, (size_t)M - row0);
    ptx::mbar_expect_tx(bar, cnt * (xb + db_ + ab));
    const uint32_t s0 = ptx::smem_u32(smem + (size_t)st * stage_bytes);
    bulk_load(s0, (const uint8_t*)x + row0 * xb, cnt * xb, bar);
    bulk_load(s0 + R * xb, (const uint8_t*)dout + row0 * db_, cnt * db_, bar);
    if (ab) bulk_load(s0 + R * (xb + db_), (const uint8_t*)add + row0 * ab, cnt * ab, bar);
  };
  if (threadIdx.x == 0)
    for (int i = 0; i < NS && i < ngr; i++) issue(i);
  const int ch = threadIdx.x;
  const bool act = ch < nch;
  float dg[8], db[8], gm[8];
#pragma unroll
  for (int j = 0; j < 8; j++) { dg[j] = 0.f; db[j] = 0.f; gm[j] = 0.f; }
  if (act) ld8(gamma, (size_t)ch * 8, p_dt, gm);
  const float invD = 1.f / (float)D;
  float mun[R], rsn[R];
#pragma unroll
  for (int r = 0; r < R; r++) {
    const size_t rr = (size_t)blockIdx.x * R + r;
    mun[r] = rr < (size_t)M ? mean[rr] : 0.f;
    rsn[r] = rr < (size_t)M ? rstd[rr] : 0.f;
  }
  for (int i = 0; i < ngr; i++) {
    const int st = i % NS, par = i & 1;
    const size_t row0 = ((size_t)blockIdx.x + (size_t)i * gridDim.x) * R;
    const int cnt = (int)min((size_t)R, (size_t)M - row0);
    float mu[R], rs[R], s1[R], s2[R];
#pragma unroll
    for (int r = 0; r < R; r++) { mu[r] = mun[r]; rs[r] = rsn[r]; }
    if (i + 1 < ngr) {                               // next group's statistics: requested a whole group ahead
      const size_t nrow0 = row0 + (size_t)gridDim.x * R;
#pragma unroll
      for (int r = 0; r < R; r++) {
        mun[r] = nrow0 + r < (size_t)M ? mean[nrow0 + r] : 0.f;
        rsn[r] = nrow0 + r < (size_t)M ? rstd[nrow0 + r] : 0.f;
      }
    }
    ptx::mbar_wait(ptx::smem_u32(&full_bar[st]), (i / NS) & 1);
    const uint8_t* sx = smem + (size_t)st * stage_bytes;
    const uint8_t* sd = sx + R * xb;
    const uint8_t* sa = sd + R * db_;
#pragma unroll
    for (int r = 0; r < R; r++) {
      s1[r] = 0.f; s2[r] = 0.f;
      if (act && r < cnt) {
        float xv[8], dv[8];
        lds8(sx + (size_t)r * xb, ch, x_dt, xv); lds8(sd + (size_t)r * db_, ch, dout_dt, dv);
#pragma unroll
        for (int j = 0; j < 8; j++) {
          const float z = (xv[j] - mu[r]) * rs[r];
          dg[j] += dv[j] * z;
          db[j] += dv[j];
          const float g = dv[j] * gm[j];
          s1[r] += g; s2[r] += g * z;
        }
      }
    }
#pragma unroll
    for (int r = 0; r < R; r++) { s1[r] = warp_sum(s1[r]); s2[r] = warp_sum(s2[r]); }
    if (lane == 0) {
#pragma unroll
      for (int r = 0; r < R; r++) { slots[par][r][w] = s1[r]; slots[par][r][SLOTS + w] = s2[r]; }
    }
    __syncthreads();                               // also: every thread has finished pass 2 of group i-1
    if (threadIdx.x == 0 && i >= 1 && i - 1 + NS < ngr) issue(i - 1 + NS);
#pragma unroll
    for (int r = 0; r < R; r++) {
      s1[r] = warp_sum(lane < nw ? slots[par][r][lane] : 0.f) * invD;
      s2[r] = warp_sum(lane < nw ? slots[par][r][SLOTS + lane] : 0.f) * invD;
    }
    if (act) {
#pragma unroll
      for (int r = 0; r < R; r++) {
        if (r < cnt) {
          float xv[8], dv[8], o[8];
          lds8(sx + (size_t)r * xb, ch, x_dt, xv); lds8(sd + (size_t)r * db_, ch, dout_dt, dv);
          if (ab) lds8(sa + (size_t)r * ab, ch, add_dt, o);
          else {
#pragma unroll
            for (int j = 0; j < 8; j++) o[j] = 0.f;
          }
#pragma unroll
          for (int j = 0; j < 8; j++) {
            const float z = (xv[j] - mu[r]) * rs[r];
            o[j] += (dv[j] * gm[j] - s1[r] - z * s2[r]) * rs[r];
          }
          const size_t off = (row0 + r) * D + (size_t)ch * 8;
          if (dx_f32) st8(dx_f32, off, ORBIT_F32, o);
          if (dx_out) st8(dx_out, off, out_dt, o);
        }
      }
    }
  }
  __syncthreads();
  float* tr = reinterpret_cast<float*>(smem) + w * 256;
  const int col0 = w * 32 * 8;
#pragma unroll
  for (int which = 0; which < 2; which++) {
#pragma unroll
    for (int j = 0; j < 8; j++) tr[lane * 8 + j] = which ? db[j] : dg[j];
    __syncwarp();
    float* acc = which ? dbeta_acc : dgamma_acc;
#pragma unroll
    for (int k = 0; k < 8; k++) {
      const int col = col0 + k * 32 + lane;
      if (col < D) atomicAdd(acc + col, tr[k * 32 + lane]);
    }
    __syncwarp();
  }
}

constexpr int SMEM_MAX = 227 * 1024 - 4096;      // dynamic shared memory per CTA (static slots / barriers, <= 3.3 KB, come on top)

// threads per CTA and chunks per thread for a row of D columns: up to 512 threads with <= 4 chunks each
bool plan(int D, int* T, int* MAXCH) {
  if (D % 8 || D <= 0) return false;
  const int nch = D / 8;
  const int mc = cdiv(nch, 512);
  if (mc > 4) return false;                      // D > 16384: the one-block kernels of rowops.cu
  *T = ((cdiv(nch, mc) + 31) / 32) * 32;
  *MAXCH = mc;
  return true;
}
// CTAs per SM and ring depth: as many CTAs as threads / registers allow (capped), then as many stages as fit
void shape(int T, int regs, size_t stage_bytes, int cap, int* per_sm, int* NS, size_t* smem) {
  int bps = 2048 / T;
  const int by_regs = 65536 / (regs * T);
  if (by_regs < bps) bps = by_regs;
  if (bps > cap) bps = cap;
  if (bps < 1) bps = 1;
  while (bps > 1 && (size_t)bps * (2 * stage_bytes + 1024) > (size_t)SMEM_MAX) bps--;
  int ns = (int)((size_t)SMEM_MAX / bps / stage_bytes);
  if (ns > 4) ns = 4;
  if (ns < 2) ns = 2;
  size_t need = (size_t)ns * stage_bytes;
  const size_t tr = (size_t)(T / 32) * 1024;
  if (need < tr) need = tr;
  *per_sm = bps; *NS = ns; *smem = need;
}
// rows per stage of the short-row kernels: ~16-24 KB per stage, and no more than leaves every SM a few groups
int rows_per_stage(size_t row_stage_bytes, int M) {
  int r = (int)(24 * 1024 / row_stage_bytes);
  while (r > 1 && M / r < 148 * 4) r >>= 1;
  return r >= 4 ? 4 : (r >= 2 ? 2 : 1);
}
}  // namespace

bool layernorm_tma_supported(int D, int x_dt, int dout_dt, int add_dt, bool has_add) {
  int t, mc;
  if (!plan(D, &t, &mc)) return false;
  (void)add_dt; (void)has_add;                    // `add` is read from global memory when it does not fit the stages
  const size_t stage = (size_t)D * (dsize(x_dt) + (dout_dt >= 0 ? dsize(dout_dt) : 0));
  return 2 * stage <= (size_t)SMEM_MAX;
}

int layernorm_fwd_tma(const void* x, int x_dt, const void* gamma, const void* beta, int p_dt, void* out, int out_dt,
                      float* mean, float* rstd, int M, int D, float eps, void* x_copy, cudaStream_t s) {
  int T, MC;
  if (!plan(D, &T, &MC)) { set_error("layernorm_tma: D=%d unsupported", D); return ORBIT_ERR_SHAPE; }
  int per_sm, NS; size_t smem;
#define LNF(C)                                                                                                       \
  do {                                                                                                               \
    static std::atomic<int> regs_c{0};   /* registers per thread: a property of the binary, not of the device */          \
    int regs = regs_c.load(std::memory_order_relaxed);                                                               \
    if (!regs) {                                                                                                     \
      cudaFuncAttributes fa;                                                                                         \
      ORBIT_CUDA_CHECK(cudaFuncGetAttributes(&fa, (const void*)ln_fwd_tma_kernel<C>));\
      regs = fa.numRegs;                                                                                             \
      regs_c.store(regs, std::memory_order_relaxed);                                                                 \
    }                                                                                                                \
    ORBIT_SMEM_ATTR(ln_fwd_tma_kernel<C>, SMEM_MAX);                                                                  \
    shape(T, regs, (size_t)D * dsize(x_dt), 8, &per_sm, &NS, &smem);                                                 \
    int grid = 148 * per_sm;                                                                                         \
    if (grid > M) grid = M;                                                                                          \
    ORBIT_CUDA_CHECK(launch_pdl(ln_fwd_tma_kernel<C>, dim3(grid), dim3(T), smem, s, x, x_dt, gamma, beta, p_dt, out, out_dt, mean, rstd, M, D, eps, x_copy, NS)); \
  } while (0)
#define LNFR(RR)                                                                                                     \
  do {                                                                                                               \
    static std::atomic<int> regs_c{0};   /* registers per thread: a property of the binary, not of the device */          \
    int regs = regs_c.load(std::memory_order_relaxed);                                                               \
    if (!regs) {                                                                                                     \
      cudaFuncAttributes fa;                                                                                         \
      ORBIT_CUDA_CHECK(cudaFuncGetAttributes(&fa, (const void*)ln_fwd_tma_rows_kernel<RR>));\
      regs = fa.numRegs;                                                                                             \
      regs_c.store(regs, std::memory_order_relaxed);                                                                 \
    }                                                                                                                \
    ORBIT_SMEM_ATTR(ln_fwd_tma_rows_kernel<RR>, SMEM_MAX);                                                                  \
    shape(T, regs, (size_t)RR * D * dsize(x_dt), 8, &per_sm, &NS, &smem);                                            \
    int grid = 148 * per_sm;                                                                                         \
    if (grid > cdiv(M, RR)) grid = cdiv(M, RR);                                                                      \
    ORBIT_CUDA_CHECK(launch_pdl(ln_fwd_tma_rows_kernel<RR>, dim3(grid), dim3(T), smem, s, x, x_dt, gamma, beta, p_dt, out, out_dt, mean, rstd, M, D, eps, x_copy, NS)); \
  } while (0)
  if (MC == 1) {
    const int R = rows_per_stage((size_t)D * dsize(x_dt), M);
    if (R == 4) LNFR(4); else if (R == 2) LNFR(2); else LNFR(1);
  } else
  switch (MC) { case 2: LNF(2); break; case 3: LNF(3); break; default: LNF(4); break; }
#undef LNFR
#undef LNF
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int layernorm_bwd_tma(const void* dout, int dout_dt, const void* x, int x_dt, const float* mean, const float* rstd,
                      const void* gamma, int p_dt, const void* add, int add_dt, float* dx_f32, void* dx_out,
                      int out_dt, float* dgamma_acc, float* dbeta_acc, int M, int D, cudaStream_t s) {
  int T, MC;
  if (!plan(D, &T, &MC)) { set_error("layernorm_tma: D=%d unsupported", D); return ORBIT_ERR_SHAPE; }
  int per_sm, NS; size_t smem;
  size_t stage = (size_t)D * (dsize(x_dt) + dsize(dout_dt) + (add ? dsize(add_dt) : 0));
  int add_direct = 0;
  if (2 * stage > (size_t)SMEM_MAX) { add_direct = 1; stage = (size_t)D * (dsize(x_dt) + dsize(dout_dt)); }
#define LNB(C)                                                                                                       \
  do {                                                                                                               \
    static std::atomic<int> regs_c{0};   /* registers per thread: a property of the binary, not of the device */          \
    int regs = regs_c.load(std::memory_order_relaxed);                                                               \
    if (!regs) {                                                                                                     \
      cudaFuncAttributes fa;                                                                                         \
      ORBIT_CUDA_CHECK(cudaFuncGetAttributes(&fa, (const void*)ln_bwd_tma_kernel<C>));\
      regs = fa.numRegs;                                                                                             \
      regs_c.store(regs, std::memory_order_relaxed);                                                                 \
    }                                                                                                                \
    ORBIT_SMEM_ATTR(ln_bwd_tma_kernel<C>, SMEM_MAX);                                                                  \
    shape(T, regs, stage, 4, &per_sm, &NS, &smem);                                                                   \
    int grid = 148 * per_sm;                                                                                         \
    if (grid > M) grid = M;                                                                                          \
    ORBIT_CUDA_CHECK(launch_pdl(ln_bwd_tma_kernel<C>, dim3(grid), dim3(T), smem, s, dout, dout_dt, x, x_dt, mean, rstd, gamma, p_dt, add, \
                                add_dt, dx_f32, dx_out, out_dt, dgamma_acc, dbeta_acc, M, D, NS, add_direct));        \
  } while (0)
#define LNBR(RR)                                                                                                     \
  do {                                                                                                               \
    static std::atomic<int> regs_c{0};   /* registers per thread: a property of the binary, not of the device */          \
    int regs = regs_c.load(std::memory_order_relaxed);                                                               \
    if (!regs) {                                                                                                     \
      cudaFuncAttributes fa;                                                                                         \
      ORBIT_CUDA_CHECK(cudaFuncGetAttributes(&fa, (const void*)ln_bwd_tma_rows_kernel<RR>));\
      regs = fa.numRegs;                                                                                             \
      regs_c.store(regs, std::memory_order_relaxed);                                                                 \
    }                                                                                                                \
    ORBIT_SMEM_ATTR(ln_bwd_tma_rows_kernel<RR>, SMEM_MAX);                                                                  \
    shape(T, regs, (size_t)RR * stage, 4, &per_sm, &NS, &smem);                                                      \
    int grid = 148 * per_sm;                                                                                         \
    if (grid > cdiv(M, RR)) grid = cdiv(M, RR);                                                                      \
    ORBIT_CUDA_CHECK(launch_pdl(ln_bwd_tma_rows_kernel<RR>, dim3(grid), dim3(T), smem, s, dout, dout_dt, x, x_dt, mean, rstd, gamma, p_dt, \
                                add, add_dt, dx_f32, dx_out, out_dt, dgamma_acc, dbeta_acc, M, D, NS));               \
  } while (0)
  if (MC == 1) {
    const int R = rows_per_stage(stage, M);
    if (R == 4) LNBR(4); else if (R == 2) LNBR(2); else LNBR(1);
  } else
  switch (MC) { case 2: LNB(2); break; case 3: LNB(3); break; default: LNB(4); break; }
#undef LNBR
#undef LNB
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

}  // namespace orbit
