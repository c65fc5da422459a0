// gemm_simt.cu -- generic fp32-FMA GEMM (any dtype / any stride) with the fused epilogue of GemmArgs.
// Used for ORBIT_F32 (true fp32 FMA, no TF32: reading R15/R17) and for small or oddly-aligned operands of
// the bf16 path; the large bf16 contractions go through gemm_tc.cu (tcgen05).
#include "common.cuh"

namespace orbit {

namespace {
constexpr int BM = 64, BN = 64, BK = 16, NT = 256;

__global__ void __launch_bounds__(NT) gemm_simt_kernel(GemmArgs g) {
  if (g.batch > 1) {   // strided batch: blockIdx.z selects the problem
    const size_t i = blockIdx.z;
    g.A = (const char*)g.A + i * g.a_bs * (g.in_dtype == ORBIT_BF16 ? 2 : 4);
    g.B = (const char*)g.B + i * g.b_bs * (g.in_dtype == ORBIT_BF16 ? 2 : 4);
    g.C = (char*)g.C + i * g.c_bs * (g.out_dtype == ORBIT_BF16 ? 2 : 4);
    if (g.bias) g.bias = (const char*)g.bias + i * g.bias_bs * (g.bias_dtype == ORBIT_BF16 ? 2 : 4);
  }
  __shared__ float As[BK][BM + 4];
  __shared__ float Bs[BK][BN + 4];
  const int t = threadIdx.x;
  const int m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;
  const int tx = t & 15, ty = t >> 4;
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; i++)
#pragma unroll
    for (int j = 0; j < 4; j++) acc[i][j] = 0.f;

  const bool a_mmajor = (g.a_rs == 1 && g.a_cs != 1);
  const bool b_nmajor = (g.b_cs == 1);
  for (int k0 = 0; k0 < g.K; k0 += BK) {
#pragma unroll
    for (int i = 0; i < 4; i++) {
      int r, k;
      if (a_mmajor) { r = t & 63; k = (t >> 6) + 4 * i; }
      else          { r = (t >> 4) + 16 * i; k = t & 15; }
      int gm = m0 + r, gk = k0 + k;
      float v = 0.f;
      if (gm < g.M && gk < g.K) v = ldf(g.A, (size_t)gm * g.a_rs + (size_t)gk * g.a_cs, g.in_dtype);
      As[k][r] = v;
    }
#pragma unroll
    for (int i = 0; i < 4; i++) {
      int c, k;
      if (b_nmajor) { c = t & 63; k = (t >> 6) + 4 * i; }
      else          { c = (t >> 4) + 16 * i; k = t & 15; }
      int gn = n0 + c, gk = k0 + k;
      float v = 0.f;
      if (gn < g.N && gk < g.K) v = ldf(g.B, (size_t)gk * g.b_rs + (size_t)gn * g.b_cs, g.in_dtype);
      Bs[k][c] = v;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < BK; k++) {
      float a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; i++) a[i] = As[k][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; j++) b[j] = Bs[k][tx * 4 + j];
#pragma unroll
      for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 4; j++) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; i++) {
    int m = m0 + ty * 4 + i;
    if (m >= g.M) continue;
#pragma unroll
    for (int j = 0; j < 4; j++) {
      int n = n0 + tx * 4 + j;
      if (n >= g.N) continue;
      float v = g.alpha * acc[i][j];
      if (g.bias) v += ldf(g.bias, n, g.bias_dtype);
      if (g.act == ACT_GELU) {
        if (g.aux_out) stf(g.aux_out, (size_t)m * g.ld_aux + n, v, g.aux_dtype);
        // the stored pre-activation is what backward sees: activate the rounded value
        if (g.aux_out && g.aux_dtype == ORBIT_BF16) v = __bfloat162float(__float2bfloat16_rn(v));
        v = gelu_f(v);
      } else if (g.act == ACT_GELU_GRAD) {
        v *= gelu_grad_f(ldf(g.aux_in, (size_t)m * g.ld_aux + n, g.aux_dtype));
      }
      if (g.resid) {
        int rm = g.resid_row_mod > 0 ? (m % g.resid_row_mod) : m;
        v += ldf(g.resid, (size_t)rm * g.ldr + n, g.resid_dtype);
      }
      size_t ci = (size_t)m * g.ldc + n;
      if (g.accumulate) v += ldf(g.C, ci, g.out_dtype);
      stf(g.C, ci, v, g.out_dtype);
    }
  }
}
}  // namespace

int gemm_simt(const GemmArgs& g, cudaStream_t s) {
  if (g.M <= 0 || g.N <= 0) return ORBIT_OK;
  dim3 grid(cdiv(g.N, BN), cdiv(g.M, BM), g.batch > 1 ? g.batch : 1);
  gemm_simt_kernel<<<grid, NT, 0, s>>>(g);
  ORBIT_LAUNCH_CHECK();
  return ORBIT_OK;
}

int gemm(const GemmArgs& g, cudaStream_t s) {
  if (g_force_simt != 1 && gemm_tc_supported(g)) return gemm_tc(g, s);
  return gemm_simt(g, s);
}

}  // namespace orbit
