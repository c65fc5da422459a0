// api_common.cu -- error state, device check, diagnostics, tokenise and Eq.(2)/(3) chain entry points.
#include <stdarg.h>
#include <stdlib.h>
#include <string.h>
#include "api_util.cuh"
#include "frontend.cuh"
#include "orbit_debug.h"

namespace orbit {
int attention_probe_read(unsigned long long* out, int n, int reset);   // attention_tc5.cu (probe build only)

static thread_local char g_err[512] = "";
thread_local long long g_launches = 0;
#ifdef ORBIT_DEBUG_SWITCH
int g_force_simt = 0;
#endif

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}

int check_device() {
  // cached per device ordinal: 0 = unknown, 1 = sm_100-class, 2 = other architecture
  static std::atomic<int> cached[ORBIT_MAX_DEV];
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) {
    cudaGetLastError();
    set_error("no usable CUDA device");
    return ORBIT_ERR_ARCH;
  }
  const bool cacheable = dev >= 0 && dev < ORBIT_MAX_DEV;
  if (cacheable && cached[dev].load(std::memory_order_relaxed) == 1) return ORBIT_OK;
  int major = 0, minor = 0;
  if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev) != cudaSuccess) {
    cudaGetLastError();
    set_error("no usable CUDA device");
    return ORBIT_ERR_ARCH;
  }
  if (major != 10) {
    set_error("device %d is sm_%d%d; liborbit is built for sm_100a only (no fallback)", dev, major, minor);
    return ORBIT_ERR_ARCH;
  }
  if (cacheable) cached[dev].store(1, std::memory_order_relaxed);
  return ORBIT_OK;
}

// ---- per-launch event timing ------------------------------------------------------------------------------------------
namespace {
struct ProfState {
  bool on = false;
  static constexpr int MAXP = 32768;
  cudaEvent_t* ev = nullptr;     // 2 * MAXP events, created on first enable
  double* work = nullptr;
  unsigned char* cat = nullptr;
  int n = 0;
} g_prof;
}  // namespace
int prof_enable(int on) {
  if (on && !g_prof.ev) {
    g_prof.ev = new cudaEvent_t[2 * ProfState::MAXP];
    g_prof.work = new double[ProfState::MAXP];
    g_prof.cat = new unsigned char[ProfState::MAXP];
    for (int i = 0; i < 2 * ProfState::MAXP; i++) ORBIT_CUDA_CHECK(cudaEventCreate(&g_prof.ev[i]));
  }
  g_prof.on = on != 0;
  g_prof.n = 0;
  return ORBIT_OK;
}
int prof_collect(int cat, double* ms, double* work, long long* launches) {
  double t = 0, w = 0;
  long long n = 0;
  for (int i = 0; i < g_prof.n; i++) {
    if (g_prof.cat[i] != cat) continue;
    float e = 0.f;
    ORBIT_CUDA_CHECK(cudaEventSynchronize(g_prof.ev[2 * i + 1]));
    ORBIT_CUDA_CHECK(cudaEventElapsedTime(&e, g_prof.ev[2 * i], g_prof.ev[2 * i + 1]));
    t += e; w += g_prof.work[i]; n++;
  }
  if (ms) *ms = t;
  if (work) *work = w;
  if (launches) *launches = n;
  return ORBIT_OK;
}
ProfScope::ProfScope(int cat, double work, cudaStream_t stream) : slot(-1), s(stream) {
  if (!g_prof.on || g_prof.n >= ProfState::MAXP) return;
  slot = g_prof.n++;
  g_prof.cat[slot] = (unsigned char)cat;
  g_prof.work[slot] = work;
  cudaEventRecord(g_prof.ev[2 * slot], s);
}
ProfScope::~ProfScope() {
  if (slot >= 0) cudaEventRecord(g_prof.ev[2 * slot + 1], s);
}

bool pdl_enabled() {
  static const int v = [] { const char* e = getenv("ORBIT_PDL"); return (e && e[0] == '0') ? 0 : 1; }();
  return v != 0;
}
int device_ordinal() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return 0; }
  return dev;
}
int smem_attr_once(SmemAttrOnce& st, const void* fn, int bytes) {
  const int dev = device_ordinal();
  if (dev >= 0 && dev < ORBIT_MAX_DEV && st.bytes[dev].load(std::memory_order_acquire) >= bytes) return ORBIT_OK;
  ORBIT_CUDA_CHECK(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  if (dev >= 0 && dev < ORBIT_MAX_DEV) {
    int cur = st.bytes[dev].load(std::memory_order_relaxed);
    while (cur < bytes && !st.bytes[dev].compare_exchange_weak(cur, bytes, std::memory_order_release)) {}
  }
  return ORBIT_OK;
}
int num_sms() {
  static std::atomic<int> n[ORBIT_MAX_DEV];
  const int dev = device_ordinal();
  const bool cacheable = dev >= 0 && dev < ORBIT_MAX_DEV;
  int v = cacheable ? n[dev].load(std::memory_order_relaxed) : 0;
  if (!v) {
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v <= 0) { cudaGetLastError(); v = 148; }
    if (cacheable) n[dev].store(v, std::memory_order_relaxed);
  }
  return v;
}

bool valid_dtype(int dt) { return dt == ORBIT_F32 || dt == ORBIT_BF16; }
bool aligned16(const void* p) { return (((uintptr_t)p) & 15) == 0; }

}  // namespace orbit

using namespace orbit;

extern "C" {

const char* orbit_last_error(void) { return g_err; }
int orbit_version(void) { return ORBIT_VERSION; }
long long orbit_launch_count(void) { return g_launches; }
void orbit_reset_launch_count(void) { g_launches = 0; }
#ifdef ORBIT_DEBUG_SWITCH
void orbit_set_debug_force_simt(int on) { g_force_simt = on; }   // csrc/orbit_debug.h; not part of include/orbit.h
#ifdef ORBIT_PROBE_TIMELINE
int orbit_debug_read_probe(unsigned long long* out, int n, int reset) { return orbit::attention_probe_read(out, n, reset); }
#endif
#endif

// ------------------------------------------------------------------------------------------------------
// a1 / a1'
// ------------------------------------------------------------------------------------------------------
static int check_embed(const orbit_embed_desc* d) {
  if (!d) { set_error("embed desc is NULL"); return ORBIT_ERR_NULL; }
  if (!valid_dtype(d->dtype)) { set_error("embed: bad dtype %d", (int)d->dtype); return ORBIT_ERR_DTYPE; }
  if (d->B <= 0 || d->V <= 0 || d->Hg <= 0 || d->Wg <= 0 || d->p <= 0 || d->D <= 0 || d->Hg % d->p || d->Wg % d->p ||
      d->D % 8 || (d->p != 1 && d->p != 2 && d->p != 4)) {
    set_error("embed: bad shape B=%d V=%d Hg=%d Wg=%d p=%d D=%d (need Hg%%p==0, Wg%%p==0, D%%8==0, p in {1,2,4})", d->B,
              d->V, d->Hg, d->Wg, d->p, d->D);
    return ORBIT_ERR_SHAPE;
  }
  return ORBIT_OK;
}

int orbit_tokenize(const orbit_embed_desc* d, const float* x, const void* Wp, const void* bp, void* tok, void* stream) {
  ORBIT_TRY(check_embed(d));
  if (!x || !Wp || !bp || !tok) { set_error("tokenize: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!aligned16(x) || !aligned16(Wp) || !aligned16(bp) || !aligned16(tok)) { set_error("tokenize: pointer not 16B aligned"); return ORBIT_ERR_ALIGN; }
  ORBIT_TRY(check_device());
  const size_t ntok = (size_t)d->B * (d->Hg / d->p) * (d->Wg / d->p) * d->V;
  ProfScope prof(PROF_FRONT, (double)ntok * d->D * dsize(d->dtype), (cudaStream_t)stream);     // a1 writes tok once
  if (g_force_simt != 1 && tokenize_tc_supported(*d)) return tokenize_fwd_tc(*d, x, Wp, bp, tok, (cudaStream_t)stream);
  return tokenize_fwd(*d, x, Wp, bp, tok, (cudaStream_t)stream);
}

size_t orbit_tokenize_bwd_workspace_bytes(const orbit_embed_desc* d) {
  if (!d) return 0;
  return align_up((size_t)d->V * (d->p * d->p + 1) * d->D * sizeof(float), 256);
}

int orbit_tokenize_bwd(const orbit_embed_desc* d, const float* x, const void* dtok, void* dWp, void* dbp, void* ws,
                       size_t ws_bytes, void* stream) {
  ORBIT_TRY(check_embed(d));
  if (!x || !dtok || !dWp || !dbp || !ws) { set_error("tokenize_bwd: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!aligned16(x) || !aligned16(dtok) || !aligned16(dWp) || !aligned16(dbp) || !aligned16(ws)) { set_error("tokenize_bwd: pointer not 16B aligned"); return ORBIT_ERR_ALIGN; }
  if (ws_bytes < orbit_tokenize_bwd_workspace_bytes(d)) { set_error("tokenize_bwd: workspace too small"); return ORBIT_ERR_WORKSPACE; }
  ORBIT_TRY(check_device());
  cudaStream_t s = (cudaStream_t)stream;
  const int P2 = d->p * d->p;
  float* accW = (float*)ws;
  float* accB = accW + (size_t)d->V * P2 * d->D;
  ORBIT_TRY(fill_zero(ws, (size_t)d->V * (P2 + 1) * d->D * sizeof(float), s));
  {
    const size_t ntok = (size_t)d->B * (d->Hg / d->p) * (d->Wg / d->p) * d->V;
    ProfScope prof(PROF_FRONT, (double)ntok * d->D * dsize(d->dtype), s);                       // a1' reads dtok once
    if (g_force_simt != 1 && tokenize_tc_supported(*d)) ORBIT_TRY(tokenize_bwd_acc_tc(*d, x, dtok, accW, accB, s));
    else ORBIT_TRY(tokenize_bwd_acc(*d, x, dtok, accW, accB, s));
  }
  ORBIT_TRY(cast_copy(accW, ORBIT_F32, dWp, d->dtype, (size_t)d->V * P2 * d->D, s));
  ORBIT_TRY(cast_copy(accB, ORBIT_F32, dbp, d->dtype, (size_t)d->V * d->D, s));
  return ORBIT_OK;
}

int orbit_profile_gemm(int on) { return prof_enable(on); }
int orbit_profile_gemm_collect(double* ms, double* flops, long long* launches) {
  return prof_collect(PROF_GEMM, ms, flops, launches);
}
int orbit_profile_collect(int category, double* ms, double* work, long long* launches) {
  if (category < 0 || category >= PROF_NCAT) { set_error("profile_collect: bad category %d", category); return ORBIT_ERR_SHAPE; }
  return prof_collect(category, ms, work, launches);
}

int orbit_debug_gemm(int M, int N, int K, orbit_dtype dtype, const void* A, long long a_rs, long long a_cs,
                     const void* B, long long b_rs, long long b_cs, float* C, void* stream) {
  if (!A || !B || !C) { set_error("debug_gemm: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!valid_dtype(dtype)) { set_error("debug_gemm: bad dtype"); return ORBIT_ERR_DTYPE; }
  if (M <= 0 || N <= 0 || K <= 0) { set_error("debug_gemm: bad shape"); return ORBIT_ERR_SHAPE; }
  ORBIT_TRY(check_device());
  GemmArgs g;
  g.A = A; g.a_rs = a_rs; g.a_cs = a_cs; g.B = B; g.b_rs = b_rs; g.b_cs = b_cs; g.C = C; g.ldc = N;
  g.M = M; g.N = N; g.K = K; g.in_dtype = dtype; g.out_dtype = ORBIT_F32;
  return gemm(g, (cudaStream_t)stream);
}

int orbit_debug_gemm_out(int M, int N, int K, orbit_dtype dtype, const void* A, long long a_rs, long long a_cs,
                         const void* B, long long b_rs, long long b_cs, orbit_dtype out_dtype, void* C, long long ldc,
                         const void* bias, void* stream) {
  if (!A || !B || !C) { set_error("debug_gemm_out: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!valid_dtype(dtype) || !valid_dtype(out_dtype)) { set_error("debug_gemm_out: bad dtype"); return ORBIT_ERR_DTYPE; }
  if (M <= 0 || N <= 0 || K <= 0 || ldc < N) { set_error("debug_gemm_out: bad shape"); return ORBIT_ERR_SHAPE; }
  ORBIT_TRY(check_device());
  GemmArgs g;
  g.A = A; g.a_rs = a_rs; g.a_cs = a_cs; g.B = B; g.b_rs = b_rs; g.b_cs = b_cs; g.C = C; g.ldc = ldc;
  g.M = M; g.N = N; g.K = K; g.in_dtype = dtype; g.out_dtype = out_dtype; g.bias = bias; g.bias_dtype = dtype;
  return gemm(g, (cudaStream_t)stream);
}

int orbit_debug_layernorm_fwd(int M, int D, orbit_dtype x_dtype, orbit_dtype p_dtype, orbit_dtype out_dtype, float eps,
                              const void* x, const void* gamma, const void* beta, void* out, float* mean, float* rstd,
                              void* stream) {
  if (!x || !gamma || !beta || !out || !mean || !rstd) { set_error("debug_layernorm_fwd: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!valid_dtype(x_dtype) || !valid_dtype(p_dtype) || !valid_dtype(out_dtype)) { set_error("debug_layernorm_fwd: bad dtype"); return ORBIT_ERR_DTYPE; }
  if (M <= 0 || D <= 0 || D % 8 || D > 65536) { set_error("debug_layernorm_fwd: bad shape M=%d D=%d (D <= 65536)", M, D); return ORBIT_ERR_SHAPE; }
  ORBIT_TRY(check_device());
  return layernorm_fwd(x, x_dtype, gamma, beta, p_dtype, out, out_dtype, mean, rstd, M, D, eps, nullptr, (cudaStream_t)stream);
}

int orbit_debug_layernorm_bwd(int M, int D, orbit_dtype dout_dtype, orbit_dtype x_dtype, orbit_dtype p_dtype,
                              orbit_dtype add_dtype, orbit_dtype out_dtype, const void* dout, const void* x,
                              const float* mean, const float* rstd, const void* gamma, const void* add, float* dx_f32,
                              void* dx_out, float* dgamma_acc, float* dbeta_acc, void* stream) {
  if (!dout || !x || !mean || !rstd || !gamma || !dgamma_acc || !dbeta_acc || (!dx_f32 && !dx_out)) {
    set_error("debug_layernorm_bwd: NULL pointer"); return ORBIT_ERR_NULL;
  }
  if (!valid_dtype(dout_dtype) || !valid_dtype(x_dtype) || !valid_dtype(p_dtype) || !valid_dtype(add_dtype) || !valid_dtype(out_dtype)) {
    set_error("debug_layernorm_bwd: bad dtype"); return ORBIT_ERR_DTYPE;
  }
  if (M <= 0 || D <= 0 || D % 8 || D > ORBIT_LN_MAX_D) { set_error("debug_layernorm_bwd: bad shape M=%d D=%d (D <= 16384)", M, D); return ORBIT_ERR_SHAPE; }
  ORBIT_TRY(check_device());
  return layernorm_bwd(dout, dout_dtype, x, x_dtype, mean, rstd, gamma, p_dtype, add, add_dtype, dx_f32, dx_out, out_dtype,
                       dgamma_acc, dbeta_acc, M, D, (cudaStream_t)stream);
}

int orbit_mse_loss_grad(orbit_dtype dtype, size_t n, const void* y, const void* t, void* dy, float* loss, void* stream) {
  if (!y || !t || !dy || !loss) { set_error("mse: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!valid_dtype(dtype)) { set_error("mse: bad dtype"); return ORBIT_ERR_DTYPE; }
  ORBIT_TRY(check_device());
  return mse_loss_grad(y, t, dtype, dy, loss, n, (cudaStream_t)stream);
}

// ------------------------------------------------------------------------------------------------------
// Eq. (2) / Eq. (3) chain
// ------------------------------------------------------------------------------------------------------
size_t orbit_chain_workspace_bytes(int m, int d, int n, int e, int T, orbit_dtype dtype) {
  if (T <= 0) return 0;
  size_t big = (size_t)(d > e ? d : e);
  return align_up((size_t)m * (n / T) * dsize(dtype), 256) + align_up((size_t)m * big * sizeof(float), 256);
}

static int chain_common(int m, int d, int n, int e, int T, orbit_dtype dtype, const void* in, const void* const* A_cols,
                        const void* const* B_rows, void* out, void* ws, size_t ws_bytes, void* stream, bool bwd) {
  if (!in || !A_cols || !B_rows || !out || !ws) { set_error("chain: NULL pointer"); return ORBIT_ERR_NULL; }
  if (!valid_dtype(dtype)) { set_error("chain: bad dtype"); return ORBIT_ERR_DTYPE; }
  if (m <= 0 || d <= 0 || n <= 0 || e <= 0 || T <= 0 || n % T) { set_error("chain: bad shape"); return ORBIT_ERR_SHAPE; }
  for (int k = 0; k < T; k++)
    if (!A_cols[k] || !B_rows[k]) { set_error("chain: NULL shard pointer"); return ORBIT_ERR_NULL; }
  if (ws_bytes < orbit_chain_workspace_bytes(m, d, n, e, T, dtype)) { set_error("chain: workspace too small"); return ORBIT_ERR_WORKSPACE; }
  ORBIT_TRY(check_device());
  cudaStream_t s = (cudaStream_t)stream;
  const int nk = n / T;
  void* tmp = ws;
  float* acc = (float*)((char*)ws + align_up((size_t)m * nk * dsize(dtype), 256));
  const int outw = bwd ? d : e;
  for (int k = 0; k < T; k++) {
    GemmArgs g1, g2;
    g1.in_dtype = g2.in_dtype = dtype;
    g1.M = m; g1.N = nk; g1.C = tmp; g1.ldc = nk; g1.out_dtype = dtype;
    g2.M = m; g2.K = nk; g2.A = tmp; g2.a_rs = nk; g2.a_cs = 1; g2.C = acc; g2.ldc = outw; g2.out_dtype = ORBIT_F32;
    g2.accumulate = k > 0; g2.N = outw;
    if (!bwd) {  // t = x A_k ; y += t B_k
      g1.K = d; g1.A = in; g1.a_rs = d; g1.a_cs = 1; g1.B = A_cols[k]; g1.b_rs = nk; g1.b_cs = 1;
      g2.B = B_rows[k]; g2.b_rs = e; g2.b_cs = 1;
    } else {     // t = dy B_k^T ; dx += t A_k^T
      g1.K = e; g1.A = in; g1.a_rs = e; g1.a_cs = 1; g1.B = B_rows[k]; g1.b_rs = 1; g1.b_cs = e;
      g2.B = A_cols[k]; g2.b_rs = 1; g2.b_cs = nk;
    }
    ORBIT_TRY(gemm(g1, s));
    ORBIT_TRY(gemm(g2, s));
  }
  return cast_copy(acc, ORBIT_F32, out, dtype, (size_t)m * outw, s);
}

int orbit_chain_fwd(int m, int d, int n, int e, int T, orbit_dtype dtype, const void* x, const void* const* A_cols,
                    const void* const* B_rows, void* y, void* ws, size_t ws_bytes, void* stream) {
  return chain_common(m, d, n, e, T, dtype, x, A_cols, B_rows, y, ws, ws_bytes, stream, false);
}
int orbit_chain_bwd(int m, int d, int n, int e, int T, orbit_dtype dtype, const void* dy, const void* const* A_cols,
                    const void* const* B_rows, void* dx, void* ws, size_t ws_bytes, void* stream) {
  return chain_common(m, d, n, e, T, dtype, dy, A_cols, B_rows, dx, ws, ws_bytes, stream, true);
}

}  // extern "C"
