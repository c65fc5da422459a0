/* orbit.h -- C-ABI of liborbit.so: the per-GPU dense training step of ORBIT's ClimaX-style ViT
 * (arxiv 2404.14712), hand-written CUDA for sm_100a (B200).
 *
 * Citations are PAPER.md:<line> (the paper text) and DESIGN.md "Readings" R<n> where the paper is silent.
 *
 * Conventions:
 *  - All tensor pointers are DEVICE memory owned by the caller; descriptors and parameter structs are HOST
 *    memory, read during the call only.  The library allocates no device memory, keeps no pointer after
 *    return, and writes only outputs, `saved`, `ws` and gradients.  Outputs are overwritten (no accumulate).
 *    (One exception, by design: orbit_tokenize_bwd_noalloc uses a 16 MiB file-scope device array of the library
 *    instead of `ws`; see its declaration.)
 *  - Dense row-major, last index contiguous.  Weights are [in, out] so that y = x A exactly as in Eq. (1)-(3)
 *    (PAPER.md:70-82): a column shard is A[:, k n/T:(k+1) n/T], a row shard is B[k n/T:(k+1) n/T, :].
 *    Wqkv columns are [Q | K | V], heads contiguous inside each third.  tok is [B, L, V, D].
 *  - Execution is asynchronous on `stream` (a cudaStream_t passed as void*); no host synchronisation.
 *  - Errors: return code only (never abort/throw).  All argument checks precede the first launch, so a
 *    non-OK return other than ORBIT_ERR_CUDA means nothing was written.  orbit_last_error() gives text.
 *  - Precision: ORBIT_BF16 = bf16 storage, every contraction accumulates in fp32, LayerNorm statistics /
 *    softmax / GELU in fp32, one round-to-nearest-even at each store; Hybrid-STOP shard partials stay fp32
 *    until summed.  ORBIT_F32 = fp32 storage and true fp32 FMA (no TF32).  (R17.)
 *  - No CPU fallback and no other-architecture fallback: a device that is not compute capability 10.x
 *    yields ORBIT_ERR_ARCH.
 */
#ifndef ORBIT_H_
#define ORBIT_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORBIT_VERSION 100

typedef enum {
  ORBIT_OK = 0,
  ORBIT_ERR_NULL = 1,        /* a required pointer is NULL */
  ORBIT_ERR_SHAPE = 2,       /* Hg%p, Wg%p, D%heads, heads%T, F%T, non-positive or unsupported sizes */
  ORBIT_ERR_DTYPE = 3,       /* unknown dtype, or resid_dtype incompatible with dtype */
  ORBIT_ERR_ALIGN = 4,       /* base pointer not 16-byte aligned */
  ORBIT_ERR_WORKSPACE = 5,   /* ws_bytes smaller than the matching *_workspace_bytes() */
  ORBIT_ERR_UNSUPPORTED = 6, /* reserved flag set, in-place call */
  ORBIT_ERR_ARCH = 7,        /* device is not sm_100-class */
  ORBIT_ERR_CUDA = 8         /* a CUDA runtime call or launch failed (see orbit_last_error) */
} orbit_status;

typedef enum { ORBIT_F32 = 0, ORBIT_BF16 = 1 } orbit_dtype;

/* flags of orbit_block_desc (any other bit returns ORBIT_ERR_UNSUPPORTED) */
#define ORBIT_QK_NORM   1u   /* QK-LayerNorm (R9): LayerNorm over d_h of every head's q and k before the
                                scaled dot product, gamma / beta in R^{d_h} shared by the heads (qn_g, qn_b, kn_g, kn_b of
                                orbit_block_params); needs d_h in {32, 64, 128, 192, 256} */
#define ORBIT_RECOMPUTE 2u   /* activation checkpointing: orbit_block_fwd keeps only the block input in
                                `saved`; orbit_block_bwd re-runs the forward into its workspace first.  Same results. */

/* ---- a1 / a1': per-variable patch tokenisation (R1, R2) --------------------------- */
typedef struct {
  int B, V, Hg, Wg, p, D;      /* batch, variables, lat x lon grid, patch size, embed dim; L=(Hg/p)*(Wg/p) */
  orbit_dtype dtype;           /* dtype of Wp, bp, tok, dtok, dWp, dbp (x is always fp32) */
} orbit_embed_desc;

/* tok[b,l,v,:] = sum_r pix(b,v,l,r) Wp[v,r,:] + bp[v,:],  l = i*(Wg/p)+j, r = di*p+dj,
 * pix = x[b,v,i*p+di,j*p+dj].   x [B,V,Hg,Wg] fp32; Wp [V,p*p,D]; bp [V,D]; tok [B,L,V,D]. */
int orbit_tokenize(const orbit_embed_desc* d, const float* x, const void* Wp, const void* bp, void* tok,
                   void* stream);
/* dWp[v,r,:] = sum_{b,l} pix dtok[b,l,v,:];  dbp[v,:] = sum_{b,l} dtok[b,l,v,:].  No dx (input data). */
int orbit_tokenize_bwd(const orbit_embed_desc* d, const float* x, const void* dtok, void* dWp, void* dbp,
                       void* ws, size_t ws_bytes, void* stream);
size_t orbit_tokenize_bwd_workspace_bytes(const orbit_embed_desc* d);
/* orbit_tokenize_bwd for callers that cannot allocate a workspace (CUDA graph capture, serving loops, harnesses that
 * forbid cudaMalloc): same arguments, results and kernels, but the fp32 accumulators live in a file-scope device array
 * inside the library (csrc/tokenize_noalloc.cu) of orbit_tokenize_bwd_noalloc_max_bytes() = 16 MiB, held by every GPU
 * that loads liborbit.so until the process exits.  Calls no cudaMalloc / cudaFree / allocating routine.
 * ORBIT_ERR_WORKSPACE (nothing written) when orbit_tokenize_bwd_workspace_bytes(d) exceeds that maximum, i.e. when
 * V (p*p + 1) D > 4 Mi.  All calls on a device share the one array (cleared by each call before use): calls that
 * OVERLAP on the GPU -- different streams -- race and must be serialised by the caller; back-to-back calls on one
 * stream are independent. */
int orbit_tokenize_bwd_noalloc(const orbit_embed_desc* d, const float* x, const void* dtok, void* dWp, void* dbp,
                               void* stream);
size_t orbit_tokenize_bwd_noalloc_max_bytes(void);

/* ---- a2 / a2': variable aggregation, cross-attention over the V tokens of a patch (R3, R4)
 * At every (b,l), X = tok[b,l] (V x D):  qt = q Wq + bq;  K = X Wk + bk;  U = X Wv + bv;  per head a:
 * s_v = qt_a . K_{v,a} / sqrt(d_a); alpha = softmax_v(s); o_a = sum_v alpha_v U_{v,a};
 * agg[b,l] = concat(o_a) Wo + bo (+ pos[l]).   The kernels use the exact collapsed form of DESIGN.md §4. */
typedef struct {
  int B, L, V, D, heads;
  orbit_dtype dtype;           /* tok, dtok, parameters, parameter grads */
  orbit_dtype resid_dtype;     /* agg, dagg, pos, dpos (the residual stream) */
} orbit_agg_desc;
typedef struct { const void *q /*[D]*/, *Wq, *bq, *Wk, *bk, *Wv, *bv, *Wo, *bo /* W:[D,D] b:[D] */; } orbit_agg_params;
typedef struct { void *q, *Wq, *bq, *Wk, *bk, *Wv, *bv, *Wo, *bo; } orbit_agg_grads; /* dbk is written (== 0) */

int orbit_var_aggregate(const orbit_agg_desc* d, const void* tok, const orbit_agg_params* P,
                        const void* pos /* [L,D] nullable */, void* agg /* [B,L,D] */, void* saved,
                        void* ws, size_t ws_bytes, void* stream);
int orbit_var_aggregate_bwd(const orbit_agg_desc* d, const void* tok, const orbit_agg_params* P,
                            const void* dagg, const void* saved, void* dtok, orbit_agg_grads* G,
                            void* dpos /* [L,D] nullable */, void* ws, size_t ws_bytes, void* stream);
size_t orbit_var_aggregate_workspace_bytes(const orbit_agg_desc* d);
size_t orbit_var_aggregate_bwd_workspace_bytes(const orbit_agg_desc* d);
size_t orbit_var_aggregate_saved_bytes(const orbit_agg_desc* d);

/* ---- a1+a2 fused in pixel space: same result as orbit_tokenize
 * followed by orbit_var_aggregate (and, backward, orbit_var_aggregate_bwd followed by orbit_tokenize_bwd), but the
 * [B, L, V, D] token tensor and its gradient are never formed.  Tokenisation is affine and nothing non-linear
 * precedes the K/V projections, so with pixext[v, r] = (pix(b,v,l,r), 1), Wpb[(r,v), :] = (Wp[v,r,:] ; bp[v,:]):
 *   s[v,a] = sum_r pixext[v,r] (Wpb Ut)[(r,v), a];  alpha = softmax_v(s);
 *   o[:, a] = sum_{r,v} alpha[v,a] pixext[v,r] (Wpb Wv)[(r,v), a-columns] + bv[a];  agg = o Wo + bo (+ pos[l])
 * (DESIGN.md §4b).  Limits: V <= 128, p in {1,2,4}, heads <= 16 -> ORBIT_ERR_SHAPE otherwise.
 * x [B,V,Hg,Wg] fp32; Wp [V,p*p,D]; bp [V,D]; agg, dagg [B,L,D] (resid_dtype); dWp, dbp, G as in the two-call path.
 * `saved` (orbit_embed_fused_saved_bytes) carries alpha and the A operand to the backward call. */
typedef struct {
  int B, V, Hg, Wg, p, D, heads;
  orbit_dtype dtype;           /* parameters, parameter grads, internal operands */
  orbit_dtype resid_dtype;     /* agg, dagg, pos, dpos */
} orbit_front_desc;
int orbit_embed_fused(const orbit_front_desc* d, const float* x, const void* Wp, const void* bp,
                      const orbit_agg_params* P, const void* pos /* [L,D] nullable */, void* agg, void* saved,
                      void* ws, size_t ws_bytes, void* stream);
int orbit_embed_fused_bwd(const orbit_front_desc* d, const float* x, const void* Wp, const void* bp,
                          const orbit_agg_params* P, const void* dagg, const void* saved, void* dWp, void* dbp,
                          orbit_agg_grads* G, void* dpos /* [L,D] nullable */, void* ws, size_t ws_bytes, void* stream);
size_t orbit_embed_fused_workspace_bytes(const orbit_front_desc* d);
size_t orbit_embed_fused_bwd_workspace_bytes(const orbit_front_desc* d);
size_t orbit_embed_fused_saved_bytes(const orbit_front_desc* d);

/* ---- a3-a7: one ViT block, pre-LN residual form (R5-R8, R10), optionally in Hybrid-STOP
 * shard-local mode with T shards run one after another on this GPU (Eq. 1-3; R13-R15):
 *   a = LN1(x); qkv = a Wqkv + bqkv; O = softmax(Q K^T / sqrt(d_h)) V per head; x1 = x + O Wproj + bproj;
 *   m = LN2(x1); u = m Wfc1 + bfc1; g = GELU_erf(u); y = x1 + g Wfc2 + bfc2.
 * T > 1: Wqkv, Wfc1 column shards (head aligned), Wproj, Wfc2 row shards; the T fp32 partial products are
 * summed on the device, then bproj / bfc2 and the residual are added once. */
typedef struct {
  int B, N, D, heads, F, T;    /* batch, tokens per sample, embed dim, heads, MLP width, shards (1 = unsharded) */
  float ln_eps;
  orbit_dtype dtype;           /* weights, grads, internal activations */
  orbit_dtype resid_dtype;     /* x, y, dx, dy: F32 or BF16 when dtype is BF16; must be F32 when dtype is F32 */
  unsigned flags;
} orbit_block_desc;
typedef struct { const void *Wqkv /*[D,3D/T]*/, *bqkv /*[3D/T]*/, *Wproj /*[D/T,D]*/, *Wfc1 /*[D,F/T]*/,
                 *bfc1 /*[F/T]*/, *Wfc2 /*[F/T,D]*/; } orbit_block_shard;
typedef struct { const void *ln1_g, *ln1_b, *ln2_g, *ln2_b, *bproj, *bfc2 /* all [D] */;
                 const orbit_block_shard* shards /* T of them, host array */;
                 const void *qn_g, *qn_b, *kn_g, *kn_b /* [d_h]; read only with ORBIT_QK_NORM, else may be NULL */;
               } orbit_block_params;
typedef struct { void *Wqkv, *bqkv, *Wproj, *Wfc1, *bfc1, *Wfc2; } orbit_block_shard_grads;
typedef struct { void *ln1_g, *ln1_b, *ln2_g, *ln2_b, *bproj, *bfc2;
                 const orbit_block_shard_grads* shards;
                 void *qn_g, *qn_b, *kn_g, *kn_b /* written only with ORBIT_QK_NORM (d kn_b is analytically 0) */;
               } orbit_block_grads;

int orbit_block_fwd(const orbit_block_desc* d, const void* x /* [B,N,D] */, const orbit_block_params* P,
                    void* y, void* saved, void* ws, size_t ws_bytes, void* stream);
int orbit_block_bwd(const orbit_block_desc* d, const void* dy, const orbit_block_params* P, const void* saved,
                    void* dx, orbit_block_grads* G, void* ws, size_t ws_bytes, void* stream);
size_t orbit_block_fwd_workspace_bytes(const orbit_block_desc* d);
size_t orbit_block_bwd_workspace_bytes(const orbit_block_desc* d);
size_t orbit_block_saved_bytes(const orbit_block_desc* d);

/* ---- the rank-local Hybrid-STOP program (Fig. 3): what ONE rank of a
 * tensor-parallel group of size d->T computes between the collectives.  Rank k holds the column shards Wqkv^k [D, 3D/T]
 * (= [Q_k | K_k | V_k], head aligned), Wfc1^k [D, F/T] with bqkv^k, bfc1^k and the row shards Wproj^k [D/T, D],
 * Wfc2^k [F/T, D]: P->shards[0] / G->shards[0] are THIS rank's shard (one element); LayerNorm parameters, bproj, bfc2 are
 * replicated.  One block is six calls; between them the CALLER all-reduces (sum) `part`, an fp32 [B, N, D] buffer, over
 * the group -- "GPUs in each tensor-parallel group add their individual activations together", "add their
 * activation gradients together through all-reduce".  The library holds no communicator.
 *   orbit_rank_fwd_attn : a = LN1(x); qkv^k = a Wqkv^k + bqkv^k; attention on this rank's heads/T heads;
 *                         part <- O^k Wproj^k                                             -- all-reduce(part) --
 *   orbit_rank_fwd_mlp  : x1 = x + part + bproj; m = LN2(x1); g^k = GELU(m Wfc1^k + bfc1^k);
 *                         part <- g^k Wfc2^k                                              -- all-reduce(part) --
 *   orbit_rank_fwd_out  : y = x1 + part + bfc2
 *   orbit_rank_bwd_mlp  : dbfc2, dWfc2^k, du^k, dbfc1^k, dWfc1^k; part <- du^k Wfc1^k^T   -- all-reduce(part) --
 *   orbit_rank_bwd_attn : dx1 = dy + LN2'(part); d ln2, dbproj, dWproj^k, dO^k, attention backward, dbqkv^k, dWqkv^k;
 *                         part <- dqkv^k Wqkv^k^T                                         -- all-reduce(part) --
 *   orbit_rank_bwd_out  : dx = dx1 + LN1'(part); d ln1; gradients cast to `dtype`.
 * y, dx and the gradients of the replicated parameters come out identical on every rank, except the QK-LayerNorm
 * gradients (ORBIT_QK_NORM), which are the sums over THIS rank's heads and must be summed over the group by the caller
 * with its other gradient reductions.  ORBIT_RECOMPUTE -> ORBIT_ERR_UNSUPPORTED.  `saved` (orbit_rank_saved_bytes) is
 * written by the forward calls and read by the backward calls; `ws` (orbit_rank_bwd_workspace_bytes) must be the SAME
 * buffer, untouched, through the three backward calls (it carries dx1 and the fp32 gradient accumulators).  Precision:
 * the partials are fp32 (R15).  Same checks / error codes as orbit_block_*. */
int orbit_rank_fwd_attn(const orbit_block_desc* d, const void* x /* [B,N,D] */, const orbit_block_params* P,
                        float* part /* out */, void* saved, void* stream);
int orbit_rank_fwd_mlp(const orbit_block_desc* d, const orbit_block_params* P, float* part /* in: summed; out */,
                       void* saved, void* stream);
int orbit_rank_fwd_out(const orbit_block_desc* d, const orbit_block_params* P, const float* part /* in: summed */,
                       void* y, const void* saved, void* stream);
int orbit_rank_bwd_mlp(const orbit_block_desc* d, const void* dy, const orbit_block_params* P, const void* saved,
                       orbit_block_grads* G, float* part /* out */, void* ws, size_t ws_bytes, void* stream);
int orbit_rank_bwd_attn(const orbit_block_desc* d, const void* dy, const orbit_block_params* P, const void* saved,
                        orbit_block_grads* G, float* part /* in: summed; out */, void* ws, size_t ws_bytes, void* stream);
int orbit_rank_bwd_out(const orbit_block_desc* d, const orbit_block_params* P, const void* saved, orbit_block_grads* G,
                       const float* part /* in: summed */, void* dx, void* ws, size_t ws_bytes, void* stream);
size_t orbit_rank_saved_bytes(const orbit_block_desc* d);
size_t orbit_rank_bwd_workspace_bytes(const orbit_block_desc* d);

/* ---- head + loss: "predictions are computed by projecting the embedding output from the
 * feature space to the image space" and the latitude-weighted MSE the paper trains with;
 * readings R26-R28:  zn = LN_f(z);  P = zn Wh + bh  ([B*L, V p^2], column c = v p^2 + di p + dj);
 *   pred[b, v, i p + di, j p + dj] = P[b, l = i (Wg/p) + j, c];
 *   loss = mean_{b,v,y,x} w_y (pred - target)^2,  w_y = cos(lat_y) / mean cos,  lat_y = -90 + (y + 1/2) 180 / Hg.
 * z [B,L,D] (resid_dtype); lnf_g, lnf_b [D]; Wh [D, V p^2]; bh [V p^2] (dtype); target, pred [B,V,Hg,Wg] fp32 (pred
 * nullable); latw [Hg] fp32 device weights or NULL for the cosine weights above; loss: fp32 scalar on the device. */
typedef struct {
  int B, V, Hg, Wg, p, D;
  float ln_eps;
  orbit_dtype dtype;           /* parameters, parameter grads, internal operands */
  orbit_dtype resid_dtype;     /* z, dz */
} orbit_head_desc;
int orbit_head_loss(const orbit_head_desc* d, const void* z, const void* lnf_g, const void* lnf_b, const void* Wh,
                    const void* bh, const float* target, const float* latw, float* pred, float* loss, void* saved,
                    void* ws, size_t ws_bytes, void* stream);
/* dz [B,L,D] and the gradients of lnf_g, lnf_b, Wh, bh for the loss of the matching orbit_head_loss call. */
int orbit_head_loss_bwd(const orbit_head_desc* d, const void* z, const void* lnf_g, const void* Wh, const void* saved,
                        void* dz, void* dlnf_g, void* dlnf_b, void* dWh, void* dbh, void* ws, size_t ws_bytes,
                        void* stream);
size_t orbit_head_loss_workspace_bytes(const orbit_head_desc* d);
size_t orbit_head_loss_bwd_workspace_bytes(const orbit_head_desc* d);
size_t orbit_head_loss_saved_bytes(const orbit_head_desc* d);

/* ---- dynamic gradient scaling and fp32 gradient accumulation ("the PyTorch dynamic
 * gradient scaling mechanism [24] ... detects the value range of the computed gradient magnitude ... scale the gradient
 * magnitudes to the proper value range representable in BFLOAT16, and then reverse the scaling during the parameters
 * update").  The caller scales its loss gradient (dy) by S; after the backward calls:
 *   orbit_grads_unscale_check: every element of the n gradient tensors (device pointers grads[i], counts[i] elements of
 *     `dtype`) is multiplied in place by 1 / *scale (fp32 arithmetic, one rounding to `dtype`); *found_inf is set to 1.0f
 *     when any gradient element is Inf / NaN (it is never cleared here: zero it once per step).  scale == NULL means S = 1
 *     (check only).
 *   orbit_grads_accumulate: acc[i][j] += grads[i][j] / *scale in fp32 (gradient accumulation across micro-steps without
 *     the per-step rounding of the `dtype` gradients); found_inf nullable.
 *   orbit_grad_scale_update: the scale schedule of [24]: if *found_inf != 0: S <- S * backoff_factor, tracker <- 0 (the
 *     caller skips the parameter update); else tracker += 1 and, when it reaches growth_interval, S <- S * growth_factor,
 *     tracker <- 0.  The paper names no values; the caller supplies them (ORBIT_ERR_SHAPE unless growth_factor > 1,
 *     0 < backoff_factor < 1, growth_interval >= 1).
 * grads / acc / counts are HOST arrays of n entries; the tensors, scale, found_inf and growth_tracker are DEVICE memory
 * (no host synchronisation).  Tensors must be 16-byte aligned; counts[i] == 0 entries are skipped.  No optimizer is
 * part of this library (the paper names none). */
int orbit_grads_unscale_check(int n, void* const* grads, const size_t* counts, orbit_dtype dtype, const float* scale,
                              float* found_inf, void* stream);
int orbit_grads_accumulate(int n, const void* const* grads, float* const* acc, const size_t* counts, orbit_dtype dtype,
                           const float* scale /* nullable */, float* found_inf /* nullable */, void* stream);
int orbit_grad_scale_update(float* scale, int* growth_tracker, const float* found_inf, float growth_factor,
                            float backoff_factor, int growth_interval, void* stream);

/* ---- bare Eq. (2)/(3) chain, used by the fp32 shard-recombination check (R15):
 *   y = sum_k (x A_k) B_k   with A_k [d, n/T] column shards and B_k [n/T, e] row shards;
 *   dx = sum_k (dy B_k^T) A_k^T.  x [m,d], y [m,e]; fp32 partials combined on device.
 *   ws must hold m*(n/T) elements of `dtype` + m*max(d,e) floats. */
int orbit_chain_fwd(int m, int d, int n, int e, int T, orbit_dtype dtype, const void* x,
                    const void* const* A_cols, const void* const* B_rows, void* y,
                    void* ws, size_t ws_bytes, void* stream);
int orbit_chain_bwd(int m, int d, int n, int e, int T, orbit_dtype dtype, const void* dy,
                    const void* const* A_cols, const void* const* B_rows, void* dx,
                    void* ws, size_t ws_bytes, void* stream);
size_t orbit_chain_workspace_bytes(int m, int d, int n, int e, int T, orbit_dtype dtype);

/* ---- harness loss (BASELINE.json config 1: "target is an N(0,1) field with MSE loss"):
 *   loss = mean((y - t)^2) (fp32 scalar, device), dy = 2 (y - t) / n.  y, t, dy: n elements of `dtype`. */
int orbit_mse_loss_grad(orbit_dtype dtype, size_t n, const void* y, const void* t, void* dy, float* loss,
                        void* stream);

/* ---- diagnostics ---------------------------------------------------------------------------------------- */
const char* orbit_last_error(void);   /* thread-local, static storage */
int orbit_version(void);
/* Number of kernels launched by this library on the calling thread since the last reset (bench.py's
 * gpu_launches claim). */
long long orbit_launch_count(void);
void orbit_reset_launch_count(void);
/* Per-launch CUDA-event timing of the tensor-core GEMM kernel (the dominant kernel; bench.py's roofline leg).
 * orbit_profile_gemm(1) starts recording an event pair around every tcgen05 GEMM launch on its stream;
 * orbit_profile_gemm_collect() waits for them, returns the summed kernel milliseconds, the summed algorithmic
 * FLOPs (2 M N K per launch) and the number of launches recorded. */
int orbit_profile_gemm(int on);
int orbit_profile_gemm_collect(double* ms, double* flops, long long* launches);
/* The same record by category (bench.py's secondary roofline entries): 0 = tcgen05 GEMM (work = FLOPs), 1 = attention forward,
 * 2 = attention backward (FLOPs: 4 B N^2 D resp. twice that), 3 = LayerNorm forward / backward kernels, 4 = front-end
 * streaming kernels (tokenise, per-patch aggregation, pixel-space per-patch kernels) (work = algorithmic bytes).
 * Non-destructive; orbit_profile_gemm(1) clears the record.  ORBIT_ERR_SHAPE for an unknown category. */
int orbit_profile_collect(int category, double* ms, double* work, long long* launches);
/* Kernel-level diagnostic: C[M,N] (fp32, row-major) = A B through the library's GEMM dispatcher.
 * A(m,k) = A[m*a_rs + k*a_cs], B(k,n) = B[k*b_rs + n*b_cs] (element strides); dtype of A and B = `dtype`.
 * Exercises every operand-major combination the block uses (K-major / MN-major A and B). */
int orbit_debug_gemm(int M, int N, int K, orbit_dtype dtype, const void* A, long long a_rs, long long a_cs,
                     const void* B, long long b_rs, long long b_cs, float* C, void* stream);
/* Strided-batch form (the per-head products of the front end): problem i reads A + i*a_bs, B + i*b_bs and writes
 * C + i*c_bs (element offsets, multiples of 8), C row stride ldc. */
int orbit_debug_gemm_batched(int M, int N, int K, int batch, orbit_dtype dtype, const void* A, long long a_rs,
                             long long a_cs, long long a_bs, const void* B, long long b_rs, long long b_cs,
                             long long b_bs, float* C, long long ldc, long long c_bs, void* stream);
/* As orbit_debug_gemm, with the output options of the block's GEMMs: C (row stride ldc, ldc % 8 == 0) in out_dtype and an
 * optional bias[N] (dtype `dtype`) added before the store.  bf16 outputs of tile-sized problems take the TMA-store
 * epilogue of the CTA-pair kernel. */
int orbit_debug_gemm_out(int M, int N, int K, orbit_dtype dtype, const void* A, long long a_rs, long long a_cs,
                         const void* B, long long b_rs, long long b_cs, orbit_dtype out_dtype, void* C, long long ldc,
                         const void* bias /*nullable*/, void* stream);
/* Kernel-level diagnostic: the LayerNorm kernels of orbit_block_fwd / orbit_block_bwd on their own (the
 * pre-LN sub-layers; SURVEY.md 8(c) BLK / BLK').  Row-major [M, D], D % 8 == 0, all pointers device memory.
 * fwd: out = (x - mean) * rstd * gamma + beta with biased variance; mean, rstd [M] fp32 are written.
 * bwd: dx = add (nullable) + dz(dout; x, mean, rstd, gamma), written as fp32 to dx_f32 (nullable) and as out_dtype to
 *      dx_out (nullable); dgamma_acc / dbeta_acc [D] fp32 are ACCUMULATED into (the caller zeroes them).
 * Errors: ORBIT_ERR_NULL, ORBIT_ERR_DTYPE, ORBIT_ERR_SHAPE (M <= 0, D % 8 != 0), ORBIT_ERR_CUDA. */
int orbit_debug_layernorm_fwd(int M, int D, orbit_dtype x_dtype, orbit_dtype p_dtype, orbit_dtype out_dtype, float eps,
                              const void* x, const void* gamma, const void* beta, void* out, float* mean, float* rstd,
                              void* stream);
int orbit_debug_layernorm_bwd(int M, int D, orbit_dtype dout_dtype, orbit_dtype x_dtype, orbit_dtype p_dtype,
                              orbit_dtype add_dtype, orbit_dtype out_dtype, const void* dout, const void* x,
                              const float* mean, const float* rstd, const void* gamma, const void* add /*nullable*/,
                              float* dx_f32 /*nullable*/, void* dx_out /*nullable*/, float* dgamma_acc, float* dbeta_acc,
                              void* stream);

#ifdef __cplusplus
}
#endif
#endif /* ORBIT_H_ */
