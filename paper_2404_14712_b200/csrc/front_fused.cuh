// front_fused.cuh -- internal launchers of the fused pixel-space front end (front_fused.cu).
#pragma once
#include "common.cuh"

namespace orbit {

constexpr int FE_HP = 16;   // heads are padded to 16 in G / dG / dsT

bool fe_supported(int V, int p, int heads);
// Wpb[(r, v), :] = Wp[v, r, :] (r < p^2) | bp[v, :] (r = p^2); rows with v >= V are zero.  [R*Vp, D]
int fe_pack_wpb(const void* Wp, const void* bp, int dt, void* Wpb, int V, int Vp, int P2, int D, cudaStream_t s);
// G[r][a][v] = sum_d Wpb[(r, v), d] Ut[d, a]    (fp32 [R][FE_HP][Vp], v fastest: coalesced for fe_patch_fwd)
int fe_make_g(const void* Wpb, int dt, const float* Ut, float* G, int KVp, int Vp, int D, int h, cudaStream_t s);
// per patch: scores from pixels and G, softmax over V -> alpha [BL, h, Vp] fp32, A [BL, h, R*Vp] = alpha * pixext
int fe_patch_fwd(const float* x, const float* G, float* alpha, void* A, int dt, int V, int Vp, int Hg, int Wg, int p, int h,
                 int BL, cudaStream_t s);
// per patch: dalpha = <dA, pixext>, ds = alpha (dalpha - sum alpha dalpha) -> dsT [Vp][BL][FE_HP] fp32
int fe_patch_bwd(const float* x, const float* alpha, const void* dA, int dt, float* dsT, int V, int Vp, int Hg, int Wg, int p,
                 int h, int BL, cudaStream_t s);
// dG[(r, v), a] += sum_bl pixext[bl, v, r] dsT[v][bl][a]   (dG zeroed by the caller)
int fe_dg(const float* x, const float* dsT, float* dG, int B, int V, int Vp, int Hg, int Wg, int p, cudaStream_t s);
// dUt[d, a] += sum_k Wpb[k, d] dG[k, a]                    (dUt zeroed by the caller)
int fe_dut(const void* Wpb, int dt, const float* dG, float* dUt, int KVp, int D, int h, cudaStream_t s);
// dWp[v, r, :] / dbp[v, :] = accW[(r, v), :] + sum_a dG[(r, v), a] Ut[:, a]
int fe_finish_dwp(const float* accW, const float* dG, const float* Ut, void* dWp, void* dbp, int dt, int V, int Vp, int P2,
                  int D, int h, cudaStream_t s);

}  // namespace orbit
