"""fp64 CPU oracle of the ORBIT per-GPU training step -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It shares no code with paper_2404_14712_b200/ (the CUDA path) and imports nothing but
numpy.  Every function is the plain definition written out in float64, in the paper's order and
notation; numpy `@` (a library matmul) is the only primitive used as a step.  No blocking, fusion or
algebraic reformulation: in particular the variable aggregation forms the K/V projections of every
variable token explicitly (the CUDA path uses a collapsed form -- that is the thing being checked).

Citations are `PAPER.md:<line>` and SURVEY.md §8(c) readings (listed in
DESIGN.md "Readings").  Where the paper is silent the reading is named.

Parity pins (tests/test_oracle_pins.py, all `-m "not gpu"`): central finite differences for every
fwd/bwd pair; softmax rows sum to 1 / shift invariance; LayerNorm zero-mean unit-variance; attention
over identical keys = mean of values; Eq. (2)/(3) shard sums = unsharded product; tokeniser = strided
convolution (torch conv2d, float64); whole block fwd+bwd = torch float64 autograd of textbook ops;
aggregation V=1 closed form, permutation invariance, dbk == 0, dbv == sum(do); patch-chunked front end
(tokenize_patches / var_aggregate / var_aggregate_bwd / tokenize_bwd_patches over a partition of the patches) = the
whole-tensor functions; QK-LayerNorm: torch
float64 autograd with F.layer_norm on the per-head q / k, finite differences, logits bounded by
sqrt(d_h) for gamma = 1, beta = 0, invariance to rescaling the pre-norm queries (eps = 0); head + wMSE: torch
float64 autograd (layer_norm, linear, permute, weighted mean), finite differences, unpatchify = inverse of
`patches`, weights with mean 1 / equator-symmetric / uniform weights = plain MSE, sum_i cos closed form.
Gradient scaling (grads_unscale_check / grads_accumulate / grad_scale_update): torch's own CPU implementation of the
mechanism the paper cites (torch._amp_foreach_non_finite_check_and_unscale_, torch._amp_update_scale_), exact
power-of-two closed forms, and a hand-worked schedule trace (tests/golden/grad_scale_trace.json).
Rank-local Hybrid-STOP program (rank_block_fwd / rank_block_bwd): world-size-2 gloo run with a real all-reduce
= the unsharded block (tests/test_multiproc.py), and a plain-sum run for T in {1, 2, 4} (tests/test_oracle_pins.py).
Parity unpinned: none.

Layout conventions (same as include/orbit.h): row-major, weights [in, out] so y = x A exactly as in
Eq. (1)-(3); Wqkv columns [Q | K | V], heads contiguous inside each third;
tok[B, L, V, D]; patches row-major over the grid, pixels row-major inside a patch.
"""
from __future__ import annotations

import math
import numpy as np

F64 = np.float64


def _f64(a):
    return np.asarray(a, dtype=F64)


# ---------------------------------------------------------------------------------------------
# elementary functions
# ---------------------------------------------------------------------------------------------
_erf = np.vectorize(math.erf, otypes=[F64])


def erf(u):
    """libm erf, elementwise (SURVEY.md §8(c) pin table: 'GELU ... libm erf')."""
    u = _f64(u)
    try:  # scipy's erf is the same libm-quality function, vectorised; fall back to math.erf
        from scipy.special import erf as _serf
        return _serf(u)
    except Exception:  # pragma: no cover
        return _erf(u)


def gelu(u):
    """GELU(u) = u * Phi(u) = 0.5 u (1 + erf(u / sqrt 2)).  PAPER.md:88 "GeLU (xA) B"; exact erf
    form (reading 7)."""
    u = _f64(u)
    return 0.5 * u * (1.0 + erf(u / math.sqrt(2.0)))


def gelu_grad(u):
    """d GELU / du = Phi(u) + u phi(u), Phi/phi the standard normal cdf/pdf."""
    u = _f64(u)
    Phi = 0.5 * (1.0 + erf(u / math.sqrt(2.0)))
    phi = np.exp(-0.5 * u * u) / math.sqrt(2.0 * math.pi)
    return Phi + u * phi


def softmax_lastdim(s):
    """softmax over the last axis with max subtraction (PAPER.md:88 softmax(QK^T)V)."""
    s = _f64(s)
    e = np.exp(s - s.max(axis=-1, keepdims=True))
    return e / e.sum(axis=-1, keepdims=True)


def layernorm(z, gamma, beta, eps):
    """LN(z)_i = gamma_i (z_i - mu) / sqrt(var + eps) + beta_i, mu and *biased* var over the last
    axis (reading 6).  Returns (out, zhat, rstd)."""
    z = _f64(z)
    mu = z.mean(axis=-1, keepdims=True)
    var = ((z - mu) ** 2).mean(axis=-1, keepdims=True)
    rstd = 1.0 / np.sqrt(var + eps)
    zhat = (z - mu) * rstd
    return zhat * _f64(gamma) + _f64(beta), zhat, rstd


def layernorm_bwd(dout, zhat, rstd, gamma):
    """Given d(out): dgamma = sum_rows dout*zhat; dbeta = sum_rows dout;
    dz = (ghat - mean(ghat) - zhat * mean(ghat*zhat)) * rstd with ghat = dout*gamma."""
    dout = _f64(dout)
    D = dout.shape[-1]
    flat = dout.reshape(-1, D)
    dgamma = (flat * zhat.reshape(-1, D)).sum(axis=0)
    dbeta = flat.sum(axis=0)
    ghat = dout * _f64(gamma)
    dz = (ghat - ghat.mean(axis=-1, keepdims=True)
          - zhat * (ghat * zhat).mean(axis=-1, keepdims=True)) * rstd
    return dz, dgamma, dbeta


# ---------------------------------------------------------------------------------------------
# TOK -- per-variable patch tokenisation ("independent patch tokenization for each
# channel input"; PAPER.md:155 sample shape; reading 1)
# ---------------------------------------------------------------------------------------------
def patches(x, p):
    """pix[b, v, l, r] = x[b, v, i*p+di, j*p+dj], l = i*(Wg/p)+j, r = di*p+dj."""
    x = _f64(x)
    B, V, Hg, Wg = x.shape
    gh, gw = Hg // p, Wg // p
    pix = x.reshape(B, V, gh, p, gw, p).transpose(0, 1, 2, 4, 3, 5)   # b v i j di dj
    return pix.reshape(B, V, gh * gw, p * p)


def tokenize(x, Wp, bp, p):
    """tok[b, l, v, :] = sum_r pix(b, v, l, r) Wp[v, r, :] + bp[v, :].   -> [B, L, V, D]"""
    pix = patches(x, p)                                             # [B, V, L, p^2]
    Wp, bp = _f64(Wp), _f64(bp)
    B, V, L, _ = pix.shape
    D = Wp.shape[2]
    tok = np.empty((B, L, V, D), dtype=F64)
    for v in range(V):                                              # independent per channel
        tok[:, :, v, :] = pix[:, v] @ Wp[v] + bp[v]
    return tok


def tokenize_bwd(x, dtok, p):
    """dWp[v, r, :] = sum_{b,l} pix(b,v,l,r) dtok[b,l,v,:];  dbp[v, :] = sum_{b,l} dtok[b,l,v,:].
    No dx (x is input data)."""
    pix = patches(x, p)
    dtok = _f64(dtok)
    B, V, L, P2 = pix.shape
    D = dtok.shape[3]
    dWp = np.empty((V, P2, D), dtype=F64)
    dbp = np.empty((V, D), dtype=F64)
    for v in range(V):
        dWp[v] = pix[:, v].reshape(B * L, P2).T @ dtok[:, :, v, :].reshape(B * L, D)
        dbp[v] = dtok[:, :, v, :].reshape(B * L, D).sum(axis=0)
    return dWp, dbp


# ---------------------------------------------------------------------------------------------
# A2 -- variable aggregation ("aggregated together across different channels using
# cross-attention"; "same as the ClimaX"; readings 3, 4)
# ---------------------------------------------------------------------------------------------
def var_aggregate(tok, P, heads, pos=None):
    """At every (b, l), X = tok[b, l] in R^{V x D}:
         qt = q Wq + bq;  K = X Wk + bk;  U = X Wv + bv;
         per head a (d_a = D/heads): s_v = qt_a . K_{v,a} / sqrt(d_a); alpha = softmax_v(s);
         o_a = sum_v alpha_v U_{v,a};  agg[b, l] = concat_a(o_a) Wo + bo (+ pos[l]).
    Returns (agg [B, L, D], cache)."""
    tok = _f64(tok)
    B, L, V, D = tok.shape
    da = D // heads
    q, Wq, bq = _f64(P["q"]), _f64(P["Wq"]), _f64(P["bq"])
    Wk, bk, Wv, bv = _f64(P["Wk"]), _f64(P["bk"]), _f64(P["Wv"]), _f64(P["bv"])
    Wo, bo = _f64(P["Wo"]), _f64(P["bo"])
    qt = q @ Wq + bq                                               # [D], data independent
    K = tok @ Wk + bk                                              # [B, L, V, D]
    U = tok @ Wv + bv
    Kh = K.reshape(B, L, V, heads, da)
    Uh = U.reshape(B, L, V, heads, da)
    qh = qt.reshape(heads, da)
    s = np.einsum("ac,blvac->blav", qh, Kh) / math.sqrt(da)        # [B, L, heads, V]
    alpha = softmax_lastdim(s)
    o = np.einsum("blav,blvac->blac", alpha, Uh).reshape(B, L, D)
    agg = o @ Wo + bo
    if pos is not None:
        agg = agg + _f64(pos)[None, :, :]
    cache = dict(tok=tok, qt=qt, Kh=Kh, Uh=Uh, alpha=alpha, o=o, heads=heads)
    return agg, cache


def var_aggregate_bwd(dagg, P, cache, want_dpos=False):
    """Backward of var_aggregate, given g = dagg[b, l]:
       dbo += g; dWo += o^T g; dpos[l] += g; do = g Wo^T;
       per head: dalpha_v = do_a . U_{v,a}; dU_{v,a} = alpha_v do_a;
                 ds_v = alpha_v (dalpha_v - sum_w alpha_w dalpha_w);
                 dqt_a += sum_v ds_v K_{v,a}/sqrt(d_a); dK_{v,a} = ds_v qt_a/sqrt(d_a);
       dWk += X^T dK; dbk += sum dK; dWv += X^T dU; dbv += sum dU; dtok = dK Wk^T + dU Wv^T;
       dbq = dqt; dWq = q^T dqt; dq = dqt Wq^T."""
    dagg = _f64(dagg)
    tok, qt, Kh, Uh, alpha, o = (cache[k] for k in ("tok", "qt", "Kh", "Uh", "alpha", "o"))
    heads = cache["heads"]
    B, L, V, D = tok.shape
    da = D // heads
    q, Wq = _f64(P["q"]), _f64(P["Wq"])
    Wk, Wv, Wo = _f64(P["Wk"]), _f64(P["Wv"]), _f64(P["Wo"])
    G = {}
    g2 = dagg.reshape(B * L, D)
    G["bo"] = g2.sum(axis=0)
    G["Wo"] = o.reshape(B * L, D).T @ g2
    dpos = dagg.sum(axis=0) if want_dpos else None
    do = (dagg @ Wo.T).reshape(B, L, heads, da)
    dalpha = np.einsum("blac,blvac->blav", do, Uh)
    dUh = np.einsum("blav,blac->blvac", alpha, do)
    ds = alpha * (dalpha - (alpha * dalpha).sum(axis=-1, keepdims=True))
    qh = qt.reshape(heads, da)
    dqt = (np.einsum("blav,blvac->ac", ds, Kh) / math.sqrt(da)).reshape(D)
    dKh = np.einsum("blav,ac->blvac", ds, qh) / math.sqrt(da)
    dK = dKh.reshape(B * L * V, D)
    dU = dUh.reshape(B * L * V, D)
    X = tok.reshape(B * L * V, D)
    G["Wk"] = X.T @ dK
    G["bk"] = dK.sum(axis=0)
    G["Wv"] = X.T @ dU
    G["bv"] = dU.sum(axis=0)
    dtok = (dK @ Wk.T + dU @ Wv.T).reshape(B, L, V, D)
    G["bq"] = dqt
    G["Wq"] = np.outer(q, dqt)
    G["q"] = dqt @ Wq.T
    return dtok, G, dpos


# ---------------------------------------------------------------------------------------------
# BLK -- one ViT block, pre-LN residual form (readings 5-8, 10)
# ---------------------------------------------------------------------------------------------
def attention(Q, K, V, heads):
    """Per (b, head j): S = Q_j K_j^T / sqrt(d_h); P = softmax over keys; O_j = P V_j
    (PAPER.md:88 softmax(QK^T)V; :114 "scaled dot product").  Q, K, V: [B, N, D] -> O [B, N, D],
    P [B, heads, N, N]."""
    B, N, D = Q.shape                       # Q may hold a subset of the query rows (N != K.shape[1])
    dh = D // heads
    O = np.empty((B, N, D), dtype=F64)
    Pm = np.empty((B, heads, N, K.shape[1]), dtype=F64)
    for b in range(B):
        for j in range(heads):
            c = slice(j * dh, (j + 1) * dh)
            S = (Q[b, :, c] @ K[b, :, c].T) / math.sqrt(dh)
            Pj = softmax_lastdim(S)
            Pm[b, j] = Pj
            O[b, :, c] = Pj @ V[b, :, c]
    return O, Pm


def attention_bwd(dO, Q, K, V, Pm, heads):
    """Per head: dV = P^T dO_j; dP = dO_j V_j^T; dS = P o (dP - rowsum(dP o P));
    dQ = dS K_j / sqrt(d_h); dK = dS^T Q_j / sqrt(d_h)."""
    B, N, D = Q.shape
    dh = D // heads
    dQ = np.empty_like(Q)
    dK = np.empty_like(K)
    dV = np.empty_like(V)
    for b in range(B):
        for j in range(heads):
            c = slice(j * dh, (j + 1) * dh)
            Pj = Pm[b, j]
            dV[b, :, c] = Pj.T @ dO[b, :, c]
            dP = dO[b, :, c] @ V[b, :, c].T
            dS = Pj * (dP - (dP * Pj).sum(axis=-1, keepdims=True))
            dQ[b, :, c] = dS @ K[b, :, c] / math.sqrt(dh)
            dK[b, :, c] = dS.T @ Q[b, :, c] / math.sqrt(dh)
    return dQ, dK, dV


def qk_layernorm(Z, heads, gamma, beta, eps):
    """QK-LayerNorm ("additional layer normalization to the queries ... and keys ... before
    computing the self-attention scaled dot product", after [8]; reading 9): LayerNorm over the d_h entries
    of every head's query (resp. key) vector, gamma / beta in R^{d_h} shared by all heads.
    Z: [B, N, heads*d_h] -> (normalised [B, N, heads*d_h], zhat [B, N, heads, d_h], rstd)."""
    B, N, Dz = Z.shape
    dh = Dz // heads
    out, zhat, rstd = layernorm(Z.reshape(B, N, heads, dh), gamma, beta, eps)
    return out.reshape(B, N, Dz), zhat, rstd


def qk_layernorm_bwd(dZn, heads, zhat, rstd, gamma):
    """Backward of qk_layernorm: (dZ [B, N, heads*d_h], dgamma [d_h], dbeta [d_h]) -- gamma / beta gradients
    sum over tokens AND heads (the parameters are shared by the heads)."""
    B, N, Dz = dZn.shape
    dh = Dz // heads
    dz, dgamma, dbeta = layernorm_bwd(_f64(dZn).reshape(B, N, heads, dh), zhat, rstd, gamma)
    return dz.reshape(B, N, Dz), dgamma, dbeta


def has_qk_norm(P):
    """A block uses QK-LayerNorm iff its parameter dict carries qn_g, qn_b, kn_g, kn_b (all [d_h])."""
    return "qn_g" in P


def block_fwd(x, P, heads, eps=1e-5):
    """a = LN1(x); [Q|K|V] = a Wqkv + bqkv; (Q, K <- QK-LayerNorm per head when P has qn_g.. : PAPER.md:114);
    O = attention; x1 = x + O Wproj + bproj;
    m = LN2(x1); u = m Wfc1 + bfc1; g = GELU(u); y = x1 + g Wfc2 + bfc2.    x: [B, N, D]."""
    x = _f64(x)
    B, N, D = x.shape
    a, xhat, rstd1 = layernorm(x, P["ln1_g"], P["ln1_b"], eps)
    qkv = a @ _f64(P["Wqkv"]) + _f64(P["bqkv"])
    Q, K, V = qkv[..., 0:D], qkv[..., D:2 * D], qkv[..., 2 * D:3 * D]
    qkn = None
    if has_qk_norm(P):
        Q, qhat, qrstd = qk_layernorm(Q, heads, P["qn_g"], P["qn_b"], eps)
        K, khat, krstd = qk_layernorm(K, heads, P["kn_g"], P["kn_b"], eps)
        qkn = dict(qhat=qhat, qrstd=qrstd, khat=khat, krstd=krstd)
    O, Pm = attention(Q, K, V, heads)
    x1 = x + O @ _f64(P["Wproj"]) + _f64(P["bproj"])
    m, x1hat, rstd2 = layernorm(x1, P["ln2_g"], P["ln2_b"], eps)
    u = m @ _f64(P["Wfc1"]) + _f64(P["bfc1"])
    g = gelu(u)
    y = x1 + g @ _f64(P["Wfc2"]) + _f64(P["bfc2"])
    cache = dict(xhat=xhat, rstd1=rstd1, a=a, Q=Q, K=K, V=V, Pm=Pm, O=O, x1=x1, x1hat=x1hat,
                 rstd2=rstd2, m=m, u=u, g=g, heads=heads, qkn=qkn)
    return y, cache


def block_bwd(dy, P, cache):
    """SURVEY.md §8(c)-BLK': dx and the 12 parameter gradients, given dy."""
    dy = _f64(dy)
    B, N, D = dy.shape
    M = B * N
    c = cache
    heads = c["heads"]
    G = {}
    dy2 = dy.reshape(M, D)
    F = c["u"].shape[-1]
    G["bfc2"] = dy2.sum(axis=0)
    G["Wfc2"] = c["g"].reshape(M, F).T @ dy2
    dg = dy @ _f64(P["Wfc2"]).T
    du = dg * gelu_grad(c["u"])
    du2 = du.reshape(M, F)
    G["bfc1"] = du2.sum(axis=0)
    G["Wfc1"] = c["m"].reshape(M, D).T @ du2
    dm = du @ _f64(P["Wfc1"]).T
    dz2, G["ln2_g"], G["ln2_b"] = layernorm_bwd(dm, c["x1hat"], c["rstd2"], P["ln2_g"])
    dx1 = dy + dz2
    dx12 = dx1.reshape(M, D)
    G["bproj"] = dx12.sum(axis=0)
    G["Wproj"] = c["O"].reshape(M, D).T @ dx12
    dO = dx1 @ _f64(P["Wproj"]).T
    dQ, dK, dV = attention_bwd(dO, c["Q"], c["K"], c["V"], c["Pm"], heads)
    if c.get("qkn") is not None:
        n = c["qkn"]
        dQ, G["qn_g"], G["qn_b"] = qk_layernorm_bwd(dQ, heads, n["qhat"], n["qrstd"], P["qn_g"])
        dK, G["kn_g"], G["kn_b"] = qk_layernorm_bwd(dK, heads, n["khat"], n["krstd"], P["kn_g"])
    dqkv = np.concatenate([dQ, dK, dV], axis=-1)
    dqkv2 = dqkv.reshape(M, 3 * D)
    G["bqkv"] = dqkv2.sum(axis=0)
    G["Wqkv"] = c["a"].reshape(M, D).T @ dqkv2
    da = dqkv @ _f64(P["Wqkv"]).T
    dz1, G["ln1_g"], G["ln1_b"] = layernorm_bwd(da, c["xhat"], c["rstd1"], P["ln1_g"])
    dx = dx1 + dz1
    return dx, G


# ---------------------------------------------------------------------------------------------
# SHARD -- Hybrid-STOP shard-local arithmetic (Eq. 1-3, Fig. 3; readings 13-16)
# implemented SEPARATELY from BLK; tests assert the two agree to ~1e-13.
# ---------------------------------------------------------------------------------------------
def chain_sharded(x, A_cols, B_rows):
    """Eq. (2):  y = sum_k (x A_{*,k}) B_{k,*}."""
    y = None
    for Ak, Bk in zip(A_cols, B_rows):
        part = (_f64(x) @ _f64(Ak)) @ _f64(Bk)
        y = part if y is None else y + part
    return y


def chain_sharded_dx(dy, A_cols, B_rows):
    """Eq. (3): row-wise dx = dy (sum_k B_{k,*}^T A_{*,k}^T); rows independent
    (the "(x) I"), so no Kronecker product is formed (reading 16)."""
    dx = None
    for Ak, Bk in zip(A_cols, B_rows):
        part = (_f64(dy) @ _f64(Bk).T) @ _f64(Ak).T
        dx = part if dx is None else dx + part
    return dx


def block_fwd_sharded(x, Pc, shards, heads, eps=1e-5):
    """Forward with T shards run one after another (Fig. 3a):
       a = LN1(x) once; for k: qkv^k = a Wqkv^k + bqkv^k -> attention on that shard's heads/T heads
       -> O^k [.., D/T] -> P^k = O^k Wproj^k;  x1 = x + sum_k P^k + bproj;
       m = LN2(x1); for k: g^k = GELU(m Wfc1^k + bfc1^k); Y^k = g^k Wfc2^k; y = x1 + sum_k Y^k + bfc2.
    Pc: the unsharded parameters ln1_g, ln1_b, ln2_g, ln2_b, bproj, bfc2 (reading 14: bias and
    residual enter once, after the combine)."""
    x = _f64(x)
    B, N, D = x.shape
    T = len(shards)
    hk = heads // T
    dc = D // T
    a, xhat, rstd1 = layernorm(x, Pc["ln1_g"], Pc["ln1_b"], eps)
    per = []
    acc = np.zeros_like(x)
    for S in shards:
        qkv = a @ _f64(S["Wqkv"]) + _f64(S["bqkv"])
        Q, K, V = qkv[..., 0:dc], qkv[..., dc:2 * dc], qkv[..., 2 * dc:3 * dc]
        qkn = None
        if has_qk_norm(Pc):          # gamma / beta in R^{d_h} are shared by the heads, hence by the shards
            Q, qhat, qrstd = qk_layernorm(Q, hk, Pc["qn_g"], Pc["qn_b"], eps)
            K, khat, krstd = qk_layernorm(K, hk, Pc["kn_g"], Pc["kn_b"], eps)
            qkn = dict(qhat=qhat, qrstd=qrstd, khat=khat, krstd=krstd)
        O, Pm = attention(Q, K, V, hk)
        acc = acc + O @ _f64(S["Wproj"])
        per.append(dict(Q=Q, K=K, V=V, Pm=Pm, O=O, qkn=qkn))
    x1 = x + acc + _f64(Pc["bproj"])
    m, x1hat, rstd2 = layernorm(x1, Pc["ln2_g"], Pc["ln2_b"], eps)
    acc2 = np.zeros_like(x)
    for S, c in zip(shards, per):
        u = m @ _f64(S["Wfc1"]) + _f64(S["bfc1"])
        g = gelu(u)
        acc2 = acc2 + g @ _f64(S["Wfc2"])
        c["u"], c["g"] = u, g
    y = x1 + acc2 + _f64(Pc["bfc2"])
    cache = dict(xhat=xhat, rstd1=rstd1, a=a, x1=x1, x1hat=x1hat, rstd2=rstd2, m=m, per=per,
                 heads=heads)
    return y, cache


def block_bwd_sharded(dy, Pc, shards, cache):
    """Backward mirror (Eq. 3): per-shard grads as in BLK' with
    dm = sum_k du^k Wfc1^k^T and da = sum_k dqkv^k Wqkv^k^T ("add their activation gradients
    together")."""
    dy = _f64(dy)
    B, N, D = dy.shape
    M = B * N
    T = len(shards)
    hk = cache["heads"] // T
    Gc = {}
    Gs = [dict() for _ in shards]
    dy2 = dy.reshape(M, D)
    Gc["bfc2"] = dy2.sum(axis=0)
    dm = np.zeros_like(dy)
    for S, c, G in zip(shards, cache["per"], Gs):
        Fk = c["u"].shape[-1]
        G["Wfc2"] = c["g"].reshape(M, Fk).T @ dy2
        du = (dy @ _f64(S["Wfc2"]).T) * gelu_grad(c["u"])
        G["bfc1"] = du.reshape(M, Fk).sum(axis=0)
        G["Wfc1"] = cache["m"].reshape(M, D).T @ du.reshape(M, Fk)
        dm = dm + du @ _f64(S["Wfc1"]).T
    dz2, Gc["ln2_g"], Gc["ln2_b"] = layernorm_bwd(dm, cache["x1hat"], cache["rstd2"], Pc["ln2_g"])
    dx1 = dy + dz2
    dx12 = dx1.reshape(M, D)
    Gc["bproj"] = dx12.sum(axis=0)
    da = np.zeros_like(dy)
    for S, c, G in zip(shards, cache["per"], Gs):
        dc = c["O"].shape[-1]
        G["Wproj"] = c["O"].reshape(M, dc).T @ dx12
        dO = dx1 @ _f64(S["Wproj"]).T
        dQ, dK, dV = attention_bwd(dO, c["Q"], c["K"], c["V"], c["Pm"], hk)
        if c.get("qkn") is not None:
            n = c["qkn"]
            dQ, gqg, gqb = qk_layernorm_bwd(dQ, hk, n["qhat"], n["qrstd"], Pc["qn_g"])
            dK, gkg, gkb = qk_layernorm_bwd(dK, hk, n["khat"], n["krstd"], Pc["kn_g"])
            for name, g in (("qn_g", gqg), ("qn_b", gqb), ("kn_g", gkg), ("kn_b", gkb)):
                Gc[name] = Gc.get(name, 0.0) + g          # shared parameters: sum over the shards
        dqkv = np.concatenate([dQ, dK, dV], axis=-1)
        G["bqkv"] = dqkv.reshape(M, 3 * dc).sum(axis=0)
        G["Wqkv"] = cache["a"].reshape(M, D).T @ dqkv.reshape(M, 3 * dc)
        da = da + dqkv @ _f64(S["Wqkv"]).T
    dz1, Gc["ln1_g"], Gc["ln1_b"] = layernorm_bwd(da, cache["xhat"], cache["rstd1"], Pc["ln1_g"])
    dx = dx1 + dz1
    return dx, Gc, Gs


# ---------------------------------------------------------------------------------------------
# RANK -- the rank-local Hybrid-STOP program (Fig. 3): what ONE rank of a tensor-parallel group
# computes between the collectives.  Rank k holds the column shards Wqkv^k, Wfc1^k (with bqkv^k, bfc1^k) and the row
# shards Wproj^k, Wfc2^k; the replicated parameters (LayerNorm gains / offsets, bproj, bfc2) live on every rank.
# "GPUs in each tensor-parallel group add their individual activations together" after the row-sharded
# products, and "add their activation gradients together through all-reduce" after the transposed
# column-sharded products: four all-reduce(sum) of an [B, N, D] partial per block.  `allreduce` is passed in (a
# function partial -> sum over the ranks), so the same code runs under torch.distributed (tests/test_multiproc.py,
# world size 2, gloo) and with a plain Python sum.  Written separately from BLK / SHARD; pinned against BLK.
# ---------------------------------------------------------------------------------------------
def rank_block_fwd(x, Pc, S, heads_local, allreduce, eps=1e-5):
    """Forward of rank k.  x: the replicated block input [B, N, D]; Pc: replicated parameters; S: this rank's shard
    (Wqkv [D, 3D/T] = [Q_k | K_k | V_k], bqkv, Wproj [D/T, D], Wfc1 [D, F/T], bfc1, Wfc2 [F/T, D]); heads_local =
    heads / T.  Returns (y, cache, partials): y is identical on every rank; `partials` are this rank's two
    pre-all-reduce partial products (what the collective sees)."""
    x = _f64(x)
    D = x.shape[-1]
    dc = _f64(S["Wproj"]).shape[0]
    a, xhat, rstd1 = layernorm(x, Pc["ln1_g"], Pc["ln1_b"], eps)
    qkv = a @ _f64(S["Wqkv"]) + _f64(S["bqkv"])
    Q, K, V = qkv[..., 0:dc], qkv[..., dc:2 * dc], qkv[..., 2 * dc:3 * dc]
    qkn = None
    if has_qk_norm(Pc):
        Q, qhat, qrstd = qk_layernorm(Q, heads_local, Pc["qn_g"], Pc["qn_b"], eps)
        K, khat, krstd = qk_layernorm(K, heads_local, Pc["kn_g"], Pc["kn_b"], eps)
        qkn = dict(qhat=qhat, qrstd=qrstd, khat=khat, krstd=krstd)
    O, Pm = attention(Q, K, V, heads_local)
    part_proj = O @ _f64(S["Wproj"])                       # row shard: a partial of the full product (Eq. 2)
    x1 = x + allreduce(part_proj) + _f64(Pc["bproj"])     # PAPER.md:98; bias and residual once, after the sum (R14)
    m, x1hat, rstd2 = layernorm(x1, Pc["ln2_g"], Pc["ln2_b"], eps)
    u = m @ _f64(S["Wfc1"]) + _f64(S["bfc1"])
    g = gelu(u)
    part_fc2 = g @ _f64(S["Wfc2"])
    y = x1 + allreduce(part_fc2) + _f64(Pc["bfc2"])
    cache = dict(xhat=xhat, rstd1=rstd1, a=a, Q=Q, K=K, V=V, Pm=Pm, O=O, qkn=qkn, x1hat=x1hat, rstd2=rstd2, m=m, u=u,
                 g=g, heads_local=heads_local)
    return y, cache, dict(proj=part_proj, fc2=part_fc2)


def rank_block_bwd(dy, Pc, S, cache, allreduce):
    """Backward of rank k (Eq. 3).  Returns (dx, Gc, Gs, partials): dx and the gradients Gc of the
    replicated parameters are identical on every rank EXCEPT the QK-LayerNorm ones (qn_g, qn_b, kn_g, kn_b), which are
    this rank's sum over its own heads and still have to be summed over the group; Gs are the gradients of this rank's
    shard; `partials` are the two pre-all-reduce activation-gradient partials."""
    dy = _f64(dy)
    B, N, D = dy.shape
    M = B * N
    c = cache
    hk = c["heads_local"]
    Fk = c["u"].shape[-1]
    dc = c["O"].shape[-1]
    Gc, Gs = {}, {}
    dy2 = dy.reshape(M, D)
    Gc["bfc2"] = dy2.sum(axis=0)
    Gs["Wfc2"] = c["g"].reshape(M, Fk).T @ dy2
    du = (dy @ _f64(S["Wfc2"]).T) * gelu_grad(c["u"])
    Gs["bfc1"] = du.reshape(M, Fk).sum(axis=0)
    Gs["Wfc1"] = c["m"].reshape(M, D).T @ du.reshape(M, Fk)
    part_dm = du @ _f64(S["Wfc1"]).T
    dm = allreduce(part_dm)
    dz2, Gc["ln2_g"], Gc["ln2_b"] = layernorm_bwd(dm, c["x1hat"], c["rstd2"], Pc["ln2_g"])
    dx1 = dy + dz2
    dx12 = dx1.reshape(M, D)
    Gc["bproj"] = dx12.sum(axis=0)
    Gs["Wproj"] = c["O"].reshape(M, dc).T @ dx12
    dO = dx1 @ _f64(S["Wproj"]).T
    dQ, dK, dV = attention_bwd(dO, c["Q"], c["K"], c["V"], c["Pm"], hk)
    if c.get("qkn") is not None:
        n = c["qkn"]
        dQ, Gc["qn_g"], Gc["qn_b"] = qk_layernorm_bwd(dQ, hk, n["qhat"], n["qrstd"], Pc["qn_g"])
        dK, Gc["kn_g"], Gc["kn_b"] = qk_layernorm_bwd(dK, hk, n["khat"], n["krstd"], Pc["kn_g"])
    dqkv = np.concatenate([dQ, dK, dV], axis=-1)
    Gs["bqkv"] = dqkv.reshape(M, 3 * dc).sum(axis=0)
    Gs["Wqkv"] = c["a"].reshape(M, D).T @ dqkv.reshape(M, 3 * dc)
    part_da = dqkv @ _f64(S["Wqkv"]).T
    da = allreduce(part_da)
    dz1, Gc["ln1_g"], Gc["ln1_b"] = layernorm_bwd(da, c["xhat"], c["rstd1"], Pc["ln1_g"])
    dx = dx1 + dz1
    return dx, Gc, Gs, dict(dm=part_dm, da=part_da)


# ---------------------------------------------------------------------------------------------
# Sampled outputs at full size.  The same formulas as TOK / A2 / BLK / BLK' restricted to the outputs a
# test samples, for sizes where the whole oracle would take too long (tests pin each of them to the
# corresponding slice of the full functions on small shapes).
# ---------------------------------------------------------------------------------------------
def tokenize_patches(x, Wp, bp, p, ls):
    """tok[:, ls, :, :] of tokenize(): tokens of the sampled patches `ls` only."""
    pix = patches(x, p)[:, :, ls, :]                                  # [B, V, S, p^2]
    Wp, bp = _f64(Wp), _f64(bp)
    B, V, S, _ = pix.shape
    tok = np.empty((B, S, V, Wp.shape[2]), dtype=F64)
    for v in range(V):
        tok[:, :, v, :] = pix[:, v] @ Wp[v] + bp[v]
    return tok


def tokenize_bwd_patches(x, dtok_s, p, ls):
    """Contribution of the sampled patches `ls` to tokenize_bwd(): dWp[v, r, :] = sum_{b, l in ls} pix dtok_s,
    dbp[v, :] = sum_{b, l in ls} dtok_s, with dtok_s = dtok[:, ls] ([B, S, V, D]).  The gradients are sums over
    (b, l), so the contributions of a partition of the patches add up to tokenize_bwd() exactly."""
    pix = patches(x, p)[:, :, ls, :]                                  # [B, V, S, p^2]
    dtok_s = _f64(dtok_s)
    B, V, S, P2 = pix.shape
    D = dtok_s.shape[3]
    dWp = np.empty((V, P2, D), dtype=F64)
    dbp = np.empty((V, D), dtype=F64)
    for v in range(V):
        dWp[v] = pix[:, v].reshape(B * S, P2).T @ dtok_s[:, :, v, :].reshape(B * S, D)
        dbp[v] = dtok_s[:, :, v, :].reshape(B * S, D).sum(axis=0)
    return dWp, dbp


def block_sampled(x, dy, P, heads, eps, rows, fcols):
    """Outputs of block_fwd / block_bwd that can be had one by one without the whole backward:
       y[:, rows, :];  dbfc2;  and for the sampled MLP columns f in fcols: dWfc2[f, :], dWfc1[:, f],
       dbfc1[f].  The first half (LN1, QKV, attention, proj, LN2) is computed in full exactly as in
       block_fwd; the MLP is evaluated on the sampled rows (for y) and the sampled columns (for grads)."""
    x, dy = _f64(x), _f64(dy)
    B, N, D = x.shape
    M = B * N
    a, _, _ = layernorm(x, P["ln1_g"], P["ln1_b"], eps)
    qkv = a @ _f64(P["Wqkv"]) + _f64(P["bqkv"])
    O, _ = attention(qkv[..., 0:D], qkv[..., D:2 * D], qkv[..., 2 * D:3 * D], heads)
    x1 = x + O @ _f64(P["Wproj"]) + _f64(P["bproj"])
    m, _, _ = layernorm(x1, P["ln2_g"], P["ln2_b"], eps)
    out = {"x1": x1}
    # y on the sampled rows: u = m Wfc1 + bfc1; g = GELU(u); y = x1 + g Wfc2 + bfc2
    Wfc1, Wfc2 = _f64(P["Wfc1"]), _f64(P["Wfc2"])
    u_r = m[:, rows, :] @ Wfc1 + _f64(P["bfc1"])
    out["y_rows"] = x1[:, rows, :] + gelu(u_r) @ Wfc2 + _f64(P["bfc2"])
    # MLP gradients on the sampled columns
    dy2, m2 = dy.reshape(M, D), m.reshape(M, D)
    out["bfc2"] = dy2.sum(axis=0)
    u_f = m2 @ Wfc1[:, fcols] + _f64(P["bfc1"])[fcols]                # [M, |f|]
    g_f = gelu(u_f)
    out["Wfc2_rows"] = g_f.T @ dy2                                    # dWfc2[f, :]
    du_f = (dy2 @ Wfc2[fcols, :].T) * gelu_grad(u_f)
    out["bfc1_cols"] = du_f.sum(axis=0)
    out["Wfc1_cols"] = m2.T @ du_f                                    # dWfc1[:, f]
    return out


# ---------------------------------------------------------------------------------------------
# Harness loss (BASELINE.json config 1: "target is an N(0,1) field with MSE loss")
# ---------------------------------------------------------------------------------------------
def mse_loss(y, t):
    """loss = mean((y - t)^2); dy = 2 (y - t) / numel."""
    y, t = _f64(y), _f64(t)
    d = y - t
    return float((d * d).mean()), 2.0 * d / d.size


# ---------------------------------------------------------------------------------------------
# HEAD -- final LayerNorm, projection "from the feature space to the image space" and the
# latitude-weighted MSE the paper trains with ("training loss computed as the latitude-weighted
# Mean Squared Error (wMSE)"); readings R26-R28 of DESIGN.md.
# ---------------------------------------------------------------------------------------------
def lat_weights(Hg):
    """w_i = cos(lat_i) / mean_i cos(lat_i) at the cell centres lat_i = -90 + (i + 1/2) 180/Hg (reading R27:
    the paper only says "latitude-weighted"; PAPER.md:171 gives the reason: cell areas shrink towards the poles)."""
    lat = -90.0 + (np.arange(Hg, dtype=F64) + 0.5) * 180.0 / Hg
    w = np.cos(np.deg2rad(lat))
    return w / w.mean()


def unpatchify(P, V, Hg, Wg, p):
    """P[b, l, v*p^2 + r] -> img[b, v, i*p+di, j*p+dj] with l = i*(Wg/p)+j, r = di*p+dj: the inverse of `patches`
    per variable (reading R26: head columns are variable-major, pixels row-major inside a patch)."""
    B, L, _ = P.shape
    gh, gw = Hg // p, Wg // p
    return P.reshape(B, gh, gw, V, p, p).transpose(0, 3, 1, 4, 2, 5).reshape(B, V, Hg, Wg)


def patchify_img(img, p):
    """Inverse of unpatchify: img[b, v, y, x] -> [b, l, v*p^2 + r]."""
    B, V, Hg, Wg = img.shape
    gh, gw = Hg // p, Wg // p
    return img.reshape(B, V, gh, p, gw, p).transpose(0, 2, 4, 1, 3, 5).reshape(B, gh * gw, V * p * p)


def head_loss(z, Ph, target, p, eps=1e-5, latw=None):
    """zn = LN_f(z); P = zn Wh + bh ([B, L, V p^2]); pred = unpatchify(P) ([B, V, Hg, Wg]);
    loss = mean_{b,v,y,x} w_y (pred - target)^2.  Ph: lnf_g, lnf_b [D], Wh [D, V p^2], bh [V p^2]."""
    z, target = _f64(z), _f64(target)
    B, V, Hg, Wg = target.shape
    w = lat_weights(Hg) if latw is None else _f64(latw)
    zn, zhat, rstd = layernorm(z, Ph["lnf_g"], Ph["lnf_b"], eps)
    P = zn @ _f64(Ph["Wh"]) + _f64(Ph["bh"])
    pred = unpatchify(P, V, Hg, Wg, p)
    diff = pred - target
    loss = float((w[None, None, :, None] * diff * diff).mean())
    cache = dict(zn=zn, zhat=zhat, rstd=rstd, diff=diff, w=w, p=p)
    return loss, pred, cache


def head_loss_bwd(Ph, cache):
    """dpred = 2 w_y (pred - target) / (B V Hg Wg); dP = patchify(dpred); dbh = sum dP; dWh = zn^T dP;
    dzn = dP Wh^T; dz, dlnf_g, dlnf_b = LayerNorm backward."""
    diff, w, p = cache["diff"], cache["w"], cache["p"]
    dpred = 2.0 * w[None, None, :, None] * diff / diff.size
    dP = patchify_img(dpred, p)
    B, L, C = dP.shape
    D = cache["zn"].shape[-1]
    G = {}
    G["bh"] = dP.reshape(B * L, C).sum(axis=0)
    G["Wh"] = cache["zn"].reshape(B * L, D).T @ dP.reshape(B * L, C)
    dzn = dP @ _f64(Ph["Wh"]).T
    dz, G["lnf_g"], G["lnf_b"] = layernorm_bwd(dzn, cache["zhat"], cache["rstd"], Ph["lnf_g"])
    return dz, G


def step_head(x, emb, agg, blocks, head, target_img, p, heads, eps=1e-5, pos=None):
    """Whole training step with the paper's loss: tokenise -> aggregate -> blocks -> head -> wMSE, and backward."""
    tok = tokenize(x, emb["Wp"], emb["bp"], p)
    z, acache = var_aggregate(tok, agg, heads, pos)
    caches = []
    h = z
    for P in blocks:
        h, c = block_fwd(h, P, heads, eps)
        caches.append(c)
    loss, pred, hc = head_loss(h, head, target_img, p, eps)
    dh, Gh = head_loss_bwd(head, hc)
    out = dict(agg=z, y=h, loss=loss, pred=pred, dy=dh, head_grads=Gh, block_grads=[None] * len(blocks))
    for i in reversed(range(len(blocks))):
        dh, G = block_bwd(dh, blocks[i], caches[i])
        out["block_grads"][i] = G
    out["dagg"] = dh
    dtok, Ga, dpos = var_aggregate_bwd(dh, agg, acache, want_dpos=pos is not None)
    out["agg_grads"], out["dpos"] = Ga, dpos
    out["dWp"], out["dbp"] = tokenize_bwd(x, dtok, p)
    return out


# ---------------------------------------------------------------------------------------------
# Whole step (tokenise -> aggregate -> depth x block, forward and backward)
# ---------------------------------------------------------------------------------------------
def step(x, emb, agg, blocks, target, p, heads, eps=1e-5, pos=None):
    """One training step of the hot path.  Returns dict with every output and gradient."""
    tok = tokenize(x, emb["Wp"], emb["bp"], p)
    z, acache = var_aggregate(tok, agg, heads, pos)
    caches = []
    h = z
    for P in blocks:
        h, c = block_fwd(h, P, heads, eps)
        caches.append(c)
    loss, dh = mse_loss(h, target)
    out = dict(tok=tok, agg=z, y=h, loss=loss, dy=dh, block_grads=[None] * len(blocks))
    for i in reversed(range(len(blocks))):
        dh, G = block_bwd(dh, blocks[i], caches[i])
        out["block_grads"][i] = G
    out["dagg"] = dh
    dtok, Ga, dpos = var_aggregate_bwd(dh, agg, acache, want_dpos=pos is not None)
    out["dtok"], out["agg_grads"], out["dpos"] = dtok, Ga, dpos
    out["dWp"], out["dbp"] = tokenize_bwd(x, dtok, p)
    return out


# ---------------------------------------------------------------------------------------------
# SCALE -- dynamic gradient scaling and fp32 gradient accumulation ("we applied the PyTorch dynamic
# gradient scaling mechanism [24] ... detects the value range of the computed gradient magnitude ... scale the gradient
# magnitudes to the proper value range representable in BFLOAT16, and then reverse the scaling during the parameters
# update").  The loss gradient is multiplied by S before the backward pass; afterwards:
# ---------------------------------------------------------------------------------------------
def grads_unscale_check(grads, scale):
    """Reverse the scaling: g / S for every gradient tensor, and detect overflow: found_inf = 1.0 iff any gradient
    element is Inf or NaN (as [24] does: the test is on the computed gradient, before it is unscaled; the step is then
    skipped).  Returns (list of unscaled fp64 arrays, found_inf)."""
    inv = 1.0 / float(scale)
    found = 0.0
    for g in grads:
        if not np.isfinite(_f64(g)).all():
            found = 1.0
    with np.errstate(invalid="ignore"):
        out = [_f64(g) * inv for g in grads]
    return out, found


def grads_accumulate(acc, grads, scale=1.0):
    """Gradient accumulation across micro-steps: acc_i + g_i / S, per tensor (new list)."""
    inv = 1.0 / float(scale)
    return [_f64(a) + _f64(g) * inv for a, g in zip(acc, grads)]


def grad_scale_update(scale, tracker, found_inf, growth_factor, backoff_factor, growth_interval):
    """The scale schedule of [24]: on overflow S <- S * backoff_factor and the count of clean steps restarts; otherwise
    the count grows by one and, when it reaches growth_interval, S <- S * growth_factor and the count restarts.
    Returns (scale, tracker).  The paper gives no values for the three constants: they are arguments."""
    if found_inf != 0.0:
        return float(scale) * backoff_factor, 0
    tracker = int(tracker) + 1
    if tracker >= growth_interval:
        return float(scale) * growth_factor, 0
    return float(scale), tracker


def rel_fro(got, ref):
    """||got - ref||_F / ||ref||_F -- the parity metric north_star names."""
    got, ref = _f64(got), _f64(ref)
    den = float(np.sqrt((ref * ref).sum()))
    num = float(np.sqrt(((got - ref) ** 2).sum()))
    return num / den if den > 0 else num
