"""Pins for the fp64 oracle (oracle/orbit_oracle.py) against things other than itself:
finite differences, closed forms, invariants, textbook/library special cases (torch float64 CPU
autograd, conv2d), Eq. (1)-(3) of the paper.  All CPU, `-m "not gpu"`.

The paper prints no worked numerical example for the per-GPU math, so there are no
printed values to match; tests/golden/ holds closed-form fixtures with their derivations."""
import json
import math
import os

import numpy as np
import pytest
import torch

from oracle import orbit_oracle as orc
from paper_2404_14712_b200 import inputs as syn

RNG = np.random.default_rng(7)
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def rnd(*shape, scale=1.0):
    return RNG.standard_normal(shape) * scale


def rand_block_params(D, F):
    P = dict(ln1_g=1 + 0.1 * rnd(D), ln1_b=0.1 * rnd(D), Wqkv=rnd(D, 3 * D) / math.sqrt(D),
             bqkv=0.1 * rnd(3 * D), Wproj=rnd(D, D) / math.sqrt(D), bproj=0.1 * rnd(D),
             ln2_g=1 + 0.1 * rnd(D), ln2_b=0.1 * rnd(D), Wfc1=rnd(D, F) / math.sqrt(D),
             bfc1=0.1 * rnd(F), Wfc2=rnd(F, D) / math.sqrt(F), bfc2=0.1 * rnd(D))
    return P


def rand_agg_params(D):
    P = {"q": rnd(D)}
    for n in ("Wq", "Wk", "Wv", "Wo"):
        P[n] = rnd(D, D) / math.sqrt(D)
    for n in ("bq", "bk", "bv", "bo"):
        P[n] = 0.1 * rnd(D)
    return P


def fd_check(f, params: dict, names, analytic: dict, h=1e-6, tol=1e-6, nsamp=6):
    """Central finite differences of scalar f() w.r.t. sampled entries of params[name]."""
    for n in names:
        arr = params[n]
        flat = arr.reshape(-1)
        idx = RNG.choice(flat.size, size=min(nsamp, flat.size), replace=False)
        for i in idx:
            old = flat[i]
            flat[i] = old + h
            fp = f()
            flat[i] = old - h
            fm = f()
            flat[i] = old
            num = (fp - fm) / (2 * h)
            ana = analytic[n].reshape(-1)[i]
            assert abs(num - ana) <= tol * max(1.0, abs(ana), abs(num)), (n, i, num, ana)


# ------------------------------------------------------------------ elementary -----------------
def test_gelu_closed_forms():
    # golden fixture: GELU(0)=0, GELU'(0)=1/2, GELU(u)-GELU(-u)=u, GELU(1)=Phi(1) (tables)
    g = json.load(open(os.path.join(GOLD, "gelu_closed_form.json")))
    for u, val in zip(g["u"], g["gelu"]):
        assert abs(float(orc.gelu(u)) - val) < 1e-12
    assert float(orc.gelu(0.0)) == 0.0
    assert abs(float(orc.gelu_grad(0.0)) - 0.5) < 1e-15
    u = rnd(100) * 3
    assert np.allclose(orc.gelu(u) - orc.gelu(-u), u, atol=1e-14)
    # derivative by FD
    h = 1e-6
    assert np.allclose((orc.gelu(u + h) - orc.gelu(u - h)) / (2 * h), orc.gelu_grad(u), atol=1e-8)
    # library cross-check
    assert np.allclose(orc.gelu(u), torch.nn.functional.gelu(torch.tensor(u)).numpy(), atol=1e-14)


def test_softmax_rows_sum_to_one_and_shift_invariance():
    s = rnd(5, 7, 33) * 10
    P = orc.softmax_lastdim(s)
    assert np.allclose(P.sum(-1), 1.0, atol=1e-14)
    assert np.allclose(orc.softmax_lastdim(s + 123.4), P, atol=1e-13)
    # golden: softmax([0, ln2, ln3]) = [1/6, 2/6, 3/6]
    g = json.load(open(os.path.join(GOLD, "softmax_closed_form.json")))
    assert np.allclose(orc.softmax_lastdim(np.log(np.array(g["exp_logits"]))), g["probs"], atol=1e-15)
    # stress: logits x30 exercise the max subtraction
    assert np.isfinite(orc.softmax_lastdim(s * 30)).all()


def test_layernorm_zero_mean_unit_variance_and_bwd_invariants():
    z = rnd(6, 40) * 3 + 2
    eps = 1e-5
    out, zhat, rstd = orc.layernorm(z, np.ones(40), np.zeros(40), eps)
    assert np.allclose(out.mean(-1), 0, atol=1e-13)
    var = z.var(-1)
    assert np.allclose(out.var(-1), var / (var + eps), atol=1e-12)
    gam = 1 + 0.1 * rnd(40)
    dz, dg, db = orc.layernorm_bwd(rnd(6, 40), zhat, rstd, gam)
    assert np.allclose(dz.sum(-1), 0, atol=1e-12)
    # sum_i dz_i zhat_i = 0 holds exactly only for eps = 0 (mean(zhat^2) = var/(var+eps))
    _, zhat0, rstd0 = orc.layernorm(z, np.ones(40), np.zeros(40), 0.0)
    dz0, _, _ = orc.layernorm_bwd(rnd(6, 40), zhat0, rstd0, gam)
    assert np.allclose((dz0 * zhat0).sum(-1), 0, atol=1e-12)
    # library cross-check incl. backward
    zt = torch.tensor(z, requires_grad=True)
    gt = torch.tensor(gam, requires_grad=True)
    bt = torch.tensor(0.1 * rnd(40), requires_grad=True)
    o = torch.nn.functional.layer_norm(zt, (40,), gt, bt, eps)
    up = rnd(6, 40)
    o.backward(torch.tensor(up))
    out2, zhat2, rstd2 = orc.layernorm(z, gam, bt.detach().numpy(), eps)
    assert np.allclose(out2, o.detach().numpy(), atol=1e-13)
    dz2, dg2, db2 = orc.layernorm_bwd(up, zhat2, rstd2, gam)
    assert np.allclose(dz2, zt.grad.numpy(), atol=1e-12)
    assert np.allclose(dg2, gt.grad.numpy(), atol=1e-12)
    assert np.allclose(db2, bt.grad.numpy(), atol=1e-12)


# ------------------------------------------------------------------ Eq. (1)-(3) ----------------
@pytest.mark.parametrize("T", [1, 2, 4, 8])
def test_eq2_eq3_shard_sums_equal_unsharded(T):
    """sum_k (x A_{*,k}) B_{k,*} = xAB and sum_k dy B_{k,*}^T A_{*,k}^T = dy B^T A^T."""
    m, d, n, e = 13, 24, 8 * T, 17
    x, A, Bm, dy = rnd(m, d), rnd(d, n), rnd(n, e), rnd(m, e)
    Ac = [A[:, k * n // T:(k + 1) * n // T] for k in range(T)]
    Br = [Bm[k * n // T:(k + 1) * n // T, :] for k in range(T)]
    y = orc.chain_sharded(x, Ac, Br)
    assert orc.rel_fro(y, x @ A @ Bm) < 1e-13
    dx = orc.chain_sharded_dx(dy, Ac, Br)
    assert orc.rel_fro(dx, dy @ Bm.T @ A.T) < 1e-13
    # rows independent (the "(x) I"): perturbing dy row 0 changes only dx row 0
    dy2 = dy.copy()
    dy2[0] += 1.0
    dx2 = orc.chain_sharded_dx(dy2, Ac, Br)
    assert np.array_equal(dx2[1:], dx[1:]) and not np.allclose(dx2[0], dx[0])
    # elementwise phi commutes with column sharding: phi(xA)_{*,k} = phi(x A_{*,k})
    full = orc.gelu(x @ A)
    for k in range(T):
        assert np.allclose(full[:, k * n // T:(k + 1) * n // T], orc.gelu(x @ Ac[k]), atol=1e-14)


def test_eq1_worked_2x2_example():
    """Golden: a hand-computed instance of Eq. (1): x[A1,A2][B1;B2] = xA1B1 + xA2B2."""
    g = json.load(open(os.path.join(GOLD, "eq1_two_shard_example.json")))
    x, A, Bm = (np.array(g[k], dtype=float) for k in ("x", "A", "B"))
    y = orc.chain_sharded(x, [A[:, :1], A[:, 1:]], [Bm[:1, :], Bm[1:, :]])
    assert np.array_equal(y, np.array(g["y"], dtype=float))


# ------------------------------------------------------------------ tokeniser ------------------
def test_tokenize_is_strided_conv_and_roundtrip():
    B, V, Hg, Wg, p, D = 2, 3, 8, 12, 2, 5
    x = rnd(B, V, Hg, Wg)
    Wp, bp = rnd(V, p * p, D), rnd(V, D)
    tok = orc.tokenize(x, Wp, bp, p)
    assert tok.shape == (B, (Hg // p) * (Wg // p), V, D)
    for v in range(V):   # = stride-p convolution of channel v (library cross-check)
        w = torch.tensor(Wp[v].T.reshape(D, 1, p, p))
        ref = torch.nn.functional.conv2d(torch.tensor(x[:, v:v + 1]), w, torch.tensor(bp[v]), stride=p)
        ref = ref.flatten(2).transpose(1, 2).numpy()       # [B, L, D], row-major patches
        assert np.allclose(tok[:, :, v, :], ref, atol=1e-13)
    # one-hot weights reproduce the pixels (un-patchify round trip)
    D2 = p * p
    tok2 = orc.tokenize(x, np.tile(np.eye(D2)[None], (V, 1, 1)), np.zeros((V, D2)), p)
    gw = Wg // p
    for (b, v, i, j, di, dj) in [(0, 0, 0, 0, 0, 0), (1, 2, 3, 5, 1, 0), (0, 1, 2, 4, 1, 1)]:
        assert tok2[b, i * gw + j, v, di * p + dj] == x[b, v, i * p + di, j * p + dj]


def test_tokenize_bwd_fd():
    B, V, Hg, Wg, p, D = 1, 3, 8, 8, 2, 8
    x = rnd(B, V, Hg, Wg)
    prm = dict(Wp=rnd(V, p * p, D), bp=rnd(V, D))
    up = rnd(B, (Hg // p) * (Wg // p), V, D)
    f = lambda: float((orc.tokenize(x, prm["Wp"], prm["bp"], p) * up).sum())
    dWp, dbp = orc.tokenize_bwd(x, up, p)
    fd_check(f, prm, ["Wp", "bp"], dict(Wp=dWp, bp=dbp))


# ------------------------------------------------------------------ attention ------------------
def test_attention_special_cases():
    B, N, D, h = 2, 9, 8, 2
    Q, V = rnd(B, N, D), rnd(B, N, D)
    # identical keys => output = mean of the values (BASELINE.json north_star)
    K = np.tile(rnd(B, 1, D), (1, N, 1))
    O, Pm = orc.attention(Q, K, V, h)
    assert np.allclose(O, np.tile(V.mean(1, keepdims=True), (1, N, 1)), atol=1e-13)
    assert np.allclose(Pm.sum(-1), 1, atol=1e-14)
    # N = 1 => O = V
    O1, _ = orc.attention(Q[:, :1], K[:, :1], V[:, :1], h)
    assert np.allclose(O1, V[:, :1], atol=1e-15)
    # permuting keys+values together leaves O unchanged
    K = rnd(B, N, D)
    O, _ = orc.attention(Q, K, V, h)
    perm = RNG.permutation(N)
    O2, _ = orc.attention(Q, K[:, perm], V[:, perm], h)
    assert np.allclose(O, O2, atol=1e-13)
    # library cross-check
    def heads(t):
        return torch.tensor(t).reshape(B, N, h, D // h).transpose(1, 2)
    ref = torch.nn.functional.scaled_dot_product_attention(heads(Q), heads(K), heads(V))
    assert np.allclose(O, ref.transpose(1, 2).reshape(B, N, D).numpy(), atol=1e-13)


def test_attention_bwd_invariants():
    B, N, D, h = 1, 7, 8, 2
    Q, K, V, dO = rnd(B, N, D), rnd(B, N, D), rnd(B, N, D), rnd(B, N, D)
    O, Pm = orc.attention(Q, K, V, h)
    dQ, dK, dV = orc.attention_bwd(dO, Q, K, V, Pm, h)
    dh = D // h
    for j in range(h):
        c = slice(j * dh, (j + 1) * dh)
        dP = dO[0, :, c] @ V[0, :, c].T
        # rowsum(dP o P) = rowsum(dO o O) (the flash-attention delta identity)
        assert np.allclose((dP * Pm[0, j]).sum(-1), (dO[0, :, c] * O[0, :, c]).sum(-1), atol=1e-13)
        dS = Pm[0, j] * (dP - (dP * Pm[0, j]).sum(-1, keepdims=True))
        assert np.allclose(dS.sum(-1), 0, atol=1e-13)


# ------------------------------------------------------------------ block ----------------------
def torch_block(x, P, heads, eps):
    """Textbook block from torch library ops (float64 autograd) -- test-only cross-check."""
    F_ = torch.nn.functional
    B, N, D = x.shape
    a = F_.layer_norm(x, (D,), P["ln1_g"], P["ln1_b"], eps)
    qkv = a @ P["Wqkv"] + P["bqkv"]
    q, k, v = qkv.split(D, dim=-1)
    sp = lambda t: t.reshape(B, N, heads, D // heads).transpose(1, 2)
    o = F_.scaled_dot_product_attention(sp(q), sp(k), sp(v)).transpose(1, 2).reshape(B, N, D)
    x1 = x + o @ P["Wproj"] + P["bproj"]
    m = F_.layer_norm(x1, (D,), P["ln2_g"], P["ln2_b"], eps)
    return x1 + F_.gelu(m @ P["Wfc1"] + P["bfc1"]) @ P["Wfc2"] + P["bfc2"]


def test_block_matches_torch_autograd():
    B, N, D, h, F = 2, 10, 16, 4, 40
    P = rand_block_params(D, F)
    x, dy = rnd(B, N, D), rnd(B, N, D)
    y, cache = orc.block_fwd(x, P, h, 1e-5)
    dx, G = orc.block_bwd(dy, P, cache)
    Pt = {k: torch.tensor(v, requires_grad=True) for k, v in P.items()}
    xt = torch.tensor(x, requires_grad=True)
    yt = torch_block(xt, Pt, h, 1e-5)
    yt.backward(torch.tensor(dy))
    assert orc.rel_fro(y, yt.detach().numpy()) < 1e-13
    assert orc.rel_fro(dx, xt.grad.numpy()) < 1e-12
    for k in P:
        assert orc.rel_fro(G[k], Pt[k].grad.numpy()) < 1e-12, k


def test_block_fd_every_parameter_and_input():
    B, N, D, h, F = 1, 5, 8, 2, 16          # the tiny shape SURVEY.md §8(c) names
    P = rand_block_params(D, F)
    prm = dict(P)
    prm["x"] = rnd(B, N, D)
    up = rnd(B, N, D)
    f = lambda: float((orc.block_fwd(prm["x"], prm, h, 1e-5)[0] * up).sum())
    y, cache = orc.block_fwd(prm["x"], prm, h, 1e-5)
    dx, G = orc.block_bwd(up, prm, cache)
    ana = dict(G)
    ana["x"] = dx
    fd_check(f, prm, list(ana.keys()), ana)


def test_block_identity_when_output_projections_are_zero():
    B, N, D, h, F = 1, 6, 8, 2, 16
    P = rand_block_params(D, F)
    for k in ("Wproj", "Wfc2", "bproj", "bfc2"):
        P[k] = np.zeros_like(P[k])
    x, dy = rnd(B, N, D), rnd(B, N, D)
    y, cache = orc.block_fwd(x, P, h)
    dx, _ = orc.block_bwd(dy, P, cache)
    assert np.array_equal(y, x) and np.allclose(dx, dy, atol=1e-15)


@pytest.mark.parametrize("T", [1, 2, 4])
def test_sharded_block_equals_unsharded(T):
    B, N, D, h, F = 2, 9, 32, 4, 64
    P = rand_block_params(D, F)
    shards = syn.shard_block_params(P, h, T)
    x, dy = rnd(B, N, D), rnd(B, N, D)
    y, c = orc.block_fwd(x, P, h)
    dx, G = orc.block_bwd(dy, P, c)
    ys, cs = orc.block_fwd_sharded(x, P, shards, h)
    dxs, Gc, Gs = orc.block_bwd_sharded(dy, P, shards, cs)
    assert orc.rel_fro(ys, y) < 1e-13 and orc.rel_fro(dxs, dx) < 1e-13
    Gu = syn.unshard_block_grads(Gs, T)
    for k in Gu:
        assert orc.rel_fro(Gu[k], G[k]) < 1e-12, k
    for k in Gc:
        assert orc.rel_fro(Gc[k], G[k]) < 1e-12, k


# ------------------------------------------------------------------ QK-LayerNorm -
def add_qk_norm_params(P, dh):
    P.update(qn_g=1 + 0.2 * rnd(dh), qn_b=0.1 * rnd(dh), kn_g=1 + 0.2 * rnd(dh), kn_b=0.1 * rnd(dh))
    return P


def torch_block_qknorm(x, P, heads, eps):
    """Textbook block with layer_norm over d_h applied to every head's q and k before the scaled dot product
    (after ref. [8]) from torch library ops in float64 -- test-only cross-check."""
    F_ = torch.nn.functional
    B, N, D = x.shape
    dh = D // heads
    a = F_.layer_norm(x, (D,), P["ln1_g"], P["ln1_b"], eps)
    qkv = a @ P["Wqkv"] + P["bqkv"]
    q, k, v = qkv.split(D, dim=-1)
    sp = lambda t: t.reshape(B, N, heads, dh).transpose(1, 2)
    qn = F_.layer_norm(sp(q), (dh,), P["qn_g"], P["qn_b"], eps)
    kn = F_.layer_norm(sp(k), (dh,), P["kn_g"], P["kn_b"], eps)
    o = F_.scaled_dot_product_attention(qn, kn, sp(v)).transpose(1, 2).reshape(B, N, D)
    x1 = x + o @ P["Wproj"] + P["bproj"]
    m = F_.layer_norm(x1, (D,), P["ln2_g"], P["ln2_b"], eps)
    return x1 + F_.gelu(m @ P["Wfc1"] + P["bfc1"]) @ P["Wfc2"] + P["bfc2"]


def test_qk_norm_block_matches_torch_autograd():
    B, N, D, h, F = 2, 10, 16, 4, 40
    P = add_qk_norm_params(rand_block_params(D, F), D // h)
    x, dy = rnd(B, N, D), rnd(B, N, D)
    y, cache = orc.block_fwd(x, P, h, 1e-5)
    dx, G = orc.block_bwd(dy, P, cache)
    Pt = {k: torch.tensor(v, requires_grad=True) for k, v in P.items()}
    xt = torch.tensor(x, requires_grad=True)
    yt = torch_block_qknorm(xt, Pt, h, 1e-5)
    yt.backward(torch.tensor(dy))
    assert orc.rel_fro(y, yt.detach().numpy()) < 1e-13
    assert orc.rel_fro(dx, xt.grad.numpy()) < 1e-12
    assert set(G) == set(P)
    for k in P:
        if k == "kn_b":     # a bias on the keys shifts every logit of a query row equally: softmax-invariant, so
            assert np.abs(G[k]).max() < 1e-12 and np.abs(Pt[k].grad.numpy()).max() < 1e-12   # d kn_b == 0
        else:
            assert orc.rel_fro(G[k], Pt[k].grad.numpy()) < 1e-12, k
    # and it is not the plain block: dropping the four parameters changes the output
    y0, _ = orc.block_fwd(x, {k: v for k, v in P.items() if k[1:3] != "n_"}, h, 1e-5)
    assert orc.rel_fro(y0, y) > 1e-3


def test_qk_norm_fd_and_invariants():
    B, N, D, h, F = 1, 5, 8, 2, 16
    dh = D // h
    P = add_qk_norm_params(rand_block_params(D, F), dh)
    prm = dict(P)
    prm["x"] = rnd(B, N, D)
    up = rnd(B, N, D)
    f = lambda: float((orc.block_fwd(prm["x"], prm, h, 1e-5)[0] * up).sum())
    y, cache = orc.block_fwd(prm["x"], prm, h, 1e-5)
    dx, G = orc.block_bwd(up, prm, cache)
    ana = dict(G)
    ana["x"] = dx
    fd_check(f, prm, list(ana.keys()), ana)
    # gamma = 1, beta = 0: every normalised q / k has squared norm d_h var/(var+eps) <= d_h, so the scaled
    # logits are bounded by sqrt(d_h) whatever the weights ("the attention logit growth is contained", :114)
    Pb = dict(P)
    Pb["Wqkv"] = P["Wqkv"] * 50.0
    Pb.update(qn_g=np.ones(dh), qn_b=np.zeros(dh), kn_g=np.ones(dh), kn_b=np.zeros(dh))
    _, c = orc.block_fwd(prm["x"], Pb, h, 1e-5)
    Qh, Kh = c["Q"].reshape(B, N, h, dh), c["K"].reshape(B, N, h, dh)
    logits = np.einsum("bnhd,bmhd->bhnm", Qh, Kh) / math.sqrt(dh)
    assert np.abs(logits).max() <= math.sqrt(dh) + 1e-9
    assert np.allclose(Qh.mean(-1), 0, atol=1e-12) and np.all((Qh ** 2).sum(-1) <= dh + 1e-9)
    # eps = 0: rescaling the pre-norm queries (Q columns of Wqkv and bqkv) by c > 0 leaves y unchanged
    P2 = dict(P)
    Wq2, bq2 = P["Wqkv"].copy(), P["bqkv"].copy()
    Wq2[:, :D] *= 7.0
    bq2[:D] *= 7.0
    P2["Wqkv"], P2["bqkv"] = Wq2, bq2
    ya, _ = orc.block_fwd(prm["x"], P, h, 0.0)
    yb, _ = orc.block_fwd(prm["x"], P2, h, 0.0)
    assert orc.rel_fro(yb, ya) < 1e-12


@pytest.mark.parametrize("T", [2, 4])
def test_qk_norm_sharded_block_equals_unsharded(T):
    B, N, D, h, F = 2, 9, 32, 4, 64
    P = add_qk_norm_params(rand_block_params(D, F), D // h)
    shards = syn.shard_block_params(P, h, T)
    x, dy = rnd(B, N, D), rnd(B, N, D)
    y, c = orc.block_fwd(x, P, h)
    dx, G = orc.block_bwd(dy, P, c)
    ys, cs = orc.block_fwd_sharded(x, P, shards, h)
    dxs, Gc, Gs = orc.block_bwd_sharded(dy, P, shards, cs)
    assert orc.rel_fro(ys, y) < 1e-13 and orc.rel_fro(dxs, dx) < 1e-13
    for k in ("qn_g", "qn_b", "kn_g"):
        assert orc.rel_fro(Gc[k], G[k]) < 1e-12, k
    assert np.abs(Gc["kn_b"]).max() < 1e-12 and np.abs(G["kn_b"]).max() < 1e-12      # analytically zero
    Gu = syn.unshard_block_grads(Gs, T)
    for k in Gu:
        assert orc.rel_fro(Gu[k], G[k]) < 1e-12, k


# ------------------------------------------------------------------ aggregation ----------------
def torch_aggregate(tok, P, heads, pos=None):
    """Library cross-check: torch's own multi-head attention with one query token per patch."""
    B, L, V, D = tok.shape
    X = tok.reshape(B * L, V, D).transpose(0, 1)                    # [V, BL, D]
    qq = P["q"].reshape(1, 1, D).expand(1, B * L, D)
    in_w = torch.cat([P["Wq"].T, P["Wk"].T, P["Wv"].T], dim=0)      # torch wants [out, in]
    in_b = torch.cat([P["bq"], P["bk"], P["bv"]])
    out, _ = torch.nn.functional.multi_head_attention_forward(
        qq, X, X, D, heads, in_w, in_b, None, None, False, 0.0, P["Wo"].T, P["bo"],
        need_weights=False)
    out = out.reshape(B, L, D)
    return out if pos is None else out + pos[None]


def test_aggregate_matches_torch_mha_and_autograd():
    B, L, V, D, h = 2, 5, 6, 16, 4
    P = rand_agg_params(D)
    tok, pos, up = rnd(B, L, V, D), rnd(L, D), rnd(B, L, D)
    agg, cache = orc.var_aggregate(tok, P, h, pos)
    dtok, G, dpos = orc.var_aggregate_bwd(up, P, cache, want_dpos=True)
    Pt = {k: torch.tensor(v, requires_grad=True) for k, v in P.items()}
    tt = torch.tensor(tok, requires_grad=True)
    pt = torch.tensor(pos, requires_grad=True)
    ref = torch_aggregate(tt, Pt, h, pt)
    ref.backward(torch.tensor(up))
    assert orc.rel_fro(agg, ref.detach().numpy()) < 1e-13
    assert orc.rel_fro(dtok, tt.grad.numpy()) < 1e-12
    assert orc.rel_fro(dpos, pt.grad.numpy()) < 1e-13
    for k in P:
        if k == "bk":
            assert np.abs(G[k]).max() < 1e-13 and np.abs(Pt[k].grad.numpy()).max() < 1e-13
        else:
            assert orc.rel_fro(G[k], Pt[k].grad.numpy()) < 1e-12, k


def test_aggregate_fd_and_invariants():
    B, L, V, D, h = 1, 3, 3, 8, 2
    prm = rand_agg_params(D)
    prm["tok"] = rnd(B, L, V, D)
    up = rnd(B, L, D)
    f = lambda: float((orc.var_aggregate(prm["tok"], prm, h)[0] * up).sum())
    agg, cache = orc.var_aggregate(prm["tok"], prm, h)
    dtok, G, _ = orc.var_aggregate_bwd(up, prm, cache)
    ana = dict(G)
    ana["tok"] = dtok
    fd_check(f, prm, list(ana.keys()), ana)
    # dbk == 0 ; dbv == sum_{b,l} do
    assert np.abs(G["bk"]).max() < 1e-13
    do = (up @ prm["Wo"].T).reshape(-1, D).sum(0)
    assert np.allclose(G["bv"], do, atol=1e-13)
    # softmax over V: rows sum to 1, sum_v ds_v = 0 is implied by dbk == 0
    assert np.allclose(cache["alpha"].sum(-1), 1, atol=1e-14)
    # permutation of the variables leaves agg unchanged
    perm = RNG.permutation(V)
    agg2, _ = orc.var_aggregate(prm["tok"][:, :, perm], prm, h)
    assert np.allclose(agg, agg2, atol=1e-13)


def test_aggregate_closed_forms():
    B, L, D, h = 2, 4, 8, 2
    P = rand_agg_params(D)
    # V = 1 => agg = (X Wv + bv) Wo + bo, independent of q, Wq, Wk
    tok = rnd(B, L, 1, D)
    agg, _ = orc.var_aggregate(tok, P, h)
    assert np.allclose(agg, (tok[:, :, 0] @ P["Wv"] + P["bv"]) @ P["Wo"] + P["bo"], atol=1e-13)
    # q~ = 0 => uniform alpha => o = mean_v U
    P0 = dict(P)
    P0["q"] = np.zeros(D)
    P0["bq"] = np.zeros(D)
    tok = rnd(B, L, 5, D)
    agg, cache = orc.var_aggregate(tok, P0, h)
    assert np.allclose(cache["alpha"], 1 / 5, atol=1e-15)
    assert np.allclose(agg, (tok.mean(2) @ P["Wv"] + P["bv"]) @ P["Wo"] + P["bo"], atol=1e-13)
    # the collapsed form the CUDA path uses equals the definition:
    #   s_v = X_v . u_a + const, u_a = Wk[:, a] qt_a / sqrt(d_a);  o_a = (sum_v alpha_v X_v) Wv[:, a] + bv[a]
    agg, cache = orc.var_aggregate(tok, P, h)
    da = D // h
    qt = P["q"] @ P["Wq"] + P["bq"]
    o = np.empty((B, L, D))
    for a in range(h):
        c = slice(a * da, (a + 1) * da)
        ua = P["Wk"][:, c] @ qt[c] / math.sqrt(da)
        al = orc.softmax_lastdim(np.einsum("blvd,d->blv", tok, ua))
        xbar = np.einsum("blv,blvd->bld", al, tok)
        o[:, :, c] = xbar @ P["Wv"][:, c] + P["bv"][c]
    assert orc.rel_fro(o @ P["Wo"] + P["bo"], agg) < 1e-13


def test_pixel_space_fused_form_equals_definition():
    """The pixel-space form behind orbit_embed_fused restated here in
    numpy -- G = Wpb Ut, H = Wpb Wv, A_a = alpha_a * pixext, o_a = A_a H_a + bv_a, and the backward chain
    dH, dA, ds, dG, dWpb = dH Wv^T + dG Ut^T -- equals tokenize -> var_aggregate (the definition) and its
    backward to ~1e-13, so a CUDA path built on it is held to the same oracle."""
    B, V, Hg, Wg, p, D, h = 2, 5, 4, 6, 2, 8, 2
    P2, R, da = p * p, p * p + 1, D // h
    x = rnd(B, V, Hg, Wg)
    Wp, bp = rnd(V, P2, D) * 0.5, 0.1 * rnd(V, D)
    P = rand_agg_params(D)
    tok = orc.tokenize(x, Wp, bp, p)
    agg, cache = orc.var_aggregate(tok, P, h)
    dagg = rnd(*agg.shape)
    dtok, Gd, _ = orc.var_aggregate_bwd(dagg, P, cache)
    dWp, dbp = orc.tokenize_bwd(x, dtok, p)
    # ---- fused form ----
    L = (Hg // p) * (Wg // p)
    pix = orc.patches(x, p).transpose(0, 2, 1, 3).reshape(B * L, V, P2)          # [BL, V, p^2]
    pixext = np.concatenate([pix, np.ones((B * L, V, 1))], axis=2)               # [BL, V, R]
    Wpb = np.concatenate([Wp, bp[:, None, :]], axis=1)                           # [V, R, D]
    qt = P["q"] @ P["Wq"] + P["bq"]
    Ut = np.stack([P["Wk"][:, a * da:(a + 1) * da] @ qt[a * da:(a + 1) * da] / math.sqrt(da) for a in range(h)], axis=1)
    Gm = np.einsum("vrd,da->vra", Wpb, Ut)
    H = np.einsum("vrd,dc->vrc", Wpb, P["Wv"])
    s = np.einsum("nvr,vra->nav", pixext, Gm)
    alpha = orc.softmax_lastdim(s)                                               # [BL, h, V]
    assert np.allclose(alpha.reshape(B, L, h, V), cache["alpha"], atol=1e-13)
    A = np.einsum("nav,nvr->navr", alpha, pixext)                                # [BL, h, V, R]
    o = np.concatenate([np.einsum("nvr,vrc->nc", A[:, a], H[:, :, a * da:(a + 1) * da]) for a in range(h)], axis=1) + P["bv"]
    agg2 = (o @ P["Wo"] + P["bo"]).reshape(B, L, D)
    assert orc.rel_fro(agg2, agg) < 1e-13
    # ---- backward ----
    g2 = dagg.reshape(B * L, D)
    do = g2 @ P["Wo"].T
    dH = np.zeros_like(H)
    dA = np.zeros_like(A)
    for a in range(h):
        c = slice(a * da, (a + 1) * da)
        dH[:, :, c] = np.einsum("nvr,nc->vrc", A[:, a], do[:, c])
        dA[:, a] = np.einsum("nc,vrc->nvr", do[:, c], H[:, :, c])
    dalpha = np.einsum("navr,nvr->nav", dA, pixext)
    ds = alpha * (dalpha - (alpha * dalpha).sum(-1, keepdims=True))
    dG = np.einsum("nav,nvr->vra", ds, pixext)
    dWpb = np.einsum("vrc,dc->vrd", dH, P["Wv"]) + np.einsum("vra,da->vrd", dG, Ut)
    assert orc.rel_fro(dWpb[:, :P2], dWp) < 1e-12 and orc.rel_fro(dWpb[:, P2], dbp) < 1e-12
    assert orc.rel_fro(np.einsum("vrd,vrc->dc", Wpb, dH), Gd["Wv"]) < 1e-12
    dUt = np.einsum("vrd,vra->da", Wpb, dG)
    dWk = np.concatenate([np.outer(dUt[:, a], qt[a * da:(a + 1) * da]) / math.sqrt(da) for a in range(h)], axis=1)
    assert orc.rel_fro(dWk, Gd["Wk"]) < 1e-12
    assert orc.rel_fro(do.sum(0), Gd["bv"]) < 1e-12


# ------------------------------------------------------------------ head + wMSE
def rand_head_params(D, C):
    return dict(lnf_g=1 + 0.1 * rnd(D), lnf_b=0.1 * rnd(D), Wh=rnd(D, C) / math.sqrt(D), bh=0.1 * rnd(C))


def test_lat_weights_and_unpatchify():
    for Hg in (4, 32, 128):
        w = orc.lat_weights(Hg)
        assert abs(w.mean() - 1) < 1e-14 and np.allclose(w, w[::-1], atol=1e-14) and w.argmax() in (Hg // 2 - 1, Hg // 2)
        # closed form: sum_i cos((i + 1/2) pi/H - pi/2) = 1 / sin(pi / (2H))  (Dirichlet-kernel sum)
        lat = -90.0 + (np.arange(Hg) + 0.5) * 180.0 / Hg
        assert abs(np.cos(np.deg2rad(lat)).sum() - 1 / math.sin(math.pi / (2 * Hg))) < 1e-9
    # unpatchify is the inverse of `patches` variable by variable, and of patchify_img
    B, V, Hg, Wg, p = 2, 3, 8, 12, 4
    img = rnd(B, V, Hg, Wg)
    P = orc.patchify_img(img, p)
    assert np.array_equal(orc.unpatchify(P, V, Hg, Wg, p), img)
    pix = orc.patches(img, p)                                   # [B, V, L, p^2]
    assert np.array_equal(P.reshape(B, -1, V, p * p), pix.transpose(0, 2, 1, 3))


def test_head_loss_matches_torch_autograd_and_special_cases():
    B, V, Hg, Wg, p, D = 2, 3, 8, 12, 2, 16
    L, C = (Hg // p) * (Wg // p), V * p * p
    Ph = rand_head_params(D, C)
    z, tgt = rnd(B, L, D), rnd(B, V, Hg, Wg)
    loss, pred, cache = orc.head_loss(z, Ph, tgt, p)
    dz, G = orc.head_loss_bwd(Ph, cache)
    F_ = torch.nn.functional
    Pt = {k: torch.tensor(v, requires_grad=True) for k, v in Ph.items()}
    zt = torch.tensor(z, requires_grad=True)
    zn = F_.layer_norm(zt, (D,), Pt["lnf_g"], Pt["lnf_b"], 1e-5)
    Pm = F_.linear(zn, Pt["Wh"].t(), Pt["bh"])
    predt = Pm.reshape(B, Hg // p, Wg // p, V, p, p).permute(0, 3, 1, 4, 2, 5).reshape(B, V, Hg, Wg)
    lat = torch.deg2rad(-90.0 + (torch.arange(Hg, dtype=torch.float64) + 0.5) * 180.0 / Hg)
    w = torch.cos(lat) / torch.cos(lat).mean()
    lt = (w[None, None, :, None] * (predt - torch.tensor(tgt)) ** 2).mean()
    lt.backward()
    assert abs(loss - lt.item()) < 1e-13 * abs(lt.item()) and orc.rel_fro(pred, predt.detach().numpy()) < 1e-13
    assert orc.rel_fro(dz, zt.grad.numpy()) < 1e-12
    for k in Ph:
        assert orc.rel_fro(G[k], Pt[k].grad.numpy()) < 1e-12, k
    # uniform weights: the plain MSE of the harness loss
    l1, pred1, _ = orc.head_loss(z, Ph, tgt, p, latw=np.ones(Hg))
    assert abs(l1 - orc.mse_loss(pred1, tgt)[0]) < 1e-14
    # a perfect prediction has zero loss and zero gradients
    l0, _, c0 = orc.head_loss(z, Ph, pred, p)
    dz0, G0 = orc.head_loss_bwd(Ph, c0)
    assert l0 == 0.0 and np.abs(dz0).max() == 0.0 and all(np.abs(g).max() == 0.0 for g in G0.values())


def test_head_loss_fd():
    B, V, Hg, Wg, p, D = 1, 2, 4, 4, 2, 8
    L, C = (Hg // p) * (Wg // p), V * p * p
    prm = rand_head_params(D, C)
    prm["z"] = rnd(B, L, D)
    tgt = rnd(B, V, Hg, Wg)
    f = lambda: orc.head_loss(prm["z"], prm, tgt, p)[0]
    _, _, cache = orc.head_loss(prm["z"], prm, tgt, p)
    dz, G = orc.head_loss_bwd(prm, cache)
    ana = dict(G)
    ana["z"] = dz
    fd_check(f, prm, list(ana.keys()), ana)


# ------------------------------------------------------------------ whole step -----------------
def test_whole_step_fd_through_everything():
    B, V, Hg, Wg, p, D, h, F = 1, 3, 8, 8, 2, 8, 2, 16     # "B1 V3 8x8 p2 D8 h2 F16"
    L = (Hg // p) * (Wg // p)
    x = rnd(B, V, Hg, Wg)
    emb = dict(Wp=rnd(V, p * p, D) * 0.5, bp=0.1 * rnd(V, D))
    agg = rand_agg_params(D)
    blocks = [rand_block_params(D, F), rand_block_params(D, F)]
    tgt = rnd(B, L, D)
    f = lambda: orc.step(x, emb, agg, blocks, tgt, p, h)["loss"]
    out = orc.step(x, emb, agg, blocks, tgt, p, h)
    fd_check(f, emb, ["Wp", "bp"], dict(Wp=out["dWp"], bp=out["dbp"]), tol=2e-6)
    fd_check(f, agg, ["q", "Wq", "Wk", "Wv", "Wo", "bq", "bv", "bo"], out["agg_grads"], tol=2e-6)
    fd_check(f, blocks[0], list(blocks[0].keys()), out["block_grads"][0], tol=2e-6, nsamp=3)
    fd_check(f, blocks[1], list(blocks[1].keys()), out["block_grads"][1], tol=2e-6, nsamp=3)


def test_bf16_rounding_helper():
    a = np.array([1.0, 1.00390625, 1.01171875, -3.3, 65504.0, 1e-30], dtype=np.float32)
    r = syn.round_bf16(a)
    ref = torch.tensor(a, dtype=torch.float32).to(torch.bfloat16).to(torch.float32).numpy()
    assert np.array_equal(r, ref)


# ------------------------------------------------------------------ sampled-output helpers -----
def test_sampled_helpers_equal_slices_of_full_functions():
    """block_sampled / tokenize_patches (used by the full-size GPU tests) are slices of the full definitions;
    attention with a query subset equals the rows of the full attention."""
    B, N, D, h, F = 2, 12, 16, 4, 40
    P = rand_block_params(D, F)
    x, dy = rnd(B, N, D), rnd(B, N, D)
    y, cache = orc.block_fwd(x, P, h, 1e-5)
    dx, G = orc.block_bwd(dy, P, cache)
    rows, fcols = np.array([0, 5, 11]), np.array([1, 7, 39])
    s = orc.block_sampled(x, dy, P, h, 1e-5, rows, fcols)
    assert orc.rel_fro(s["y_rows"], y[:, rows]) < 1e-13
    assert orc.rel_fro(s["x1"], cache["x1"]) < 1e-14
    assert orc.rel_fro(s["bfc2"], G["bfc2"]) < 1e-13
    assert orc.rel_fro(s["Wfc2_rows"], G["Wfc2"][fcols]) < 1e-13
    assert orc.rel_fro(s["Wfc1_cols"], G["Wfc1"][:, fcols]) < 1e-13
    assert orc.rel_fro(s["bfc1_cols"], G["bfc1"][fcols]) < 1e-13
    Q, K, V = rnd(B, N, D), rnd(B, N, D), rnd(B, N, D)
    O, _ = orc.attention(Q, K, V, h)
    Os, _ = orc.attention(Q[:, rows], K, V, h)
    assert np.allclose(Os, O[:, rows], atol=1e-14)
    xf = rnd(2, 3, 8, 12)
    Wp, bp = rnd(3, 4, 5), rnd(3, 5)
    ls = np.array([0, 7, 23])
    assert np.array_equal(orc.tokenize_patches(xf, Wp, bp, 2, ls), orc.tokenize(xf, Wp, bp, 2)[:, ls])


def test_patch_chunked_front_end_equals_whole_tensor_functions():
    """tests/parity.front_oracle_chunked (the full-size C3 GPU tests: oracle front end accumulated over chunks of
    patches, oracle/ functions only) equals tokenize -> var_aggregate -> var_aggregate_bwd -> tokenize_bwd on the
    whole tensors: agg, dpos assembled by patch, every parameter gradient summed over the chunks (ragged last chunk)."""
    import parity
    B, V, Hg, Wg, p, D, h = 2, 3, 8, 12, 2, 8, 2
    L = (Hg // p) * (Wg // p)
    x = rnd(B, V, Hg, Wg)
    emb = {"Wp": rnd(V, p * p, D), "bp": rnd(V, D)}
    A = rand_agg_params(D)
    pos, dagg = rnd(L, D), rnd(B, L, D)
    tok = orc.tokenize(x, emb["Wp"], emb["bp"], p)
    agg, cache = orc.var_aggregate(tok, A, h, pos)
    dtok, G, dpos = orc.var_aggregate_bwd(dagg, A, cache, want_dpos=True)
    dWp, dbp = orc.tokenize_bwd(x, dtok, p)
    agg_c, dWp_c, dbp_c, G_c, dpos_c = parity.front_oracle_chunked(orc, x, emb, A, dagg, p, h, 5, pos=pos)
    assert orc.rel_fro(agg_c, agg) < 1e-14 and orc.rel_fro(dpos_c, dpos) < 1e-14
    assert orc.rel_fro(dWp_c, dWp) < 1e-13 and orc.rel_fro(dbp_c, dbp) < 1e-13
    for k in G:
        if k == "bk":
            assert np.abs(G_c[k]).max() < 1e-12
        else:
            assert orc.rel_fro(G_c[k], G[k]) < 1e-13, k
    # tokenize_bwd_patches over one chunk is the restriction of tokenize_bwd's sums to those patches
    ls = np.array([1, 4, 9])
    w, b = orc.tokenize_bwd_patches(x, dtok[:, ls], p, ls)
    pix = orc.patches(x, p)
    assert np.allclose(b, dtok[:, ls].sum(axis=(0, 1)), atol=1e-13)
    assert np.allclose(w[1, 2], np.einsum("bs,bsd->d", pix[:, 1, ls, 2], dtok[:, ls, 1, :]), atol=1e-13)


class _LockstepGroup:
    """Plain-Python stand-in for an all-reduce over T ranks run as T threads: every rank deposits its partial, a barrier,
    every rank reads the sum (ranks added in rank order)."""

    def __init__(self, T):
        import threading
        self.T, self.slots, self.bar = T, [None] * T, threading.Barrier(T)

    def allreduce(self, rank):
        def f(part):
            self.slots[rank] = part
            self.bar.wait()
            total = sum(self.slots[1:], self.slots[0])
            self.bar.wait()
            return total
        return f


@pytest.mark.parametrize("T", [1, 2, 4])
@pytest.mark.parametrize("qk_norm", [False, True])
def test_rank_local_program_equals_unsharded_block(T, qk_norm):
    """RANK (oracle rank_block_fwd / rank_block_bwd: one rank's program between the four all-reduces)
    run for all T ranks in lock step = the unsharded BLK oracle: y, dx, replicated-parameter gradients identical on every
    rank, shard gradients = the column / row slices of the unsharded gradients, partials sum to the combined products."""
    import threading
    B, N, D, h, F = 2, 6, 16, 4, 32
    P = rand_block_params(D, F)
    if qk_norm:
        dh = D // h
        P.update(qn_g=1 + 0.1 * rnd(dh), qn_b=0.1 * rnd(dh), kn_g=1 + 0.1 * rnd(dh), kn_b=0.1 * rnd(dh))
    x, dy = rnd(B, N, D), rnd(B, N, D)
    y, cache = orc.block_fwd(x, P, h, 1e-5)
    dx, G = orc.block_bwd(dy, P, cache)
    shards = syn.shard_block_params(P, h, T)
    grp = _LockstepGroup(T)
    res = [None] * T

    def run(k):
        yk, ck, pf = orc.rank_block_fwd(x, P, shards[k], h // T, grp.allreduce(k), 1e-5)
        dxk, Gc, Gs, pb = orc.rank_block_bwd(dy, P, shards[k], ck, grp.allreduce(k))
        res[k] = (yk, dxk, Gc, Gs, pf, pb)
    ts = [threading.Thread(target=run, args=(k,)) for k in range(T)]
    [t.start() for t in ts]
    [t.join() for t in ts]
    for k in range(T):
        yk, dxk, Gc, Gs, pf, pb = res[k]
        assert orc.rel_fro(yk, y) < 1e-13 and orc.rel_fro(dxk, dx) < 1e-12
        for name in ("ln1_g", "ln1_b", "ln2_g", "ln2_b", "bproj", "bfc2"):
            assert orc.rel_fro(Gc[name], G[name]) < 1e-12, name
    Gu = syn.unshard_block_grads([r[3] for r in res], T)
    for name in Gu:
        assert orc.rel_fro(Gu[name], G[name]) < 1e-12, name
    if qk_norm:      # shared by the heads: each rank holds the sum over ITS heads
        for name in ("qn_g", "qn_b", "kn_g"):
            assert orc.rel_fro(sum(r[2][name] for r in res), G[name]) < 1e-12, name
    # what the collectives see: the partials add up to the unsharded products (Eq. 2 forward, Eq. 3 backward)
    assert orc.rel_fro(sum(r[4]["proj"] for r in res), cache["O"] @ P["Wproj"]) < 1e-13
    assert orc.rel_fro(sum(r[4]["fc2"] for r in res), cache["g"] @ P["Wfc2"]) < 1e-13


# ------------------------------------------------------------------ dynamic gradient scaling -----
def test_grad_scale_schedule_golden_trace_and_torch():
    """grad_scale_update against the hand-worked trace (tests/golden/grad_scale_trace.json) and against torch's CPU
    implementation of the mechanism the paper cites (torch._amp_update_scale_)."""
    tr = json.load(open(os.path.join(GOLD, "grad_scale_trace.json")))
    s, t = tr["scale0"], 0
    ts, tt = torch.tensor([tr["scale0"]], dtype=torch.float32), torch.zeros(1, dtype=torch.int32)
    for f, s_want, t_want in zip(tr["found_inf"], tr["scale_after"], tr["tracker_after"]):
        s, t = orc.grad_scale_update(s, t, float(f), tr["growth_factor"], tr["backoff_factor"], tr["growth_interval"])
        assert s == s_want and t == t_want
        torch._amp_update_scale_(ts, tt, torch.tensor([float(f)]), tr["growth_factor"], tr["backoff_factor"], tr["growth_interval"])
        assert float(ts) == s and int(tt) == t


def test_grads_unscale_check_and_accumulate():
    """Unscaling by a power of two is exact (= ldexp); overflow detection fires on Inf and NaN only; equals torch's
    _amp_foreach_non_finite_check_and_unscale_ on CPU; accumulation of k micro-steps of g with scale S = k g / S."""
    gs = [rnd(5, 7) * 1e3, rnd(11) * 1e-3, rnd(2, 3, 4)]
    out, found = orc.grads_unscale_check(gs, 1024.0)
    assert found == 0.0
    for o, g in zip(out, gs):
        assert np.array_equal(o, np.ldexp(g, -10))
    tg = [torch.tensor(g, dtype=torch.float64) for g in gs]
    tf = torch.zeros(1, dtype=torch.float32)
    torch._amp_foreach_non_finite_check_and_unscale_(tg, tf, torch.tensor([1.0 / 1024.0], dtype=torch.float32))
    assert float(tf) == 0.0
    for o, g in zip(out, tg):
        assert np.array_equal(o, g.numpy())
    for bad in (np.inf, -np.inf, np.nan):
        g2 = [g.copy() for g in gs]
        g2[1][3] = bad
        _, found = orc.grads_unscale_check(g2, 3.0)
        assert found == 1.0
        tg = [torch.tensor(g, dtype=torch.float64) for g in g2]
        tf = torch.zeros(1, dtype=torch.float32)
        torch._amp_foreach_non_finite_check_and_unscale_(tg, tf, torch.tensor([1.0 / 3.0], dtype=torch.float32))
        assert float(tf) == 1.0
    acc = [np.zeros_like(g) for g in gs]
    for _ in range(4):
        acc = orc.grads_accumulate(acc, gs, 8.0)
    for a, g in zip(acc, gs):
        assert np.allclose(a, 4 * g / 8.0, rtol=1e-15)
