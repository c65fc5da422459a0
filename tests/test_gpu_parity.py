"""GPU parity: the CUDA path (through the C-ABI via paper_2404_14712_b200.binding) against the fp64 oracle,
element by element on the same seeded inputs.  Tolerances (north_star): relative Frobenius error <= 1e-2 for
bf16 paths, <= 1e-4 for fp32 and for the fp32 shard-recombination check.
"""
import math

import numpy as np
import pytest
import torch

import parity
from oracle import orbit_oracle as orc
from paper_2404_14712_b200 import inputs as syn

pytestmark = pytest.mark.gpu

TOL = {"f32": 1e-4, "bf16": 1e-2}


@pytest.fixture(scope="module")
def ob():
    from paper_2404_14712_b200 import binding
    return binding


@pytest.fixture(scope="module")
def rn():
    from paper_2404_14712_b200 import runner
    return runner


def check(name, got, ref, tol):
    """relative Frobenius error <= tol AND the element-wise bound of tests/parity.py."""
    return parity.check(name, got, ref, tol)


def make_block_case(seed, B, N, D, heads, F, T, dtype, resid_dtype):
    P = syn.block_params(seed, D, F, dtype)
    shards = syn.shard_block_params(P, heads, T)
    x = syn.normal(seed, "blk.x", (B, N, D), dtype=resid_dtype)
    dy = syn.normal(seed, "blk.dy", (B, N, D), dtype=resid_dtype)
    return P, shards, x, dy


def run_block(rn, B, N, D, heads, F, T, dtype, resid_dtype, P, shards, x, dy, recompute=False):
    br = rn.BlockRunner(B, N, D, heads, F, T, dtype, resid_dtype, P, shards, recompute=recompute)
    xd, dyd = rn.to_dev(x, resid_dtype), rn.to_dev(dy, resid_dtype)
    y = br.fwd(xd)
    dx = br.bwd(dyd)
    torch.cuda.synchronize()
    return br, y, dx


def compare_block(br, y, dx, P, x, dy, heads, T, tol, eps=1e-5):
    yo, cache = orc.block_fwd(x, P, heads, eps)
    dxo, G = orc.block_bwd(dy, P, cache)
    errs = {"y": check("y", y, yo, tol), "dx": check("dx", dx, dxo, tol)}
    for k in br.COMMON:
        errs[k] = check("d" + k, br.gcommon[k], G[k], tol)
    if br.qk_norm:
        for k in ("qn_g", "qn_b", "kn_g"):
            errs[k] = check("d" + k, br.gcommon[k], G[k], tol)
        got = br.gcommon["kn_b"].detach().to(torch.float32).cpu().numpy()        # analytically zero (softmax shift invariance)
        assert np.abs(got).max() <= tol * max(1e-6, np.abs(G["qn_b"]).max()), "d kn_b must vanish"
    gs = [{k: v.detach().to(torch.float32).cpu().numpy() for k, v in S.items()} for S in br.gshards]
    Gu = syn.unshard_block_grads(gs, T)
    for k in Gu:
        errs[k] = check("d" + k, Gu[k], G[k], tol)
    return errs


# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("T", [1, 2, 4, 8])      # T = 8: more bias-gradient segments than the one-launch tail of the backward takes
def test_block_fp32_shard_recombination(rn, T):
    """fp32 shard-recombination check (north_star; R15): sharded CUDA block (fp32 storage, true fp32
    FMA, fp32 partials) vs the UNSHARDED fp64 oracle, <= 1e-4."""
    B, N, D, heads, F = 2, 256, 256, 8, 1024
    P, shards, x, dy = make_block_case(11, B, N, D, heads, F, T, "f32", "f32")
    br, y, dx = run_block(rn, B, N, D, heads, F, T, "f32", "f32", P, shards, x, dy)
    compare_block(br, y, dx, P, x, dy, heads, T, 1e-4)


def test_block_fp32_c1_shape_ragged_tokens(rn):
    """C1's block shape with a ragged token count (N = 100 is not a multiple of any tile)."""
    B, N, D, heads, F = 2, 100, 128, 4, 512
    P, shards, x, dy = make_block_case(12, B, N, D, heads, F, 1, "f32", "f32")
    br, y, dx = run_block(rn, B, N, D, heads, F, 1, "f32", "f32", P, shards, x, dy)
    compare_block(br, y, dx, P, x, dy, heads, 1, 1e-4)


def test_block_softmax_stress_logits_x30(rn):
    """Logits scaled x30 exercise the max-subtraction path."""
    B, N, D, heads, F = 1, 96, 64, 2, 128
    P, shards, x, dy = make_block_case(13, B, N, D, heads, F, 1, "f32", "f32")
    P["Wqkv"] = (P["Wqkv"] * np.float32(math.sqrt(30.0) * 3)).astype(np.float32)
    shards = syn.shard_block_params(P, heads, 1)
    br, y, dx = run_block(rn, B, N, D, heads, F, 1, "f32", "f32", P, shards, x, dy)
    compare_block(br, y, dx, P, x, dy, heads, 1, 2e-4)


@pytest.mark.parametrize("dh", [64, 128])
def test_block_bf16_runaway_logits_stay_finite(rn, dh):
    """Runaway attention logits (the regime QK-LayerNorm targets) on the tcgen05 attention path: logits of
    order 1e5 (beyond an int16 row-max reference in log2 units) must give finite y / dx / gradients, as on every other
    path.  No oracle comparison: at this magnitude the softmax is an arg-max decided by the bf16 rounding of q and k
    (one ulp of a logit is ~4e2), so only the property is checked."""
    B, N, heads, F = 1, 256, 2, 256
    D = heads * dh
    P, shards, x, dy = make_block_case(15, B, N, D, heads, F, 1, "bf16", "bf16")
    def max_logit(Wm):          # harness-side magnitude estimate (LN1 keeps the rows at unit scale)
        qkv = x.reshape(-1, D).astype(np.float64) @ Wm.astype(np.float64)
        return np.abs(qkv[:, :dh] @ qkv[:, D:D + dh].T).max() / math.sqrt(dh)
    W = P["Wqkv"].copy()
    W[:, :2 * D] *= np.float32(math.sqrt(1e5 / max_logit(W)))                             # |q.k| / sqrt(d_h) ~ 1e5
    P["Wqkv"] = syn.round_storage(W, "bf16")
    shards = syn.shard_block_params(P, heads, 1)
    br, y, dx = run_block(rn, B, N, D, heads, F, 1, "bf16", "bf16", P, shards, x, dy)
    big = max_logit(P["Wqkv"])
    assert big > 4e4, big                                 # log2 units: > 5.7e4, past the int16 range
    assert torch.isfinite(y.float()).all() and torch.isfinite(dx.float()).all()
    for k in br.SHARD:
        assert torch.isfinite(br.gshards[0][k].float()).all(), k


@pytest.mark.parametrize("shape", [
    (2, 384, 512, 8, 2048, 1, "bf16"),      # several 128x256 tiles, d_h = 64
    (1, 200, 256, 2, 1024, 1, "f32"),       # d_h = 128, ragged N, fp32 residual stream
    (2, 256, 512, 4, 1536, 2, "bf16"),      # Hybrid-STOP T = 2, d_h = 128
    (1, 520, 1024, 8, 4096, 4, "f32"),      # T = 4, ragged N spanning tile tails
])
def test_block_bf16_vs_oracle(rn, shape):
    B, N, D, heads, F, T, rdt = shape
    P, shards, x, dy = make_block_case(21, B, N, D, heads, F, T, "bf16", rdt)
    br, y, dx = run_block(rn, B, N, D, heads, F, T, "bf16", rdt, P, shards, x, dy)
    errs = compare_block(br, y, dx, P, x, dy, heads, T, 1e-2)
    print("bf16 block errs", {k: f"{v:.2e}" for k, v in errs.items()})


@pytest.mark.parametrize("shape", [
    (1, 384, 768, 4, 1536, 1, "bf16"),      # d_h 192 (113B and 1B rows), three 128-row tiles
    (2, 200, 512, 2, 1024, 1, "f32"),       # d_h 256 (10B row), ragged N (one full + one partial query tile; 7 key tiles of 32)
    (1, 520, 768, 4, 1536, 2, "bf16"),      # d_h 192, Hybrid-STOP T = 2, ragged N spanning tile tails
    (1, 333, 1024, 4, 2048, 1, "bf16"),     # d_h 256, odd N: ragged 64-key / 32-row tiles, dK/dV computed in two column slices
])
@pytest.mark.parametrize("qkn", [False, True])
def test_block_bf16_paper_head_widths(rn, shape, qkn):
    """The paper's own head widths d_h = 192 and 256 on the tcgen05 attention path (64-row key tiles
    forward, 32-row streamed tiles backward), with and without QK-LayerNorm."""
    B, N, D, heads, F, T, rdt = shape
    P, shards, x, dy = make_block_case(23, B, N, D, heads, F, T, "bf16", rdt)
    if qkn:
        P.update(syn.qk_norm_params(23, D // heads, "bf16"))
    br, y, dx = run_block(rn, B, N, D, heads, F, T, "bf16", rdt, P, shards, x, dy)
    errs = compare_block(br, y, dx, P, x, dy, heads, T, 1e-2)
    print("paper head widths", shape, qkn, {k: f"{v:.2e}" for k, v in errs.items()})


@pytest.mark.parametrize("T", [1, 2])
def test_block_qk_norm_fp32(rn, T):
    """QK-LayerNorm (ORBIT_QK_NORM) in fp32, d_h = 32, also sharded: <= 1e-4 vs the unsharded oracle."""
    B, N, D, heads, F = 2, 100, 128, 4, 256
    P, shards, x, dy = make_block_case(14, B, N, D, heads, F, T, "f32", "f32")
    P.update(syn.qk_norm_params(14, D // heads, "f32"))
    br, y, dx = run_block(rn, B, N, D, heads, F, T, "f32", "f32", P, shards, x, dy)
    compare_block(br, y, dx, P, x, dy, heads, T, 1e-4)


@pytest.mark.parametrize("shape", [
    (2, 384, 512, 8, 1024, 1, "bf16"),      # d_h = 64 on the tcgen05 attention path
    (1, 200, 256, 2, 512, 1, "f32"),        # d_h = 128, ragged N
    (2, 256, 512, 4, 1024, 2, "bf16"),      # Hybrid-STOP T = 2, d_h = 128: gamma / beta grads summed over shards
])
@pytest.mark.parametrize("recompute", [False, True])
def test_block_qk_norm_bf16(rn, shape, recompute):
    B, N, D, heads, F, T, rdt = shape
    P, shards, x, dy = make_block_case(22, B, N, D, heads, F, T, "bf16", rdt)
    P.update(syn.qk_norm_params(22, D // heads, "bf16"))
    br, y, dx = run_block(rn, B, N, D, heads, F, T, "bf16", rdt, P, shards, x, dy, recompute=recompute)
    errs = compare_block(br, y, dx, P, x, dy, heads, T, 1e-2)
    print("qk-norm bf16 errs", {k: f"{v:.2e}" for k, v in errs.items()})


def test_block_recompute_matches_and_saves_memory(ob, rn):
    """ORBIT_RECOMPUTE (activation checkpointing): same outputs / gradients as the stored-activation
    path within tolerance of the oracle, with `saved` reduced to the block input."""
    B, N, D, heads, F, T = 2, 320, 512, 8, 2048, 1
    P, shards, x, dy = make_block_case(23, B, N, D, heads, F, T, "bf16", "bf16")
    br, y, dx = run_block(rn, B, N, D, heads, F, T, "bf16", "bf16", P, shards, x, dy, recompute=True)
    compare_block(br, y, dx, P, x, dy, heads, T, 1e-2)
    d0 = ob.block_desc(B, N, D, heads, F, T, 1e-5, "bf16", "bf16", 0)
    assert ob.orbit_block_saved_bytes(br.desc) == B * N * D * 2
    assert ob.orbit_block_saved_bytes(br.desc) * 8 < ob.orbit_block_saved_bytes(d0)
    br0, y0, dx0 = run_block(rn, B, N, D, heads, F, T, "bf16", "bf16", P, shards, x, dy)
    assert torch.equal(y, y0) and torch.equal(br.gshards[0]["Wfc1"], br0.gshards[0]["Wfc1"])


def test_chain_eq2_eq3(ob, rn):
    """Bare Eq. (2)/(3) chain on the GPU in fp32: sum_k (x A_k) B_k vs x A B in fp64."""
    m, d, n, e, T = 300, 256, 512, 192, 4
    x = syn.normal(31, "ch.x", (m, d))
    A = syn.xavier_uniform(31, "ch.A", (d, n), d, n)
    Bm = syn.xavier_uniform(31, "ch.B", (n, e), n, e)
    dy = syn.normal(31, "ch.dy", (m, e))
    Ac = [np.ascontiguousarray(A[:, k * n // T:(k + 1) * n // T]) for k in range(T)]
    Br = [np.ascontiguousarray(Bm[k * n // T:(k + 1) * n // T]) for k in range(T)]
    Ad = [rn.to_dev(a, "f32") for a in Ac]
    Bd = [rn.to_dev(b, "f32") for b in Br]
    ws = torch.empty(ob.orbit_chain_workspace_bytes(m, d, n, e, T, "f32"), dtype=torch.uint8, device="cuda")
    y = torch.empty(m, e, device="cuda", dtype=torch.float32)
    dx = torch.empty(m, d, device="cuda", dtype=torch.float32)
    ob.orbit_chain_fwd(m, d, n, e, T, "f32", rn.to_dev(x, "f32"), Ad, Bd, y, ws)
    ob.orbit_chain_bwd(m, d, n, e, T, "f32", rn.to_dev(dy, "f32"), Ad, Bd, dx, ws)
    torch.cuda.synchronize()
    x64, A64, B64, dy64 = (np.asarray(t, dtype=np.float64) for t in (x, A, Bm, dy))
    check("chain y", y, x64 @ A64 @ B64, 1e-4)
    check("chain dx", dx, dy64 @ B64.T @ A64.T, 1e-4)
    check("chain y vs sharded oracle", y, orc.chain_sharded(x, Ac, Br), 1e-4)


# ---------------------------------------------------------------------------------------------------------
def make_step_case(cfg, seed, depth=None):
    depth = cfg.depth if depth is None else depth
    emb = syn.embed_params(seed, cfg.V, cfg.p, cfg.D, cfg.dtype)
    agg = syn.agg_params(seed, cfg.D, cfg.dtype)
    blocks = [syn.block_params(seed, cfg.D, cfg.F, cfg.dtype, tag=f"blk{i}") for i in range(depth)]
    x = syn.fields(seed, cfg.B, cfg.V, cfg.Hg, cfg.Wg, per_variable_scale=cfg.name != "C1")
    tgt = syn.normal(seed, "target", (cfg.B, cfg.L, cfg.D), dtype=cfg.resid_dtype)
    pos = syn.normal(seed, "pos", (cfg.L, cfg.D), 0.02, dtype=cfg.resid_dtype)
    return emb, agg, blocks, x, tgt, pos


def run_and_compare_step(rn, cfg, seed, tol, with_pos=True, fused=False):
    """fused=True runs the front end through orbit_embed_fused(_bwd) (pixel-space form, no tok / dtok); its
    outputs are held to the same oracle (tokenize -> var_aggregate and their backward)."""
    emb, agg, blocks, x, tgt, pos = make_step_case(cfg, seed)
    if not with_pos:
        pos = None
    sr = rn.StepRunner(cfg, emb, agg, [(P, syn.shard_block_params(P, cfg.heads, 1)) for P in blocks], pos,
                       fused_front=fused)
    loss = sr.step(rn.to_dev(x, "f32"), rn.to_dev(tgt, cfg.resid_dtype))
    torch.cuda.synchronize()
    out = orc.step(x, emb, agg, blocks, tgt, cfg.p, cfg.heads, cfg.ln_eps, pos)
    errs = {}
    if not fused:
        errs["tok"] = check("tok", sr.front.tok, out["tok"], tol)
    errs["agg"] = check("agg", sr.front.out, out["agg"], tol)
    errs["y"] = check("y", sr.blocks[-1].y, out["y"], tol)
    assert abs(float(loss.item()) - out["loss"]) <= 5 * tol * abs(out["loss"])
    for i, br in enumerate(sr.blocks):
        G = out["block_grads"][i]
        for k in br.COMMON:
            errs[f"b{i}.{k}"] = check(f"b{i}.d{k}", br.gcommon[k], G[k], tol)
        for k in br.SHARD:
            errs[f"b{i}.{k}"] = check(f"b{i}.d{k}", br.gshards[0][k], G[k], tol)
    errs["dagg"] = check("dagg", sr.blocks[0].dx, out["dagg"], tol)
    if not fused:
        errs["dtok"] = check("dtok", sr.front.dtok, out["dtok"], tol)
    for k, g in out["agg_grads"].items():
        if k == "bk":   # analytically zero: compare absolutely against the scale of its siblings
            got = rn.to_np(sr.front.gagg[k])
            assert np.abs(got).max() <= 1e-6 * max(1.0, np.abs(out["agg_grads"]["bv"]).max())
        else:
            errs["agg." + k] = check("agg.d" + k, sr.front.gagg[k], g, tol)
    if pos is not None:
        errs["dpos"] = check("dpos", sr.front.dpos, out["dpos"], tol)
    errs["dWp"] = check("dWp", sr.front.dWp, out["dWp"], tol)
    errs["dbp"] = check("dbp", sr.front.dbp, out["dbp"], tol)
    return errs


def test_c1_full_step_fp32(rn):
    """BASELINE.json config 1 (tiny ORBIT step, fp32): tokenise + aggregate + block fwd+bwd + MSE, <= 1e-4."""
    errs = run_and_compare_step(rn, syn.CONFIGS["C1"], syn.seed_of("C1"), 1e-4)
    print("C1 max err", max(errs.values()))


def test_small_bf16_full_step(rn):
    """A shrunken C2 (bf16 storage, fp32 residual stream, V = 7 variables, patch 2, depth 2), <= 1e-2."""
    cfg = syn.Config("S2", B=2, V=7, Hg=16, Wg=32, p=2, D=256, heads=4, F=1024, depth=2, dtype="bf16",
                     resid_dtype="f32")
    errs = run_and_compare_step(rn, cfg, 42, 1e-2)
    print("S2 errs", {k: f"{v:.2e}" for k, v in errs.items()})


def test_front_end_v91_ragged(rn):
    """Front end with V = 91 (odd, > 64), patch 4, no positional embedding, bf16 stream."""
    cfg = syn.Config("S3", B=1, V=91, Hg=16, Wg=24, p=4, D=128, heads=16, F=256, depth=1, dtype="bf16",
                     resid_dtype="bf16")
    run_and_compare_step(rn, cfg, 43, 1e-2, with_pos=False)


def test_c1_full_step_fp32_fused_front(rn):
    """C1 with the pixel-space fused front end (orbit_embed_fused), fp32: <= 1e-4 against the two-step oracle."""
    errs = run_and_compare_step(rn, syn.CONFIGS["C1"], syn.seed_of("C1"), 1e-4, fused=True)
    print("C1 fused max err", max(errs.values()))


@pytest.mark.parametrize("with_pos", [True, False])
def test_small_bf16_full_step_fused_front(rn, with_pos):
    cfg = syn.Config("S2", B=2, V=7, Hg=16, Wg=32, p=2, D=256, heads=4, F=1024, depth=2, dtype="bf16",
                     resid_dtype="f32")
    errs = run_and_compare_step(rn, cfg, 42, 1e-2, with_pos=with_pos, fused=True)
    print("S2 fused errs", {k: f"{v:.2e}" for k, v in errs.items()})


@pytest.mark.parametrize("case", [
    dict(B=1, V=91, Hg=16, Wg=24, p=4, D=128, heads=16, rd="bf16"),     # V odd and > 64 (two variable pairs per lane)
    dict(B=3, V=48, Hg=12, Wg=20, p=2, D=256, heads=16, rd="bf16"),     # C2-like V, ragged patch count (BL = 180)
    dict(B=2, V=5, Hg=6, Wg=10, p=1, D=64, heads=8, rd="f32"),          # patch 1, tiny
    dict(B=1, V=128, Hg=8, Wg=8, p=4, D=128, heads=2, rd="f32"),        # V at the limit
])
def test_front_end_fused_shapes(rn, case):
    cfg = syn.Config("SF", B=case["B"], V=case["V"], Hg=case["Hg"], Wg=case["Wg"], p=case["p"], D=case["D"],
                     heads=case["heads"], F=2 * case["D"], depth=1, dtype="bf16", resid_dtype=case["rd"])
    errs = run_and_compare_step(rn, cfg, 44, 1e-2, with_pos=False, fused=True)
    print("fused front", case, {k: f"{v:.2e}" for k, v in errs.items() if not k.startswith("b0")})


@pytest.mark.parametrize("case", [
    dict(B=1, V=128, Hg=8, Wg=8, p=4, D=128, heads=2, rd="f32"),        # V at the limit of the TMA-fed kernels, 2 heads of 16
    dict(B=3, V=48, Hg=24, Wg=20, p=2, D=256, heads=16, rd="bf16"),     # BL = 360: 2-3 patches per CTA through one ring
    dict(B=2, V=5, Hg=6, Wg=10, p=1, D=128, heads=8, rd="f32"),         # patch 1, V < 16 (one row tile, 11 zero rows)
    dict(B=5, V=17, Hg=16, Wg=16, p=2, D=384, heads=12, rd="bf16"),     # odd chunk count (D = 6 x 64), V = 16 + 1, BL = 320
    dict(B=1, V=9, Hg=8, Wg=8, p=2, D=4096, heads=16, rd="bf16"),       # widest D of the TMA kernels: the [16][D] dUt accumulator fills
                                                                        # all 512 TMEM columns (64 chunks x 4 columns x 2 warps per quarter)
    dict(B=2, V=6, Hg=12, Wg=20, p=2, D=192, heads=4, rd="bf16"),       # tcgen05 tokeniser with an odd number of 64-column boxes (the last
                                                                        # 128-column group is half loaded); SIMT aggregation (D % 128 != 0)
    dict(B=3, V=3, Hg=20, Wg=28, p=4, D=64, heads=4, rd="f32"),         # one 64-column box, p = 4, B L = 105 (one ragged stage)
])
def test_front_end_twocall_shapes(rn, case):
    """orbit_tokenize + orbit_var_aggregate (+ backward) on the tensor-core / TMA kernels over edge shapes, <= 1e-2."""
    cfg = syn.Config("ST", B=case["B"], V=case["V"], Hg=case["Hg"], Wg=case["Wg"], p=case["p"], D=case["D"],
                     heads=case["heads"], F=2 * case["D"], depth=1, dtype="bf16", resid_dtype=case["rd"])
    errs = run_and_compare_step(rn, cfg, 47, 1e-2, with_pos=False, fused=False)
    print("two-call front", case, {k: f"{v:.2e}" for k, v in errs.items() if not k.startswith("b0")})


def test_front_end_fused_fp32_shapes(rn):
    """fp32 storage (SIMT GEMMs, strided batch over heads) on an odd shape: <= 1e-4."""
    cfg = syn.Config("SF32", B=2, V=9, Hg=8, Wg=12, p=2, D=64, heads=4, F=128, depth=1, dtype="f32", resid_dtype="f32")
    run_and_compare_step(rn, cfg, 45, 1e-4, fused=True)


@pytest.mark.parametrize("case", [
    dict(name="C1", fused=False, tol=1e-4),
    dict(name="C1", fused=True, tol=1e-4),
    dict(name="S2", fused=True, tol=1e-2),
])
def test_full_step_with_head_and_wmse(rn, case):
    """The paper's training step (NEXT-3): ... -> blocks -> final LayerNorm -> image-space head -> latitude-weighted MSE
    (PAPER.md:46, :169), forward + backward through everything, against orc.step_head."""
    if case["name"] == "C1":
        cfg, seed = syn.CONFIGS["C1"], syn.seed_of("C1")
    else:
        cfg, seed = syn.Config("S2", B=2, V=6, Hg=16, Wg=32, p=2, D=256, heads=4, F=1024, depth=2, dtype="bf16",
                               resid_dtype="f32"), 46
    tol = case["tol"]
    emb, agg, blocks, x, _, pos = make_step_case(cfg, seed)
    head = syn.head_params(seed, cfg.D, cfg.V, cfg.p, cfg.dtype)
    timg = syn.fields(seed + 7, cfg.B, cfg.V, cfg.Hg, cfg.Wg, per_variable_scale=False)
    sr = rn.StepRunner(cfg, emb, agg, [(P, syn.shard_block_params(P, cfg.heads, 1)) for P in blocks], pos,
                       fused_front=case["fused"], head=head)
    loss = sr.step_head(rn.to_dev(x, "f32"), rn.to_dev(timg, "f32"))
    torch.cuda.synchronize()
    out = orc.step_head(x, emb, agg, blocks, head, timg, cfg.p, cfg.heads, cfg.ln_eps, pos)
    assert abs(float(loss.item()) - out["loss"]) <= 5 * tol * abs(out["loss"])
    errs = {"pred": check("pred", sr.head.pred, out["pred"], tol), "dy": check("dy", sr.head.dz, out["dy"], tol)}
    for k in ("lnf_g", "lnf_b", "Wh", "bh"):
        errs["head." + k] = check("head.d" + k, sr.head.G[k], out["head_grads"][k], tol)
    errs["dagg"] = check("dagg", sr.blocks[0].dx, out["dagg"], tol)
    errs["dWp"] = check("dWp", sr.front.dWp, out["dWp"], tol)
    errs["dbp"] = check("dbp", sr.front.dbp, out["dbp"], tol)
    errs["dWqkv0"] = check("dWqkv0", sr.blocks[0].gshards[0]["Wqkv"], out["block_grads"][0]["Wqkv"], tol)
    print("head step errs", case, {k: f"{v:.2e}" for k, v in errs.items()})


def test_head_loss_user_weights_and_errors(ob, rn):
    """Explicit weights (uniform = plain MSE) and argument checks of orbit_head_loss."""
    B, V, Hg, Wg, p, D = 2, 4, 8, 16, 2, 64
    head = syn.head_params(5, D, V, p, "f32")
    z = syn.normal(5, "z", (B, (Hg // p) * (Wg // p), D))
    timg = syn.fields(6, B, V, Hg, Wg, per_variable_scale=False)
    hr = rn.HeadRunner(B, V, Hg, Wg, p, D, "f32", "f32", head)
    ones = torch.ones(Hg, device="cuda")
    hr.loss_and_grad(rn.to_dev(z, "f32"), rn.to_dev(timg, "f32"), ones)
    torch.cuda.synchronize()
    l, pred, c = orc.head_loss(z, head, timg, p, latw=np.ones(Hg))
    dz, G = orc.head_loss_bwd(head, c)
    assert abs(float(hr.loss.item()) - l) <= 1e-5 * l
    check("pred", hr.pred, pred, 1e-4); check("dz", hr.dz, dz, 1e-4); check("dWh", hr.G["Wh"], G["Wh"], 1e-4)
    hr.hd.V = 3                                      # V p^2 = 12 is not a multiple of 8
    with pytest.raises(ob.OrbitError) as e:
        hr.loss_and_grad(rn.to_dev(z, "f32"), rn.to_dev(timg, "f32"))
    assert e.value.status == 2


def test_fused_front_error_codes(ob, rn):
    cfg = syn.Config("SE", B=1, V=4, Hg=8, Wg=8, p=2, D=64, heads=4, F=128, depth=1, dtype="bf16", resid_dtype="bf16")
    emb, agg, blocks, x, tgt, pos = make_step_case(cfg, 3)
    fr = rn.FusedFrontRunner(1, 4, 8, 8, 2, 64, 4, "bf16", "bf16", emb, agg)
    fr.fd.V = 129                                    # above the V <= 128 limit
    with pytest.raises(ob.OrbitError) as e:
        fr.fwd_keep(rn.to_dev(x, "f32"))
    assert e.value.status == 2                      # ORBIT_ERR_SHAPE
    fr.fd.V = 4
    fr.fd.p = 3                                      # Hg % p != 0 and unsupported patch size
    with pytest.raises(ob.OrbitError) as e:
        fr.fwd_keep(rn.to_dev(x, "f32"))
    assert e.value.status == 2


# ---------------------------------------------------------------------------------------------------------
def test_error_codes(ob, rn):
    P = syn.block_params(1, 64, 128, "bf16")
    with pytest.raises(ob.OrbitError) as e:          # D % heads != 0
        br = rn.BlockRunner(1, 16, 64, 3, 128, 1, "bf16", "bf16", P, syn.shard_block_params(P, 1, 1))
        br.fwd(torch.zeros(1, 16, 64, device="cuda", dtype=torch.bfloat16))
    assert e.value.status == 2                      # ORBIT_ERR_SHAPE
    P = syn.block_params(1, 64, 128, "bf16")
    br = rn.BlockRunner(1, 16, 64, 2, 128, 1, "bf16", "bf16", P, syn.shard_block_params(P, 2, 1))
    br.desc.flags = 4                               # unknown flag bit
    with pytest.raises(ob.OrbitError) as e:
        br.fwd(torch.zeros(1, 16, 64, device="cuda", dtype=torch.bfloat16))
    assert e.value.status == 6                      # ORBIT_ERR_UNSUPPORTED
    br.desc.flags = 1                               # QK-LayerNorm without its parameters
    with pytest.raises(ob.OrbitError) as e:
        br.fwd(torch.zeros(1, 16, 64, device="cuda", dtype=torch.bfloat16))
    assert e.value.status == 1                      # ORBIT_ERR_NULL
    br.desc.flags = 0
    br.ws_f = torch.empty(16, dtype=torch.uint8, device="cuda")
    with pytest.raises(ob.OrbitError) as e:
        br.fwd(torch.zeros(1, 16, 64, device="cuda", dtype=torch.bfloat16))
    assert e.value.status == 5                      # ORBIT_ERR_WORKSPACE


def test_step_replayed_from_cuda_graph_matches_oracle(rn):
    """StepRunner.capture: the whole step (fused front end + 2 blocks + MSE, fwd + bwd) captured into a CUDA graph and
    replayed on FRESH inputs written into the captured buffers must match the oracle like the eager step does -- every
    entry point only enqueues kernels on the caller's stream (include/orbit.h "Execution")."""
    cfg = syn.Config("S2", B=2, V=7, Hg=16, Wg=32, p=2, D=256, heads=4, F=1024, depth=2, dtype="bf16",
                     resid_dtype="f32")
    emb, agg, blocks, x, tgt, pos = make_step_case(cfg, 44)
    sr = rn.StepRunner(cfg, emb, agg, [(P, syn.shard_block_params(P, cfg.heads, 1)) for P in blocks], pos,
                       fused_front=True)
    x_d = torch.zeros(x.shape, device="cuda", dtype=torch.float32)          # captured with other contents
    t_d = torch.zeros(tgt.shape, device="cuda", dtype=torch.float32)
    replay = sr.capture(lambda: sr.step(x_d, t_d))
    x_d.copy_(torch.from_numpy(x))
    t_d.copy_(torch.from_numpy(np.asarray(tgt, dtype=np.float32)))
    replay()
    torch.cuda.synchronize()
    out = orc.step(x, emb, agg, blocks, tgt, cfg.p, cfg.heads, cfg.ln_eps, pos)
    check("graph y", sr.blocks[-1].y, out["y"], 1e-2)
    check("graph dagg", sr.blocks[0].dx, out["dagg"], 1e-2)
    check("graph dWp", sr.front.dWp, out["dWp"], 1e-2)
    check("graph b1.dWfc1", sr.blocks[1].gshards[0]["Wfc1"], out["block_grads"][1]["Wfc1"], 1e-2)
    assert abs(float(sr.loss.item()) - out["loss"]) <= 5e-2 * abs(out["loss"])


# ---- degenerate cases of the method (SURVEY.md 8(c) pins, here on the CUDA path) ---------------------------------
@pytest.mark.parametrize("N", [1, 2, 3])
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_block_tiny_sequences(rn, N, dtype):
    """N = 1: softmax over one key is 1 and O = V (the oracle pin 'N = 1 => O = V'); N = 2, 3: every tile is a tail."""
    B, D, heads, F = 3, 128, 4, 256
    P, shards, x, dy = make_block_case(31, B, N, D, heads, F, 1, dtype, "f32")
    br, y, dx = run_block(rn, B, N, D, heads, F, 1, dtype, "f32", P, shards, x, dy)
    compare_block(br, y, dx, P, x, dy, heads, 1, 1e-4 if dtype == "f32" else 1e-2)


@pytest.mark.parametrize("fused", [False, True])
@pytest.mark.parametrize("V", [1, 2])
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_front_end_one_and_two_variables(rn, V, fused, dtype):
    """V = 1: alpha = 1, the aggregation is (X Wv + bv) Wo + bo whatever q, Wq, Wk are and their gradients vanish
    (oracle pin); V = 2 is the smallest real softmax.  Both front ends."""
    cfg = syn.Config("SV", B=2, V=V, Hg=8, Wg=16, p=2, D=64, heads=4, F=128, depth=1, dtype=dtype, resid_dtype="f32")
    tol = 1e-4 if dtype == "f32" else 1e-2
    emb, agg, blocks, x, tgt, pos = make_step_case(cfg, 46)
    sr = rn.StepRunner(cfg, emb, agg, [(P, syn.shard_block_params(P, cfg.heads, 1)) for P in blocks], pos, fused_front=fused)
    sr.step(rn.to_dev(x, "f32"), rn.to_dev(tgt, cfg.resid_dtype))
    torch.cuda.synchronize()
    out = orc.step(x, emb, agg, blocks, tgt, cfg.p, cfg.heads, cfg.ln_eps, pos)
    check("agg", sr.front.out, out["agg"], tol)
    check("dWp", sr.front.dWp, out["dWp"], tol)
    check("dWv", sr.front.gagg["Wv"], out["agg_grads"]["Wv"], tol)
    check("dWo", sr.front.gagg["Wo"], out["agg_grads"]["Wo"], tol)
    if V == 1:        # gradients of the query path are analytically zero: compare absolutely against the scale of dWv
        scale = np.abs(out["agg_grads"]["Wv"]).max()
        for k in ("q", "Wq", "bq", "Wk"):
            got = sr.front.gagg[k].detach().to(torch.float32).cpu().numpy()
            assert np.abs(got).max() <= tol * scale, f"d{k} must vanish for V = 1"
    else:
        check("dWk", sr.front.gagg["Wk"], out["agg_grads"]["Wk"], tol)
        check("dq", sr.front.gagg["q"], out["agg_grads"]["q"], tol)


def test_single_patch_single_sample(rn):
    """B = 1 and one patch (L = 1): the smallest whole step (M = 1 row in every GEMM, attention over one token)."""
    cfg = syn.Config("S1", B=1, V=3, Hg=4, Wg=4, p=4, D=64, heads=4, F=128, depth=1, dtype="f32", resid_dtype="f32")
    run_and_compare_step(rn, cfg, 47, 1e-4)
    run_and_compare_step(rn, cfg, 47, 1e-4, fused=True)
