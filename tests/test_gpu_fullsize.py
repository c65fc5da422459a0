"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

* C5 (113B-class block, the bench workload): the COMPLETE fp64 oracle -- y, dx and all 12 gradients (about 2.3e13 fp64
  FLOP on the host cores: a minute or two).
* C4 (10B-class, Hybrid-STOP T=4, bf16): complete comparison against the UNSHARDED oracle.
* C3 blocks: one block at C3's size (B 4, N 2048, D 2048, F 8192, fp32 residual stream), complete.
* C3 front end, fused pixel-space path (the bench default, orbit_embed_fused): agg on every patch and ALL gradients
  (dWp, dbp, the nine aggregation gradients, dpos) against the oracle's tokenize -> var_aggregate definition
  accumulated over chunks of patches (tests/parity.front_oracle_chunked; pinned on CPU).
* C3 front end, two-call path: tok / agg / dtok on sampled patches (patches are independent), and the tokeniser
  gradients from a seeded synthetic dtok.
* C2 (ClimaX-scale, depth 8, V=48): the whole step against the whole oracle.
Tolerance: relative Frobenius error <= 1e-2 (bf16), as north_star states, plus the element-wise bound of
tests/parity.py so that a single mis-addressed tile fails.
"""
import gc

import numpy as np
import pytest
import torch

import parity
from oracle import orbit_oracle as orc
from paper_2404_14712_b200 import inputs as syn

pytestmark = [pytest.mark.gpu, pytest.mark.slow]
TOL = 1e-2


@pytest.fixture(scope="module")
def rn():
    from paper_2404_14712_b200 import runner
    return runner


def rel(got, ref, name="tensor"):
    return parity.check(name, got, ref, TOL)


def run_block_complete(rn, cfg, seed, tag):
    """One block of cfg's size through orbit_block_fwd / orbit_block_bwd against the complete oracle."""
    P = syn.block_params(seed, cfg.D, cfg.F, cfg.dtype)
    x = syn.normal(seed, "blk.x", (cfg.B, cfg.L, cfg.D), dtype=cfg.resid_dtype)
    dy = syn.normal(seed, "blk.dy", (cfg.B, cfg.L, cfg.D), dtype=cfg.resid_dtype)
    br = rn.BlockRunner(cfg.B, cfg.L, cfg.D, cfg.heads, cfg.F, 1, cfg.dtype, cfg.resid_dtype, P,
                        syn.shard_block_params(P, cfg.heads, 1))
    y = br.fwd(rn.to_dev(x, cfg.resid_dtype))
    dx = br.bwd(rn.to_dev(dy, cfg.resid_dtype))
    torch.cuda.synchronize()
    yo, cache = orc.block_fwd(x, P, cfg.heads, cfg.ln_eps)
    errs = {"y": rel(y, yo, "y")}
    del yo
    dxo, G = orc.block_bwd(dy, P, cache)
    del cache
    gc.collect()
    errs["dx"] = rel(dx, dxo, "dx")
    for k in br.COMMON:
        errs[k] = rel(br.gcommon[k], G[k], "d" + k)
    for k in br.SHARD:
        errs[k] = rel(br.gshards[0][k], G.pop(k), "d" + k)     # pop: frees the 5 GB fp64 gradients one by one
        gc.collect()
    print(tag, "complete oracle errs", {k: f"{v:.2e}" for k, v in errs.items()})
    assert max(errs.values()) <= TOL, errs


def test_c5_fullsize_complete_oracle(rn):
    """BASELINE.json config 5, the workload bench.py times: y, dx and all 12 gradients at D = 12288 / 96 heads."""
    run_block_complete(rn, syn.CONFIGS["C5"], syn.seed_of("C5"), "C5")


def test_c3_size_block_complete_oracle(rn):
    """One block at C3's size: B 4, N 2048, D 2048, heads 16 (d_h 128), F 8192, bf16 with an fp32 residual stream."""
    run_block_complete(rn, syn.CONFIGS["C3"], syn.seed_of("C3"), "C3 block")


def test_c3_fused_front_end_fullsize_all_gradients(rn):
    """BASELINE.json config 3's front end through the pixel-space fused path bench.py times by default
    (V 91, 128 x 256, p 4, D 2048, heads 16): agg on every patch, dWp, dbp, all aggregation gradients and dpos."""
    cfg = syn.CONFIGS["C3"]
    seed = syn.seed_of("C3")
    emb = syn.embed_params(seed, cfg.V, cfg.p, cfg.D, cfg.dtype)
    agg = syn.agg_params(seed, cfg.D, cfg.dtype)
    x = syn.fields(seed, cfg.B, cfg.V, cfg.Hg, cfg.Wg, per_variable_scale=True)
    pos = syn.normal(seed, "pos", (cfg.L, cfg.D), 0.02, dtype=cfg.resid_dtype)
    dagg = syn.normal(seed, "dagg", (cfg.B, cfg.L, cfg.D), 1.0 / cfg.D, dtype=cfg.resid_dtype)
    fr = rn.FusedFrontRunner(cfg.B, cfg.V, cfg.Hg, cfg.Wg, cfg.p, cfg.D, cfg.heads, cfg.dtype, cfg.resid_dtype, emb, agg,
                             pos=pos)
    out = fr.fwd_keep(rn.to_dev(x, "f32"))
    fr.bwd(rn.to_dev(dagg, cfg.resid_dtype))
    torch.cuda.synchronize()
    # the fused path never rounds tokens to storage: the oracle consumes its own fp64 tokens (the definition)
    agg_o, dWp_o, dbp_o, G_o, dpos_o = parity.front_oracle_chunked(orc, x, emb, agg, dagg, cfg.p, cfg.heads, 64, pos=pos)
    errs = {"agg": rel(out, agg_o, "agg"), "dWp": rel(fr.dWp, dWp_o, "dWp"), "dbp": rel(fr.dbp, dbp_o, "dbp"),
            "dpos": rel(fr.dpos, dpos_o, "dpos")}
    for k, gk in G_o.items():
        if k == "bk":       # analytically zero: compared absolutely against the scale of dbq
            got = parity.to_np(fr.gagg[k])
            assert np.abs(got).max() <= TOL * max(1e-12, np.abs(G_o["bq"]).max()), "dbk must vanish"
        else:
            errs["agg." + k] = rel(fr.gagg[k], gk, "agg.d" + k)
    print("C3 fused front end errs", {k: f"{v:.2e}" for k, v in errs.items()})
    assert max(errs.values()) <= TOL, errs


def test_c4_fullsize_hybrid_stop_vs_unsharded_oracle(rn):
    cfg = syn.CONFIGS["C4"]
    seed = syn.seed_of("C4")
    P = syn.block_params(seed, cfg.D, cfg.F, cfg.dtype)
    x = syn.normal(seed, "blk.x", (cfg.B, cfg.L, cfg.D), dtype=cfg.resid_dtype)
    dy = syn.normal(seed, "blk.dy", (cfg.B, cfg.L, cfg.D), dtype=cfg.resid_dtype)
    br = rn.BlockRunner(cfg.B, cfg.L, cfg.D, cfg.heads, cfg.F, cfg.T, cfg.dtype, cfg.resid_dtype, P,
                        syn.shard_block_params(P, cfg.heads, cfg.T))
    y = br.fwd(rn.to_dev(x, cfg.resid_dtype))
    dx = br.bwd(rn.to_dev(dy, cfg.resid_dtype))
    torch.cuda.synchronize()
    yo, cache = orc.block_fwd(x, P, cfg.heads, cfg.ln_eps)          # UNSHARDED oracle
    dxo, G = orc.block_bwd(dy, P, cache)
    errs = {"y": rel(y, yo), "dx": rel(dx, dxo)}
    for k in br.COMMON:
        errs[k] = rel(br.gcommon[k], G[k])
    gs = [{k: v.detach().to(torch.float32).cpu().numpy() for k, v in S.items()} for S in br.gshards]
    Gu = syn.unshard_block_grads(gs, cfg.T)
    for k in Gu:
        errs[k] = rel(Gu[k], G[k])
    print("C4 errs", {k: f"{v:.2e}" for k, v in errs.items()})
    assert max(errs.values()) <= TOL, errs
    # the same block as the rank-local program (orbit_rank_*): 4 ranks in lock step on this GPU, the fp32 partials summed
    # between the calls as an all-reduce would, against the same unsharded oracle
    del br
    from test_gpu_rank import run_ranks
    runners, _ = run_ranks(rn, (cfg.B, cfg.L, cfg.D, cfg.heads, cfg.F), cfg.T, cfg.dtype, cfg.resid_dtype, P, x, dy)
    errs = {}
    for k, r in enumerate(runners):
        errs[f"r{k}.y"] = rel(r.y, yo, f"rank{k}.y")
        errs[f"r{k}.dx"] = rel(r.dx, dxo, f"rank{k}.dx")
        for name in r.COMMON:
            errs[f"r{k}.{name}"] = rel(r.gcommon[name], G[name], f"rank{k}.d{name}")
    Gu = syn.unshard_block_grads([{n: parity.to_np(v) for n, v in r.gshard.items()} for r in runners], cfg.T)
    for name in Gu:
        errs["rank." + name] = rel(Gu[name], G[name], "rank-local d" + name)
    print("C4 rank-local errs", {k: f"{v:.2e}" for k, v in errs.items() if not k.startswith(("r1", "r2", "r3"))})
    assert max(errs.values()) <= TOL, errs


def test_c3_front_end_fullsize_sampled_patches(rn):
    cfg = syn.CONFIGS["C3"]
    seed = syn.seed_of("C3")
    emb = syn.embed_params(seed, cfg.V, cfg.p, cfg.D, cfg.dtype)
    agg = syn.agg_params(seed, cfg.D, cfg.dtype)
    x = syn.fields(seed, cfg.B, cfg.V, cfg.Hg, cfg.Wg, per_variable_scale=True)
    dagg = syn.normal(seed, "dagg", (cfg.B, cfg.L, cfg.D), 1.0 / cfg.D, dtype=cfg.resid_dtype)
    fr = rn.FrontRunner(cfg.B, cfg.V, cfg.Hg, cfg.Wg, cfg.p, cfg.D, cfg.heads, cfg.dtype, cfg.resid_dtype, emb, agg)
    xd = rn.to_dev(x, "f32")
    out = fr.fwd_keep(xd)
    fr.bwd(rn.to_dev(dagg, cfg.resid_dtype))
    torch.cuda.synchronize()
    g = np.random.default_rng(6)
    ls = np.sort(g.choice(cfg.L, size=40, replace=False))
    ls[0], ls[-1] = 0, cfg.L - 1
    lsd = torch.from_numpy(ls).cuda()
    tok_s = orc.tokenize_patches(x, emb["Wp"], emb["bp"], cfg.p, ls)             # [B, S, V, D]
    e_tok = rel(fr.tok[:, lsd], tok_s)
    # the aggregation oracle consumes the storage-rounded tokens the GPU aggregation consumed
    agg_s, cache = orc.var_aggregate(syn.round_storage(tok_s, cfg.dtype), agg, cfg.heads)
    e_agg = rel(out[:, lsd], agg_s)
    dtok_s, _, _ = orc.var_aggregate_bwd(dagg[:, ls], agg, cache)
    e_dtok = rel(fr.dtok[:, lsd], dtok_s)
    print(f"C3 front end: tok {e_tok:.2e} agg {e_agg:.2e} dtok {e_dtok:.2e}")
    assert max(e_tok, e_agg, e_dtok) <= TOL
    # a1' in full: tokeniser gradients from a seeded synthetic dtok
    dtok = syn.normal(seed, "dtok", (cfg.B, cfg.L, cfg.V, cfg.D), 0.05, dtype=cfg.dtype)
    from paper_2404_14712_b200 import binding as ob
    dtd = rn.to_dev(dtok, cfg.dtype)
    ob.orbit_tokenize_bwd(fr.ed, xd, dtd, fr.dWp, fr.dbp, fr.ws_t)
    torch.cuda.synchronize()
    pix = orc.patches(x, cfg.p)
    e_w, e_b = 0.0, 0.0
    for v in range(cfg.V):                                                    # every variable, in full
        dWp_v = pix[:, v].reshape(cfg.B * cfg.L, -1).T @ dtok[:, :, v, :].reshape(cfg.B * cfg.L, cfg.D).astype(np.float64)
        dbp_v = dtok[:, :, v, :].reshape(cfg.B * cfg.L, cfg.D).astype(np.float64).sum(0)
        e_w = max(e_w, rel(fr.dWp[v], dWp_v))
        e_b = max(e_b, rel(fr.dbp[v], dbp_v))
    print(f"C3 tokenize_bwd: dWp {e_w:.2e} dbp {e_b:.2e}")
    assert max(e_w, e_b) <= TOL


def test_c2_fullsize_whole_step(rn):
    cfg = syn.CONFIGS["C2"]
    seed = syn.seed_of("C2")
    emb = syn.embed_params(seed, cfg.V, cfg.p, cfg.D, cfg.dtype)
    agg = syn.agg_params(seed, cfg.D, cfg.dtype)
    blocks = [syn.block_params(seed, cfg.D, cfg.F, cfg.dtype, tag=f"blk{i}") for i in range(cfg.depth)]
    x = syn.fields(seed, cfg.B, cfg.V, cfg.Hg, cfg.Wg, per_variable_scale=True)
    tgt = syn.normal(seed, "target", (cfg.B, cfg.L, cfg.D), dtype=cfg.resid_dtype)
    sr = rn.StepRunner(cfg, emb, agg, [(P, syn.shard_block_params(P, cfg.heads, 1)) for P in blocks])
    loss = sr.step(rn.to_dev(x, "f32"), rn.to_dev(tgt, cfg.resid_dtype))
    torch.cuda.synchronize()
    out = orc.step(x, emb, agg, blocks, tgt, cfg.p, cfg.heads, cfg.ln_eps)
    errs = {"tok": rel(sr.front.tok, out["tok"]), "agg": rel(sr.front.out, out["agg"]),
            "y": rel(sr.blocks[-1].y, out["y"]), "dagg": rel(sr.blocks[0].dx, out["dagg"]),
            "dtok": rel(sr.front.dtok, out["dtok"]), "dWp": rel(sr.front.dWp, out["dWp"]),
            "dbp": rel(sr.front.dbp, out["dbp"])}
    for i in (0, cfg.depth - 1):
        G = out["block_grads"][i]
        for k in sr.blocks[i].COMMON:
            errs[f"b{i}.{k}"] = rel(sr.blocks[i].gcommon[k], G[k])
        for k in sr.blocks[i].SHARD:
            errs[f"b{i}.{k}"] = rel(sr.blocks[i].gshards[0][k], G[k])
    for k, gk in out["agg_grads"].items():
        if k != "bk":
            errs["agg." + k] = rel(sr.front.gagg[k], gk)
    print("C2 errs", {k: f"{v:.2e}" for k, v in errs.items()})
    assert abs(float(loss.item()) - out["loss"]) <= 5 * TOL * abs(out["loss"])
    assert max(errs.values()) <= TOL, errs
