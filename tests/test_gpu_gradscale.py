"""GPU parity of the dynamic gradient scaling / fp32 accumulation calls against the
oracle: orbit_grads_unscale_check, orbit_grads_accumulate, orbit_grad_scale_update."""
import json
import os

import numpy as np
import pytest
import torch

import parity
from oracle import orbit_oracle as orc
from paper_2404_14712_b200 import inputs as syn

pytestmark = pytest.mark.gpu
GOLD = os.path.join(os.path.dirname(__file__), "golden")
SIZES = [(12288,), (1, 7), (2048, 1031), (3, 8192 + 5), (8,), (4096, 1536)]      # ragged tails, several chunks, tiny tensors


@pytest.fixture(scope="module")
def ob():
    from paper_2404_14712_b200 import binding
    return binding


def make(dtype, scale_mag=1.0):
    return [syn.normal(61, f"g{i}", sh, scale_mag * (1 + i), dtype=dtype) for i, sh in enumerate(SIZES)]


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
@pytest.mark.parametrize("S", [1024.0, 3.0])
def test_unscale_check_matches_oracle(ob, dtype, S):
    gs = make(dtype, 50.0)
    dev = [torch.from_numpy(g).cuda().to(ob.TORCH_DTYPES[dtype]) for g in gs]
    scale = torch.tensor([S], dtype=torch.float32, device="cuda")
    found = torch.zeros(1, dtype=torch.float32, device="cuda")
    ob.orbit_grads_unscale_check(dev, dtype, scale, found)
    torch.cuda.synchronize()
    want, f = orc.grads_unscale_check(gs, S)
    assert float(found.item()) == f == 0.0
    for i, (d, w) in enumerate(zip(dev, want)):
        if S == 1024.0:                     # a power of two: exact in any binary format
            assert np.array_equal(parity.to_np(d).astype(np.float64), w), i
        else:
            parity.check(f"g{i}", d, w, 1e-2 if dtype == "bf16" else 1e-6, store=dtype)


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
@pytest.mark.parametrize("bad", [float("inf"), float("-inf"), float("nan")])
def test_unscale_check_detects_non_finite_anywhere(ob, dtype, bad):
    """One non-finite element in the LAST element of a ragged tail / the first element of a tiny tensor sets the flag;
    all other elements are still unscaled."""
    for which, pos in ((3, -1), (1, 0), (5, 12345)):
        gs = make(dtype)
        dev = [torch.from_numpy(g).cuda().to(ob.TORCH_DTYPES[dtype]) for g in gs]
        dev[which].view(-1)[pos] = bad
        scale = torch.tensor([2.0], dtype=torch.float32, device="cuda")
        found = torch.zeros(1, dtype=torch.float32, device="cuda")
        ob.orbit_grads_unscale_check(dev, dtype, scale, found)
        torch.cuda.synchronize()
        gs[which].reshape(-1)[pos] = bad
        want, f = orc.grads_unscale_check(gs, 2.0)
        assert float(found.item()) == f == 1.0
        got = parity.to_np(dev[which]).reshape(-1).astype(np.float64)
        ok = np.isfinite(want[which].reshape(-1))
        assert np.array_equal(got[ok], want[which].reshape(-1)[ok]) and not np.isfinite(got[~ok]).any()


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_accumulate_micro_steps_fp32(ob, dtype):
    """4 micro-steps of different gradients accumulated in fp32 with unscaling: equals the oracle to fp32 rounding, i.e.
    without the per-step bf16 rounding a `dtype` accumulator would add."""
    S = 8.0
    steps = [[syn.normal(62 + k, f"g{i}", sh, 1.0 + i, dtype=dtype) for i, sh in enumerate(SIZES)] for k in range(4)]
    acc = [torch.zeros(sh, dtype=torch.float32, device="cuda") for sh in SIZES]
    ref = [np.zeros(sh) for sh in SIZES]
    scale = torch.tensor([S], dtype=torch.float32, device="cuda")
    found = torch.zeros(1, dtype=torch.float32, device="cuda")
    for gs in steps:
        dev = [torch.from_numpy(g).cuda().to(ob.TORCH_DTYPES[dtype]) for g in gs]
        ob.orbit_grads_accumulate(dev, acc, dtype, scale, found)
        ref = orc.grads_accumulate(ref, gs, S)
    torch.cuda.synchronize()
    assert float(found.item()) == 0.0
    for i, (a, r) in enumerate(zip(acc, ref)):
        parity.check(f"acc{i}", a, r, 1e-6, store="f32")


def test_scale_update_golden_trace(ob):
    tr = json.load(open(os.path.join(GOLD, "grad_scale_trace.json")))
    scale = torch.tensor([tr["scale0"]], dtype=torch.float32, device="cuda")
    tracker = torch.zeros(1, dtype=torch.int32, device="cuda")
    s, t = tr["scale0"], 0
    for f, s_want, t_want in zip(tr["found_inf"], tr["scale_after"], tr["tracker_after"]):
        found = torch.tensor([float(f)], dtype=torch.float32, device="cuda")
        ob.orbit_grad_scale_update(scale, tracker, found, tr["growth_factor"], tr["backoff_factor"], tr["growth_interval"])
        s, t = orc.grad_scale_update(s, t, float(f), tr["growth_factor"], tr["backoff_factor"], tr["growth_interval"])
        assert float(scale.item()) == s == s_want and int(tracker.item()) == t == t_want


def test_scaled_step_round_trip(ob):
    """The mechanism end to end on a block: dy * S into orbit_block_bwd, then unscale: gradients match the oracle's
    unscaled backward (S a power of two: only the bf16 range changes)."""
    from paper_2404_14712_b200 import runner as rn
    B, N, D, heads, F, S = 1, 256, 256, 4, 1024, 4096.0
    P = syn.block_params(63, D, F, "bf16")
    x = syn.normal(63, "blk.x", (B, N, D), dtype="bf16")
    dy = syn.normal(63, "blk.dy", (B, N, D), 1e-3, dtype="bf16")
    br = rn.BlockRunner(B, N, D, heads, F, 1, "bf16", "bf16", P, syn.shard_block_params(P, heads, 1))
    br.fwd(rn.to_dev(x, "bf16"))
    br.bwd(rn.to_dev(dy * np.float32(S), "bf16"))
    grads = list(br.gcommon.values()) + list(br.gshards[0].values())
    scale = torch.tensor([S], dtype=torch.float32, device="cuda")
    found = torch.zeros(1, dtype=torch.float32, device="cuda")
    ob.orbit_grads_unscale_check(grads, "bf16", scale, found)
    torch.cuda.synchronize()
    assert float(found.item()) == 0.0
    yo, c = orc.block_fwd(x, P, heads)
    _, G = orc.block_bwd(dy, P, c)
    for k in br.COMMON:
        parity.check("d" + k, br.gcommon[k], G[k], 1e-2)
    for k in br.SHARD:
        parity.check("d" + k, br.gshards[0][k], G[k], 1e-2)
