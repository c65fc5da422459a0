"""GPU parity of the rank-local Hybrid-STOP program (orbit_rank_*):
 * T ranks run on this one GPU as T host threads in lock step, the all-reduce being a sum over the threads' partials --
   every rank's pre-all-reduce partial is compared with the oracle's rank_block_* partial of the same rank, and y, dx and
   all gradients with the UNSHARDED oracle block (fp32: 1e-4, the shard-recombination tolerance; bf16: 1e-2);
 * two PROCESSES sharing the GPU with a real torch.distributed all-reduce (gloo; NCCL needs one GPU per rank) at the
   four combine points.
"""
import os
import sys
import threading

import numpy as np
import pytest
import torch

import parity
from oracle import orbit_oracle as orc
from paper_2404_14712_b200 import inputs as syn

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


class LockstepSum:
    """all-reduce(sum) over T host threads of one process: deposit, barrier, sum in rank order, barrier."""

    def __init__(self, T):
        self.T, self.slots, self.bar = T, [None] * T, threading.Barrier(T)

    def allreduce(self, rank):
        def f(t):
            self.slots[rank] = t.clone()
            self.bar.wait()
            total = self.slots[0].clone()
            for k in range(1, self.T):
                total += self.slots[k]
            self.bar.wait()
            t.copy_(total)
        return f


def run_ranks(rn, shape, T, dtype, rdt, P, x, dy):
    B, N, D, heads, F = shape
    shards = syn.shard_block_params(P, heads, T)
    grp = LockstepSum(T)
    runners = [rn.RankBlockRunner(B, N, D, heads, F, T, dtype, rdt, P, shards[k], allreduce=grp.allreduce(k)) for k in range(T)]
    xd, dyd = rn.to_dev(x, rdt), rn.to_dev(dy, rdt)
    errs = [None] * T

    def run(k):
        try:
            runners[k].partials = {}
            runners[k].fwd(xd)
            runners[k].bwd(dyd)
            torch.cuda.synchronize()
        except Exception as e:            # a dead rank would leave the others at the barrier
            errs[k] = e
            grp.bar.abort()
    ts = [threading.Thread(target=run, args=(k,)) for k in range(T)]
    [t.start() for t in ts]
    [t.join() for t in ts]
    for e in errs:
        if e is not None:
            raise e
    return runners, shards


def oracle_ranks(P, shards, x, dy, heads, T, eps=1e-5):
    """The oracle's rank-local program (rank_block_fwd / rank_block_bwd) for all T ranks in lock step: per rank
    (y, dx, Gc, Gs, forward partials, backward partials)."""
    slots, bar, res = [None] * T, threading.Barrier(T), [None] * T

    def allreduce(k):
        def f(part):
            slots[k] = part
            bar.wait()
            total = sum(slots[1:], slots[0])
            bar.wait()
            return total
        return f

    def run(k):
        yk, ck, pf = orc.rank_block_fwd(x, P, shards[k], heads // T, allreduce(k), eps)
        dxk, Gc, Gs, pb = orc.rank_block_bwd(dy, P, shards[k], ck, allreduce(k))
        res[k] = (yk, dxk, Gc, Gs, pf, pb)
    ts = [threading.Thread(target=run, args=(k,)) for k in range(T)]
    [t.start() for t in ts]
    [t.join() for t in ts]
    return res


def compare_ranks(runners, shards, P, x, dy, heads, T, tol, eps=1e-5):
    yo, cache = orc.block_fwd(x, P, heads, eps)               # the UNSHARDED oracle: what every rank must end up with
    dxo, G = orc.block_bwd(dy, P, cache)
    errs = {}
    for k, r in enumerate(runners):
        errs[f"r{k}.y"] = parity.check(f"rank{k}.y", r.y, yo, tol)
        errs[f"r{k}.dx"] = parity.check(f"rank{k}.dx", r.dx, dxo, tol)
        for name in r.COMMON:
            errs[f"r{k}.{name}"] = parity.check(f"rank{k}.d{name}", r.gcommon[name], G[name], tol)
    gs = [{n: parity.to_np(v) for n, v in r.gshard.items()} for r in runners]
    Gu = syn.unshard_block_grads(gs, T)
    for name in Gu:
        errs[name] = parity.check("d" + name, Gu[name], G[name], tol)
    if runners[0].qk_norm:                  # partial sums over each rank's heads: summed by the caller
        for name in ("qn_g", "qn_b", "kn_g"):
            tot = sum(parity.to_np(r.gcommon[name]).astype(np.float64) for r in runners)
            errs[name] = parity.check("d" + name, tot, G[name], tol)
    # what the collective sees: every rank's four pre-all-reduce partials against the oracle's rank-local program
    ref = oracle_ranks(P, shards, x, dy, heads, T, eps)
    for k, r in enumerate(runners):
        for name, want in list(ref[k][4].items()) + list(ref[k][5].items()):
            errs[f"r{k}.part.{name}"] = parity.check(f"rank{k}.part.{name}", r.partials[name], want, tol, store="f32")
    return errs


@pytest.fixture(scope="module")
def rn():
    from paper_2404_14712_b200 import runner
    return runner


@pytest.mark.parametrize("T", [1, 2, 4])
def test_rank_local_fp32_shard_recombination(rn, T):
    """fp32 storage, fp32 partials exchanged between ranks: <= 1e-4 against the UNSHARDED oracle (north_star's fp32
    shard-recombination check, here with the partial leaving the kernel sequence at every combine point)."""
    shape = (2, 256, 256, 8, 1024)
    P = syn.block_params(51, shape[2], shape[4], "f32")
    x = syn.normal(51, "blk.x", shape[:3])
    dy = syn.normal(51, "blk.dy", shape[:3])
    runners, shards = run_ranks(rn, shape, T, "f32", "f32", P, x, dy)
    compare_ranks(runners, shards, P, x, dy, shape[3], T, 1e-4)


@pytest.mark.parametrize("case", [
    ((2, 384, 512, 8, 2048), 2, "bf16", False),      # d_h 64, tcgen05 GEMMs with N = 3D/T = 768
    ((1, 520, 1024, 8, 4096), 4, "f32", False),      # d_h 128, ragged N, fp32 residual stream
    ((2, 256, 512, 4, 1024), 2, "bf16", True),       # QK-LayerNorm: head-shared gradients are per-rank partial sums
])
def test_rank_local_bf16(rn, case):
    shape, T, rdt, qkn = case
    P = syn.block_params(52, shape[2], shape[4], "bf16")
    if qkn:
        P.update(syn.qk_norm_params(52, shape[2] // shape[3], "bf16"))
    x = syn.normal(52, "blk.x", shape[:3], dtype=rdt)
    dy = syn.normal(52, "blk.dy", shape[:3], dtype=rdt)
    runners, shards = run_ranks(rn, shape, T, "bf16", rdt, P, x, dy)
    errs = compare_ranks(runners, shards, P, x, dy, shape[3], T, 1e-2)
    print("rank-local bf16", case, {k: f"{v:.1e}" for k, v in errs.items() if not k.startswith("r1") and not k.startswith("r2")})


def test_rank_local_rejects_recompute_and_null(rn):
    from paper_2404_14712_b200 import binding as ob
    d = ob.block_desc(1, 64, 128, 4, 256, 2, 1e-5, "bf16", "bf16", ob.ORBIT_RECOMPUTE)
    assert ob.lib.orbit_rank_fwd_attn(ob.C.byref(d), None, None, None, None, None) == 6      # ERR_UNSUPPORTED
    d = ob.block_desc(1, 64, 128, 4, 256, 2)
    assert ob.lib.orbit_rank_fwd_attn(ob.C.byref(d), None, None, None, None, None) == 1      # ERR_NULL
    d = ob.block_desc(1, 64, 128, 4, 256, 3)                                                 # heads % T != 0
    assert ob.lib.orbit_rank_fwd_attn(ob.C.byref(d), None, None, None, None, None) == 2      # ERR_SHAPE


# ---- two processes, one GPU, real all-reduce through torch.distributed (gloo) --------------------------------------------
def _proc(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from paper_2404_14712_b200 import runner as rn
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)

    def allreduce(t):
        torch.cuda.current_stream().synchronize()      # the partial is produced on the stream; gloo reads it from the host side
        try:
            dist.all_reduce(t)                           # gloo accepts CUDA tensors (staged through pinned host memory)
        except RuntimeError:
            h = t.cpu()
            dist.all_reduce(h)
            t.copy_(h)

    shape = (2, 256, 256, 8, 1024)
    B, N, D, heads, F = shape
    P = syn.block_params(53, D, F, "bf16")
    x = syn.normal(53, "blk.x", (B, N, D), dtype="f32")
    dy = syn.normal(53, "blk.dy", (B, N, D), dtype="f32")
    S = syn.shard_block_params(P, heads, world)[rank]
    r = rn.RankBlockRunner(B, N, D, heads, F, world, "bf16", "f32", P, S, allreduce=allreduce)
    r.fwd(rn.to_dev(x, "f32"))
    r.bwd(rn.to_dev(dy, "f32"))
    torch.cuda.synchronize()
    out[rank] = dict(y=rn.to_np(r.y), dx=rn.to_np(r.dx), gc={k: rn.to_np(v) for k, v in r.gcommon.items()},
                     gs={k: rn.to_np(v) for k, v in r.gshard.items()})
    dist.destroy_process_group()


def test_rank_local_two_processes_gloo_allreduce():
    import torch.multiprocessing as mp
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_proc, args=(2, 29631, out), nprocs=2, join=True)
    shape = (2, 256, 256, 8, 1024)
    B, N, D, heads, F = shape
    P = syn.block_params(53, D, F, "bf16")
    x = syn.normal(53, "blk.x", (B, N, D), dtype="f32")
    dy = syn.normal(53, "blk.dy", (B, N, D), dtype="f32")
    yo, cache = orc.block_fwd(x, P, heads, 1e-5)
    dxo, G = orc.block_bwd(dy, P, cache)
    for r in range(2):
        parity.check(f"rank{r}.y", out[r]["y"], yo, 1e-2)
        parity.check(f"rank{r}.dx", out[r]["dx"], dxo, 1e-2)
        for k in ("ln1_g", "ln1_b", "ln2_g", "ln2_b", "bproj", "bfc2"):
            parity.check(f"rank{r}.d{k}", out[r]["gc"][k], G[k], 1e-2)
    Gu = syn.unshard_block_grads([out[0]["gs"], out[1]["gs"]], 2)
    for k in Gu:
        parity.check("d" + k, Gu[k], G[k], 1e-2)
