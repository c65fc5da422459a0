"""N > 1 plumbing of bench.py on CPU (gloo, world_size 2): the path itself does not shard (replicas only), so
what there is to check is the max-over-ranks timing reduction and that the reference arm prints exactly one line from rank 0."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    got = bench.max_over_ranks(10.0 + 5.0 * rank, world, "cpu")     # rank 1 is the slow one
    out[rank] = got
    dist.destroy_process_group()


def test_max_over_ranks_gloo_world2():
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, 29613, out), nprocs=2, join=True)
    assert out[0] == 15.0 and out[1] == 15.0


def test_reference_arm_under_torchrun_prints_one_line():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29617", os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
           "--warmup", "0", "--workload", "C2"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0


# ---- the rank-local Hybrid-STOP program with a REAL all-reduce, world size 2, gloo, CPU ---------------
def _rank_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import numpy as np
    from oracle import orbit_oracle as orc
    from paper_2404_14712_b200 import inputs as syn
    dist.init_process_group("gloo", rank=rank, world_size=world)

    def allreduce(part):
        t = torch.from_numpy(np.ascontiguousarray(part))
        dist.all_reduce(t)                       # sum over the tensor-parallel group
        return t.numpy()

    B, N, D, h, F = 2, 10, 32, 4, 64
    P = syn.block_params(77, D, F, "f32")
    P.update(syn.qk_norm_params(77, D // h, "f32"))
    x = syn.normal(77, "x", (B, N, D))
    dy = syn.normal(77, "dy", (B, N, D))
    S = syn.shard_block_params(P, h, world)[rank]           # every rank slices ITS shard from the same seeded parameters
    y, cache, _ = orc.rank_block_fwd(x, P, S, h // world, allreduce, 1e-5)
    dx, Gc, Gs, _ = orc.rank_block_bwd(dy, P, S, cache, allreduce)
    for k in ("qn_g", "qn_b", "kn_g", "kn_b"):            # head-shared parameters: partial sums over this rank's heads
        Gc[k] = allreduce(Gc[k])
    out[rank] = dict(y=y, dx=dx, Gc=Gc, Gs=Gs)
    dist.destroy_process_group()


def test_rank_local_hybrid_stop_gloo_world2_equals_unsharded_oracle():
    """Two processes, each running oracle.rank_block_fwd / rank_block_bwd on ITS shard with torch.distributed all-reduce
    (gloo) at the four combine points: y, dx and every gradient equal the unsharded oracle block."""
    import numpy as np
    sys.path.insert(0, ROOT)
    from oracle import orbit_oracle as orc
    from paper_2404_14712_b200 import inputs as syn
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_rank_worker, args=(2, 29623, out), nprocs=2, join=True)
    B, N, D, h, F = 2, 10, 32, 4, 64
    P = syn.block_params(77, D, F, "f32")
    P.update(syn.qk_norm_params(77, D // h, "f32"))
    x = syn.normal(77, "x", (B, N, D))
    dy = syn.normal(77, "dy", (B, N, D))
    y, cache = orc.block_fwd(x, P, h, 1e-5)
    dx, G = orc.block_bwd(dy, P, cache)
    for r in range(2):
        assert orc.rel_fro(out[r]["y"], y) < 1e-13 and orc.rel_fro(out[r]["dx"], dx) < 1e-12
        for k in ("ln1_g", "ln1_b", "ln2_g", "ln2_b", "bproj", "bfc2", "qn_g", "qn_b", "kn_g"):
            assert orc.rel_fro(out[r]["Gc"][k], G[k]) < 1e-12, k
    Gu = syn.unshard_block_grads([out[0]["Gs"], out[1]["Gs"]], 2)
    for k in Gu:
        assert orc.rel_fro(Gu[k], G[k]) < 1e-12, k
