"""Boundary contract "thread-safe for distinct streams" (include/orbit.h): two host threads drive two blocks on two
streams at the same time through the C-ABI (ctypes releases the GIL inside a call); results must equal the same calls
issued alone.  Covers the per-device once-only launch setup (cudaFuncSetAttribute records) and the thread-local error /
launch-count state."""
import threading

import pytest
import torch

from paper_2404_14712_b200 import inputs as syn

pytestmark = pytest.mark.gpu


def _make(rn, seed, shape, dtype, rdt):
    B, N, D, heads, F, T = shape
    P = syn.block_params(seed, D, F, dtype)
    br = rn.BlockRunner(B, N, D, heads, F, T, dtype, rdt, P, syn.shard_block_params(P, heads, T))
    x = rn.to_dev(syn.normal(seed, "blk.x", (B, N, D), dtype=rdt), rdt)
    dy = rn.to_dev(syn.normal(seed, "blk.dy", (B, N, D), dtype=rdt), rdt)
    return br, x, dy


def _run(br, x, dy, stream, reps, out, idx, ob):
    try:
        ob.orbit_reset_launch_count()
        with torch.cuda.stream(stream):
            for _ in range(reps):
                y = br.fwd(x)
                dx = br.bwd(dy)
        stream.synchronize()
        out[idx] = (y.clone(), dx.clone(), {k: v.clone() for k, v in br.gshards[0].items()}, ob.orbit_launch_count())
    except Exception as e:        # surfaced by the main thread
        out[idx] = e


def test_two_threads_two_streams_match_serial_runs():
    from paper_2404_14712_b200 import binding as ob, runner as rn
    cases = [(31, (2, 384, 512, 8, 2048, 1), "bf16", "bf16"),      # tcgen05 GEMMs + tcgen05 attention, d_h 64
             (32, (1, 200, 256, 2, 1024, 2), "bf16", "f32")]       # d_h 128, ragged N, Hybrid-STOP T = 2
    runners = [_make(rn, *c) for c in cases]
    torch.cuda.synchronize()
    serial = [None, None]
    for i, (br, x, dy) in enumerate(runners):
        _run(br, x, dy, torch.cuda.Stream(), 1, serial, i, ob)
        assert not isinstance(serial[i], Exception), serial[i]
    both = [None, None]
    threads = [threading.Thread(target=_run, args=(br, x, dy, torch.cuda.Stream(), 6, both, i, ob))
               for i, (br, x, dy) in enumerate(runners)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    for i in range(2):
        assert not isinstance(both[i], Exception), both[i]
        ys, dxs, gs, n1 = serial[i]
        yt, dxt, gt, n6 = both[i]
        assert n6 == 6 * n1 and n1 > 0          # launch counter is per thread
        assert torch.equal(ys, yt)              # forward: no atomics, bit-identical
        # backward: LN / bias gradients use fp32 atomics (order varies), everything else is deterministic
        assert torch.allclose(dxs.float(), dxt.float(), rtol=1e-2, atol=1e-5)
        for k in gs:
            assert torch.allclose(gs[k].float(), gt[k].float(), rtol=2e-2, atol=1e-4), k
