"""orbit_tokenize_bwd_noalloc (include/orbit.h; csrc/tokenize_noalloc.cu): the a1' tokeniser backward with its fp32
accumulators in a device array inside the library, for callers that cannot cudaMalloc a workspace.  Checked against the
existing caller-workspace path orbit_tokenize_bwd on the same inputs, on two calls in a row with DIFFERENT inputs (the
shared array keeps the previous call's contents: the second result must not contain the first's).

Collected last on purpose (pytest -x: a failure here must not hide other tests); passes alone in a fresh
process and after the other tests.
"""
import numpy as np
import pytest
import torch

import parity
from paper_2404_14712_b200 import inputs as syn

pytestmark = pytest.mark.gpu

# (B, V, Hg, Wg, p, D, dtype): tensor-core path (bf16), fp32 FMA path, a shape whose accumulators nearly fill the array
CASES = [
    (2, 5, 16, 32, 2, 256, "bf16"),
    (1, 3, 8, 24, 4, 136, "f32"),
    (1, 48, 16, 16, 4, 4096, "bf16"),      # 48 x 17 x 4096 fp32 = 12.75 MiB of the 16 MiB
]


@pytest.fixture(scope="module")
def ob():
    from paper_2404_14712_b200 import binding
    return binding


def _inputs(ob, seed, B, V, Hg, Wg, p, D, dtype):
    L = (Hg // p) * (Wg // p)
    x = torch.from_numpy(syn.normal(seed, "x", (B, V, Hg, Wg))).to(torch.float32).cuda()
    dtok = torch.from_numpy(syn.normal(seed, "dtok", (B, L, V, D), dtype=dtype)).cuda().to(ob.TORCH_DTYPES[dtype])
    return x, dtok


@pytest.mark.parametrize("case", CASES)
def test_noalloc_matches_workspace_path_twice(ob, case):
    B, V, Hg, Wg, p, D, dtype = case
    d = ob.embed_desc(B, V, Hg, Wg, p, D, dtype)
    tdt = ob.TORCH_DTYPES[dtype]
    tol = 1e-2 if dtype == "bf16" else 1e-4
    assert ob.orbit_tokenize_bwd_workspace_bytes(d) <= ob.orbit_tokenize_bwd_noalloc_max_bytes()
    ws = torch.empty(ob.orbit_tokenize_bwd_workspace_bytes(d), dtype=torch.uint8, device="cuda")
    ins = [_inputs(ob, 71 + k, B, V, Hg, Wg, p, D, dtype) for k in range(2)]
    outs = [[torch.full((V, p * p, D), float("nan"), dtype=tdt, device="cuda"),
             torch.full((V, D), float("nan"), dtype=tdt, device="cuda")] for _ in range(4)]
    torch.cuda.synchronize()
    free0 = None
    for k, (x, dtok) in enumerate(ins):                 # two calls in a row, different inputs, same shared array
        if k == 1:
            torch.cuda.synchronize()
            free0 = torch.cuda.mem_get_info()[0]
        ob.orbit_tokenize_bwd_noalloc(d, x, dtok, outs[k][0], outs[k][1])
        if k == 1:
            torch.cuda.synchronize()
            assert torch.cuda.mem_get_info()[0] >= free0, "the no-alloc entry point took device memory"
    for k, (x, dtok) in enumerate(ins):                 # the existing path, caller workspace
        ob.orbit_tokenize_bwd(d, x, dtok, outs[2 + k][0], outs[2 + k][1], ws)
    torch.cuda.synchronize()
    for k in range(2):
        for name, got, want in (("dWp", outs[k][0], outs[2 + k][0]), ("dbp", outs[k][1], outs[2 + k][1])):
            parity.check(f"call{k}.{name}", got, parity.to_np(want).astype(np.float64), tol, store=dtype)
    # the two calls had different inputs: had the array not been cleared, call 1 would carry call 0's sums
    assert not torch.equal(outs[0][0], outs[1][0])


def test_noalloc_rejects_sizes_beyond_the_array(ob):
    d = ob.embed_desc(1, 91, 8, 8, 4, 4096, "bf16")     # 91 x 17 x 4096 fp32 = 24.2 MiB > 16 MiB
    assert ob.orbit_tokenize_bwd_workspace_bytes(d) > ob.orbit_tokenize_bwd_noalloc_max_bytes()
    x = torch.zeros((1, 91, 8, 8), dtype=torch.float32, device="cuda")
    dtok = torch.zeros((1, 4, 91, 4096), dtype=torch.bfloat16, device="cuda")
    dWp = torch.full((91, 16, 4096), 7.0, dtype=torch.bfloat16, device="cuda")
    dbp = torch.full((91, 4096), 7.0, dtype=torch.bfloat16, device="cuda")
    with pytest.raises(ob.OrbitError) as e:
        ob.orbit_tokenize_bwd_noalloc(d, x, dtok, dWp, dbp)
    assert e.value.status == 5 and "exceed" in str(e.value)          # ORBIT_ERR_WORKSPACE, nothing written
    torch.cuda.synchronize()
    assert bool((dWp == 7.0).all()) and bool((dbp == 7.0).all())
    assert ob.lib.orbit_tokenize_bwd_noalloc(None, None, None, None, None, None) == 1      # ORBIT_ERR_NULL
