"""Kernel-level parity of the LayerNorm kernels (PAPER.md:88 pre-LN sub-layers; SURVEY.md 8(c) BLK / BLK') against
oracle.layernorm / oracle.layernorm_bwd (fp64 definition), through orbit_debug_layernorm_fwd / _bwd.

The shapes walk every launch configuration of layernorm_tma.cu: one chunk per thread with 1, 2 or 4 rows per stage and
a ragged last row group, 2 / 3 / 4 chunks per thread, a ragged last chunk (D/8 not a multiple of 32), the case where the
`add` slice does not fit the stages and is read from global memory, and a row too long for two stages (the one-block
kernels of rowops.cu)."""
import numpy as np
import pytest
import torch

from oracle import orbit_oracle as oracle
from paper_2404_14712_b200 import inputs as syn

pytestmark = pytest.mark.gpu
EPS = 1e-5


@pytest.fixture(scope="module")
def ob():
    from paper_2404_14712_b200 import binding
    return binding


def _dev(ob, a, dt):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda().to(ob.TORCH_DTYPES[dt])


def _host(t):
    return t.float().cpu().numpy().astype(np.float64)


# (M, D, x dtype, out / param dtype)
FWD = [
    (5, 296, "f32", "f32"),          # tiny, 37 chunks: ragged warp
    (700, 128, "f32", "f32"),        # C1 width
    (4099, 512, "bf16", "bf16"),     # 4 rows per stage, 3 rows in the last group
    (1201, 2048, "f32", "bf16"),     # 2 rows per stage, ragged last group, fp32 residual stream (C3)
    (300, 4096, "bf16", "bf16"),     # 512 threads, one chunk each
    (130, 5000, "bf16", "bf16"),     # 2 chunks per thread, 625 chunks
    (64, 12288, "bf16", "bf16"),     # 3 chunks per thread (C5)
    (40, 16376, "f32", "bf16"),      # 4 chunks per thread, ragged
    (9, 16392, "bf16", "bf16"),      # beyond 4 x 512 chunks: one-block kernel
    (6, 32768, "f32", "f32"),        # two fp32 rows do not fit the stages: one-block kernel
]


@pytest.mark.parametrize("M,D,xdt,odt", FWD)
def test_layernorm_fwd(ob, M, D, xdt, odt):
    x = syn.normal(11, f"lnx{M}x{D}", (M, D), dtype=xdt) * 1.7 + 0.3
    g = syn.normal(11, f"lng{D}", (D,), dtype=odt) * 0.1 + 1.0
    b = syn.normal(11, f"lnb{D}", (D,), dtype=odt) * 0.1
    xd, gd, bd = _dev(ob, x, xdt), _dev(ob, g, odt), _dev(ob, b, odt)
    out = torch.full((M, D), float("nan"), device="cuda", dtype=ob.TORCH_DTYPES[odt])
    mean = torch.full((M,), float("nan"), device="cuda")
    rstd = torch.full((M,), float("nan"), device="cuda")
    ob.orbit_debug_layernorm_fwd(M, D, xdt, odt, odt, EPS, xd, gd, bd, out, mean, rstd)
    torch.cuda.synchronize()
    ref, zhat, rs = oracle.layernorm(_host(xd), _host(gd), _host(bd), EPS)
    tol = 1e-4 if odt == "f32" else 1e-2
    assert oracle.rel_fro(_host(out), ref) < tol
    assert oracle.rel_fro(_host(rstd), rs[:, 0]) < 1e-5
    mu = _host(xd).mean(axis=1)
    assert np.abs(_host(mean) - mu).max() < 1e-5 * (1 + np.abs(mu).max())


# (M, D, dout dtype, x dtype, add dtype or None, out dtype, also fp32 copy)
BWD = [
    (5, 296, "f32", "f32", None, "f32", False),
    (700, 128, "f32", "f32", "f32", "f32", True),
    (4099, 512, "f32", "bf16", "bf16", "bf16", True),     # 2-4 rows per stage, ragged last group
    (1201, 2048, "f32", "f32", "f32", "f32", False),
    (300, 4096, "f32", "bf16", "bf16", "bf16", True),     # C4: LN2 backward
    (130, 5000, "bf16", "bf16", None, "bf16", False),     # 2 chunks per thread
    (64, 12288, "f32", "bf16", "bf16", "bf16", True),     # C5: LN2 backward, x | dout | add staged
    (64, 12288, "f32", "bf16", "f32", "bf16", False),     # C5: LN1 backward, add read from global memory
    (40, 16376, "f32", "bf16", "bf16", "bf16", False),    # 4 chunks per thread, ragged
]


@pytest.mark.parametrize("M,D,ddt,xdt,adt,odt,want_f32", BWD)
def test_layernorm_bwd(ob, M, D, ddt, xdt, adt, odt, want_f32):
    x = syn.normal(12, f"lnx{M}x{D}", (M, D), dtype=xdt) * 1.3 - 0.2
    dout = syn.normal(12, f"lnd{M}x{D}", (M, D), dtype=ddt)
    g = syn.normal(12, f"lng{D}", (D,), dtype=odt) * 0.1 + 1.0
    xd, dd, gd = _dev(ob, x, xdt), _dev(ob, dout, ddt), _dev(ob, g, odt)
    ad = _dev(ob, syn.normal(12, f"lna{M}x{D}", (M, D), dtype=adt), adt) if adt else None
    # statistics as the forward kernel saves them (fp32), from the oracle
    _, zhat, rs = oracle.layernorm(_host(xd), np.ones(D), np.zeros(D), EPS)
    mean = torch.from_numpy(_host(xd).mean(axis=1).astype(np.float32)).cuda()
    rstd = torch.from_numpy(rs[:, 0].astype(np.float32)).cuda()
    dx = torch.full((M, D), float("nan"), device="cuda", dtype=ob.TORCH_DTYPES[odt])
    dxf = torch.full((M, D), float("nan"), device="cuda") if want_f32 else None
    dg = torch.zeros(D, device="cuda")
    db = torch.zeros(D, device="cuda")
    ob.orbit_debug_layernorm_bwd(M, D, ddt, xdt, odt, adt or "f32", odt, dd, xd, mean, rstd, gd, ad, dxf, dx, dg, db)
    torch.cuda.synchronize()
    dz, dgam, dbet = oracle.layernorm_bwd(_host(dd), zhat, rs, _host(gd))
    ref = dz + (_host(ad) if adt else 0.0)
    tol = 1e-4 if odt == "f32" else 1e-2
    assert oracle.rel_fro(_host(dx), ref) < tol
    if want_f32:
        assert oracle.rel_fro(_host(dxf), ref) < 1e-4
    assert oracle.rel_fro(_host(dg), dgam) < 1e-4
    assert oracle.rel_fro(_host(db), dbet) < 1e-4


def test_layernorm_bwd_row_too_long(ob):
    """Backward keeps 16 column sums per chunk in registers: rows beyond 4 x 512 chunks (D > 16384) are refused with
    ORBIT_ERR_SHAPE before any launch (include/orbit.h error contract)."""
    M, D = 4, 16392
    z = torch.zeros((M, D), device="cuda")
    v = torch.zeros((M,), device="cuda")
    g = torch.ones((D,), device="cuda")
    acc = torch.zeros((D,), device="cuda")
    with pytest.raises(ob.OrbitError) as e:
        ob.orbit_debug_layernorm_bwd(M, D, "f32", "f32", "f32", "f32", "f32", z, z, v, v, g, None, None, z.clone(), acc, acc.clone())
    assert e.value.status == 2          # ORBIT_ERR_SHAPE (include/orbit.h)
