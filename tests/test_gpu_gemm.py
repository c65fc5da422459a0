"""Kernel-level parity of the GEMM dispatcher (tcgen05 path for bf16, fp32-FMA path otherwise) against the
definition C = A B evaluated in float64 (numpy matmul), for every operand-major combination the block uses
(forward x A, backward dy B^T, weight gradient x^T dy) and for ragged sizes that leave partial
tiles in M, N and K."""
import numpy as np
import pytest
import torch

from paper_2404_14712_b200 import inputs as syn

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ob():
    from paper_2404_14712_b200 import binding
    return binding


def run_gemm(ob, M, N, K, a_major, b_major, dtype):
    A = syn.normal(5, f"A{M}{K}", (M, K), dtype=dtype)
    B = syn.normal(5, f"B{K}{N}", (K, N), dtype=dtype)
    td = ob.TORCH_DTYPES[dtype]
    At, Bt = torch.from_numpy(A).cuda().to(td), torch.from_numpy(B).cuda().to(td)
    if a_major == "K":
        Ad, a_rs, a_cs = At.contiguous(), K, 1
    else:
        Ad, a_rs, a_cs = At.t().contiguous(), 1, M
    if b_major == "N":
        Bd, b_rs, b_cs = Bt.contiguous(), N, 1
    else:
        Bd, b_rs, b_cs = Bt.t().contiguous(), 1, K
    C = torch.full((M, N), float("nan"), device="cuda", dtype=torch.float32)
    ob.orbit_debug_gemm(M, N, K, dtype, Ad, a_rs, a_cs, Bd, b_rs, b_cs, C)
    torch.cuda.synchronize()
    ref = A.astype(np.float64) @ B.astype(np.float64)
    got = C.cpu().numpy().astype(np.float64)
    assert np.isfinite(got).all()
    return np.linalg.norm(got - ref) / np.linalg.norm(ref)


SHAPES = [(128, 256, 64), (256, 512, 256), (200, 264, 136), (1024, 768, 520), (2048, 1024, 2048), (64, 64, 32),
          (2048, 3072, 512), (1800, 2904, 264),     # two rounds of 256 x 256 CTA-pair tiles, ragged N tail
          (2048, 12288, 320), (1800, 9992, 136)]    # 384 / 320 tiles on 74 clusters: the 14 / 24 tiles of the last round run as
                                                    # 256 x 128 column sub-tiles (gemm_tc2.cu Sched), full and ragged N


@pytest.mark.parametrize("a_major", ["K", "M"])
@pytest.mark.parametrize("b_major", ["N", "K"])
@pytest.mark.parametrize("shape", SHAPES)
def test_gemm_bf16_tensor_core(ob, shape, a_major, b_major):
    M, N, K = shape
    err = run_gemm(ob, M, N, K, a_major, b_major, "bf16")
    assert err < 1e-4, f"{shape} A:{a_major}-major B:{b_major}-major rel err {err:.3e}"


@pytest.mark.parametrize("a_major", ["K", "M"])
@pytest.mark.parametrize("b_major", ["N", "K"])
def test_gemm_fp32_fma(ob, a_major, b_major):
    err = run_gemm(ob, 200, 264, 136, a_major, b_major, "f32")
    assert err < 1e-5
    # bf16 operands whose N is not a multiple of 8 take the fp32-FMA kernel as well (no TMA row stride)
    err = run_gemm(ob, 200, 260, 136, a_major, b_major, "bf16")
    assert err < 1e-5


@pytest.mark.parametrize("case", [
    # (M, N, K, batch): the three per-head products of the front end (N = d_a = 128; ragged M / K tails)
    (1000, 128, 1632, 4), (1632, 128, 520, 3), (520, 1632, 128, 5), (300, 64, 72, 2), (512, 512, 256, 3),
])
@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_gemm_strided_batch(ob, case, dtype):
    """Strided-batch GEMM (3-D TMA maps, batch folded into the persistent tile loop) against float64 per problem:
    A_i = columns [i*K, (i+1)*K) of one [M, batch*K] matrix, B_i / C_i = column blocks of [K, batch*N] / [M, batch*N]."""
    M, N, K, nb = case
    rng = np.random.default_rng(5)
    tdt = torch.bfloat16 if dtype == "bf16" else torch.float32
    A = torch.from_numpy(rng.standard_normal((M, nb * K)).astype(np.float32)).to(tdt)
    B = torch.from_numpy(rng.standard_normal((K, nb * N)).astype(np.float32)).to(tdt)
    Ad, Bd = A.cuda().contiguous(), B.cuda().contiguous()
    C = torch.full((M, nb * N), float("nan"), device="cuda", dtype=torch.float32)
    ob.orbit_debug_gemm_batched(M, N, K, nb, dtype, Ad, nb * K, 1, K, Bd, nb * N, 1, N, C, nb * N, N)
    torch.cuda.synchronize()
    got = C.cpu().numpy().astype(np.float64)
    assert np.isfinite(got).all()
    A64, B64 = A.to(torch.float64).numpy(), B.to(torch.float64).numpy()
    for i in range(nb):
        ref = A64[:, i * K:(i + 1) * K] @ B64[:, i * N:(i + 1) * N]
        err = np.linalg.norm(got[:, i * N:(i + 1) * N] - ref) / np.linalg.norm(ref)
        assert err < 1e-4, f"{case} {dtype} batch {i}: rel err {err:.3e}"


# ---- bf16 outputs (+ bias): the TMA-store epilogue of the CTA-pair kernel, ragged in M and N, padded row stride ----
OUT_SHAPES = [(256, 256, 64, 256), (520, 776, 136, 776), (1800, 2904, 264, 2912), (300, 264, 520, 272), (2048, 3072, 512, 3072),
              (2048, 12288, 192, 12288)]          # last round of 14 tiles split into column sub-tiles (TMA-store epilogue)


@pytest.mark.parametrize("a_major", ["K", "M"])
@pytest.mark.parametrize("with_bias", [False, True])
@pytest.mark.parametrize("shape", OUT_SHAPES)
def test_gemm_bf16_out_tma_store(ob, shape, a_major, with_bias):
    M, N, K, ldc = shape
    A = syn.normal(6, f"A{M}{K}", (M, K), dtype="bf16")
    B = syn.normal(6, f"B{K}{N}", (K, N), dtype="bf16")
    bias = syn.normal(6, f"b{N}", (N,), dtype="bf16") if with_bias else None
    At, Bt = torch.from_numpy(A).cuda().bfloat16(), torch.from_numpy(B).cuda().bfloat16()
    if a_major == "K":
        Ad, a_rs, a_cs = At.contiguous(), K, 1
    else:
        Ad, a_rs, a_cs = At.t().contiguous(), 1, M
    bd = torch.from_numpy(bias).cuda().bfloat16() if with_bias else None
    C = torch.full((M, ldc), float("nan"), device="cuda", dtype=torch.bfloat16)
    ob.orbit_debug_gemm_out(M, N, K, "bf16", Ad, a_rs, a_cs, Bt.contiguous(), N, 1, "bf16", C, ldc, bd)
    torch.cuda.synchronize()
    ref = A.astype(np.float64) @ B.astype(np.float64) + (bias.astype(np.float64) if with_bias else 0.0)
    got = C.float().cpu().numpy().astype(np.float64)
    assert np.isfinite(got[:, :N]).all()
    assert np.isnan(got[:, N:]).all(), "columns beyond N (row padding) must not be written"
    err = np.linalg.norm(got[:, :N] - ref) / np.linalg.norm(ref)
    assert err < 4e-3, f"{shape} rel err {err:.3e}"        # one bf16 rounding of the fp32 accumulator (2^-9 relative, rms ~1.7e-3)
