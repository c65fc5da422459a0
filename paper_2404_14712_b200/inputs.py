"""Seeded synthetic inputs for the ORBIT hot path.

This module holds NO arithmetic of the method: only random draws, the Xavier bounds the configs
name, and rounding to the storage dtype.  Both the fp64 oracle (via tests/) and the CUDA path are
fed the arrays produced here, so that parity measures the compute path and not input quantisation.

Stand-in for CMIP6 / ERA5 fields (128x256xC_d samples, C_d in {48, 91}), which
are not available offline: white-noise Gaussian fields with per-variable offset/scale.
"""
from __future__ import annotations

import dataclasses
import math
import numpy as np


# --------------------------------------------------------------------------------------------
# Configurations (BASELINE.json `configs`, in order).  C1..C5.
# --------------------------------------------------------------------------------------------
@dataclasses.dataclass(frozen=True)
class Config:
    name: str
    B: int
    D: int
    heads: int
    F: int
    depth: int
    dtype: str            # "f32" | "bf16"   storage dtype of weights / activations / grads
    resid_dtype: str      # dtype of the residual stream x, y, dx, dy
    T: int = 1            # Hybrid-STOP shards
    # front end (None for block-only configs)
    V: int | None = None
    Hg: int | None = None
    Wg: int | None = None
    p: int | None = None
    N: int | None = None  # tokens per sample (block-only configs)
    ln_eps: float = 1e-5

    @property
    def L(self) -> int:
        if self.N is not None:
            return self.N
        return (self.Hg // self.p) * (self.Wg // self.p)

    @property
    def M(self) -> int:
        return self.B * self.L

    def block_flops_fwd(self) -> float:
        """Model FLOPs of one block forward: 2*M*D*(3D + D + 2F) + 4*B*N^2*D."""
        M, D, F, N, B = self.M, self.D, self.F, self.L, self.B
        return 2.0 * M * D * (3 * D + D + 2 * F) + 4.0 * B * N * N * D


CONFIGS = {
    "C1": Config("C1", B=2, V=4, Hg=32, Wg=64, p=4, D=128, heads=4, F=512, depth=1,
                 dtype="f32", resid_dtype="f32"),
    "C2": Config("C2", B=8, V=48, Hg=32, Wg=64, p=2, D=1024, heads=16, F=4096, depth=8,
                 dtype="bf16", resid_dtype="f32"),
    "C3": Config("C3", B=4, V=91, Hg=128, Wg=256, p=4, D=2048, heads=16, F=8192, depth=4,
                 dtype="bf16", resid_dtype="f32"),
    "C4": Config("C4", B=2, N=2048, D=4096, heads=32, F=16384, depth=1, T=4,
                 dtype="bf16", resid_dtype="bf16"),
    "C5": Config("C5", B=1, N=2048, D=12288, heads=96, F=49152, depth=1,
                 dtype="bf16", resid_dtype="bf16"),
    # the paper's own layer shapes (PAPER.md:140 model table), one block each: not BASELINE.json
    # configs, benchmarked with `bench.py --workload P113 / P10B`
    "P113": Config("P113", B=1, N=2048, D=12288, heads=64, F=49152, depth=1,       # 113B: 12288 wide, 64 heads => d_h 192
                   dtype="bf16", resid_dtype="bf16"),
    "P10B": Config("P10B", B=2, N=2048, D=8192, heads=32, F=32768, depth=1,        # 10B: 8192 wide, 32 heads => d_h 256
                   dtype="bf16", resid_dtype="bf16"),
}


# --------------------------------------------------------------------------------------------
# Storage rounding
# --------------------------------------------------------------------------------------------
def round_bf16(a: np.ndarray) -> np.ndarray:
    """Round float64/float32 values to the nearest bfloat16 (ties to even); returns float32 holding
    bf16-exact values."""
    f = np.ascontiguousarray(a, dtype=np.float32)
    u = f.view(np.uint32)
    r = (u >> np.uint32(16)) & np.uint32(1)      # uint32 arithmetic: finite inputs cannot wrap
    r += np.uint32(0x7FFF)
    r += u
    r &= np.uint32(0xFFFF0000)
    return r.view(np.float32).reshape(f.shape)


def round_storage(a: np.ndarray, dtype: str) -> np.ndarray:
    """Round once to the storage dtype; result is float32 that is exact in that dtype."""
    if dtype == "bf16":
        return round_bf16(a)
    if dtype == "f32":
        return np.ascontiguousarray(a, dtype=np.float32)
    raise ValueError(dtype)


# --------------------------------------------------------------------------------------------
# Draws
# --------------------------------------------------------------------------------------------
def _rng(seed: int, name: str) -> np.random.Generator:
    # one sub-stream per tensor name: stable under adding/removing other tensors
    tag = int.from_bytes(name.encode()[:8].ljust(8, b"\0"), "little") ^ (len(name) * 0x9E3779B97F4A7C15 & (2**63 - 1))
    return np.random.Generator(np.random.Philox(key=[seed & (2**64 - 1), tag & (2**64 - 1)]))


_CHUNK = 1 << 22   # elements per independently seeded chunk (result does not depend on the thread count)


def _draw(seed, name, shape, kind, a, b, dtype):
    """Fill an array of `shape` chunk by chunk (chunk c draws from sub-stream (seed, name, c)); chunks are
    generated on a thread pool.  kind "normal": a*N(0,1)+b ; kind "uniform": U(a, b)."""
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.float32)

    def fill(c):
        lo, hi = c * _CHUNK, min(n, (c + 1) * _CHUNK)
        g = _rng(seed, f"{name}#{c}" if c else name)
        if kind == "normal":
            v = g.standard_normal(size=hi - lo, dtype=np.float32)
            if a != 1.0:
                v *= np.float32(a)
            if b != 0.0:
                v += np.float32(b)
        else:
            v = g.random(size=hi - lo, dtype=np.float32)
            v *= np.float32(b - a)
            v += np.float32(a)
        out[lo:hi] = round_storage(v, dtype)

    nchunks = (n + _CHUNK - 1) // _CHUNK
    if nchunks <= 1:
        fill(0)
    else:
        from concurrent.futures import ThreadPoolExecutor
        import os
        with ThreadPoolExecutor(max_workers=min(16, os.cpu_count() or 1)) as ex:
            list(ex.map(fill, range(nchunks)))
    return out.reshape(shape)


def normal(seed, name, shape, scale=1.0, loc=0.0, dtype="f32"):
    return _draw(seed, name, shape, "normal", float(scale), float(loc), dtype)


def xavier_uniform(seed, name, shape, fan_in, fan_out, dtype="f32"):
    """U(+-sqrt(6/(fan_in+fan_out))) as BASELINE.json's configs say ("Xavier-uniform from a seed")."""
    bound = math.sqrt(6.0 / (fan_in + fan_out))
    return _draw(seed, name, shape, "uniform", -bound, bound, dtype)


# --------------------------------------------------------------------------------------------
# Parameter sets.  Layout conventions (include/orbit.h): weights are [in, out]; Wqkv columns are
# [Q | K | V], heads contiguous inside each third.
# --------------------------------------------------------------------------------------------
def block_params(seed: int, D: int, F: int, dtype: str, tag: str = "blk0") -> dict:
    """Unsharded parameters of one ViT block (non-degenerate biases/gains)."""
    P = {}
    P["ln1_g"] = round_storage(1.0 + normal(seed, tag + ".ln1_g", (D,), 0.1), dtype)
    P["ln1_b"] = normal(seed, tag + ".ln1_b", (D,), 0.1, dtype=dtype)
    P["Wqkv"] = xavier_uniform(seed, tag + ".Wqkv", (D, 3 * D), D, 3 * D, dtype)
    P["bqkv"] = normal(seed, tag + ".bqkv", (3 * D,), 0.02, dtype=dtype)
    P["Wproj"] = xavier_uniform(seed, tag + ".Wproj", (D, D), D, D, dtype)
    P["bproj"] = normal(seed, tag + ".bproj", (D,), 0.02, dtype=dtype)
    P["ln2_g"] = round_storage(1.0 + normal(seed, tag + ".ln2_g", (D,), 0.1), dtype)
    P["ln2_b"] = normal(seed, tag + ".ln2_b", (D,), 0.1, dtype=dtype)
    P["Wfc1"] = xavier_uniform(seed, tag + ".Wfc1", (D, F), D, F, dtype)
    P["bfc1"] = normal(seed, tag + ".bfc1", (F,), 0.02, dtype=dtype)
    P["Wfc2"] = xavier_uniform(seed, tag + ".Wfc2", (F, D), F, D, dtype)
    P["bfc2"] = normal(seed, tag + ".bfc2", (D,), 0.02, dtype=dtype)
    return P


def head_params(seed: int, D: int, V: int, p: int, dtype: str) -> dict:
    """Final LayerNorm and image-space head (R23, R26): Wh [D, V p^2] Xavier-uniform."""
    C = V * p * p
    return {
        "lnf_g": round_storage(1.0 + normal(seed, "head.lnf_g", (D,), 0.1), dtype),
        "lnf_b": normal(seed, "head.lnf_b", (D,), 0.1, dtype=dtype),
        "Wh": xavier_uniform(seed, "head.Wh", (D, C), D, C, dtype),
        "bh": normal(seed, "head.bh", (C,), 0.02, dtype=dtype),
    }


def qk_norm_params(seed: int, dh: int, dtype: str, tag: str = "blk0") -> dict:
    """QK-LayerNorm parameters (R9, R23): gains 1 + 0.1 N(0,1), biases 0.1 N(0,1), all [d_h]."""
    return {
        "qn_g": round_storage(1.0 + normal(seed, tag + ".qn_g", (dh,), 0.1), dtype),
        "qn_b": normal(seed, tag + ".qn_b", (dh,), 0.1, dtype=dtype),
        "kn_g": round_storage(1.0 + normal(seed, tag + ".kn_g", (dh,), 0.1), dtype),
        "kn_b": normal(seed, tag + ".kn_b", (dh,), 0.1, dtype=dtype),
    }


def shard_block_params(P: dict, heads: int, T: int) -> list[dict]:
    """Split unsharded block parameters into T Hybrid-STOP shards (Eq. 1-2):
    Wqkv, Wfc1 by columns (head-aligned; shard k's Wqkv is [Q_k | K_k | V_k]); Wproj, Wfc2 by rows.
    Pure slicing -- no arithmetic."""
    D = P["Wproj"].shape[0]
    F = P["Wfc1"].shape[1]
    assert heads % T == 0 and F % T == 0 and D % heads == 0
    dc, fc = D // T, F // T
    shards = []
    for k in range(T):
        cs = slice(k * dc, (k + 1) * dc)
        Wq, Wk, Wv = P["Wqkv"][:, 0:D], P["Wqkv"][:, D:2 * D], P["Wqkv"][:, 2 * D:3 * D]
        bq, bk, bv = P["bqkv"][0:D], P["bqkv"][D:2 * D], P["bqkv"][2 * D:3 * D]
        shards.append({
            "Wqkv": np.ascontiguousarray(np.concatenate([Wq[:, cs], Wk[:, cs], Wv[:, cs]], axis=1)),
            "bqkv": np.ascontiguousarray(np.concatenate([bq[cs], bk[cs], bv[cs]])),
            "Wproj": np.ascontiguousarray(P["Wproj"][cs, :]),
            "Wfc1": np.ascontiguousarray(P["Wfc1"][:, k * fc:(k + 1) * fc]),
            "bfc1": np.ascontiguousarray(P["bfc1"][k * fc:(k + 1) * fc]),
            "Wfc2": np.ascontiguousarray(P["Wfc2"][k * fc:(k + 1) * fc, :]),
        })
    return shards


def unshard_block_grads(gshards: list[dict], T: int) -> dict:
    """Inverse of shard_block_params for the sharded tensors (re-assembles shard gradients)."""
    D3 = gshards[0]["Wqkv"].shape[1] * T
    D = D3 // 3
    dc = D // T
    Wq = np.concatenate([g["Wqkv"][:, 0:dc] for g in gshards], axis=1)
    Wk = np.concatenate([g["Wqkv"][:, dc:2 * dc] for g in gshards], axis=1)
    Wv = np.concatenate([g["Wqkv"][:, 2 * dc:3 * dc] for g in gshards], axis=1)
    bq = np.concatenate([g["bqkv"][0:dc] for g in gshards])
    bk = np.concatenate([g["bqkv"][dc:2 * dc] for g in gshards])
    bv = np.concatenate([g["bqkv"][2 * dc:3 * dc] for g in gshards])
    return {
        "Wqkv": np.concatenate([Wq, Wk, Wv], axis=1),
        "bqkv": np.concatenate([bq, bk, bv]),
        "Wproj": np.concatenate([g["Wproj"] for g in gshards], axis=0),
        "Wfc1": np.concatenate([g["Wfc1"] for g in gshards], axis=1),
        "bfc1": np.concatenate([g["bfc1"] for g in gshards]),
        "Wfc2": np.concatenate([g["Wfc2"] for g in gshards], axis=0),
    }


def embed_params(seed: int, V: int, p: int, D: int, dtype: str) -> dict:
    """Per-variable patch-embedding weights Wp[V, p*p, D] (Xavier, fan_in=p^2, fan_out=D) and bias
    bp[V, D] (patch-embed bias + variable embedding folded)."""
    return {
        "Wp": xavier_uniform(seed, "emb.Wp", (V, p * p, D), p * p, D, dtype),
        "bp": normal(seed, "emb.bp", (V, D), 0.02, dtype=dtype),
    }


def agg_params(seed: int, D: int, dtype: str) -> dict:
    """Variable-aggregation cross-attention parameters."""
    P = {"q": normal(seed, "agg.q", (D,), 1.0, dtype=dtype)}
    for n in ("Wq", "Wk", "Wv", "Wo"):
        P[n] = xavier_uniform(seed, "agg." + n, (D, D), D, D, dtype)
    for n in ("bq", "bk", "bv", "bo"):
        P[n] = normal(seed, "agg." + n, (D,), 0.02, dtype=dtype)
    return P


def fields(seed: int, B: int, V: int, Hg: int, Wg: int, per_variable_scale: bool) -> np.ndarray:
    """Input fields x[B, V, Hg, Wg] (always fp32 storage).  C1: N(0,1).  C2/C3: N(mu_v, sigma_v^2)
    with mu_v ~ U(-1,1), sigma_v ~ U(0.5,2) -- un-normalised physical channels."""
    x = normal(seed, "x", (B, V, Hg, Wg))
    if per_variable_scale:
        g = _rng(seed, "x.stats")
        mu = g.uniform(-1.0, 1.0, size=(V,)).astype(np.float32)
        sg = g.uniform(0.5, 2.0, size=(V,)).astype(np.float32)
        x = x * sg[None, :, None, None] + mu[None, :, None, None]
    return np.ascontiguousarray(x, dtype=np.float32)


def seed_of(cfg_name: str) -> int:
    if cfg_name.startswith("P"):                  # paper-shaped workloads
        return 1100 + int("".join(ch for ch in cfg_name if ch.isdigit()))
    return 1000 + int(cfg_name[1:])
