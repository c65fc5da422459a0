"""Thin ctypes binding over liborbit.so -- same names as the C entry points of include/orbit.h.

Argument marshalling only: every step of the path runs in the CUDA kernels behind the C-ABI.  torch is used
for device memory and streams (tensor.data_ptr(), torch.cuda.current_stream()).  There is NO fallback: if
liborbit.so is missing or fails to load, importing this module raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# ORBIT_LIB=dbg selects the A/B build (liborbit_dbg.so, `ORBIT_DEBUG_SWITCH=1 python -m paper_2404_14712_b200.build`)
LIB_PATH = os.path.join(_HERE, "liborbit_dbg.so" if os.environ.get("ORBIT_LIB") == "dbg" else "liborbit.so")
if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} not found: build it with `python -m paper_2404_14712_b200.build` "
        "(there is no CPU or PyTorch fallback for the ORBIT hot path)")
lib = C.CDLL(LIB_PATH)

ORBIT_OK = 0
ORBIT_F32, ORBIT_BF16 = 0, 1
STATUS_NAMES = {0: "OK", 1: "ERR_NULL", 2: "ERR_SHAPE", 3: "ERR_DTYPE", 4: "ERR_ALIGN", 5: "ERR_WORKSPACE",
                6: "ERR_UNSUPPORTED", 7: "ERR_ARCH", 8: "ERR_CUDA"}
DTYPES = {"f32": ORBIT_F32, "bf16": ORBIT_BF16}
TORCH_DTYPES = {"f32": torch.float32, "bf16": torch.bfloat16}


class OrbitError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = lib.orbit_last_error().decode(errors="replace")
        super().__init__(f"{where}: {STATUS_NAMES.get(status, status)}: {msg}")


# ---- descriptor / parameter structs (mirror include/orbit.h) -------------------------------------------
class orbit_embed_desc(C.Structure):
    _fields_ = [("B", C.c_int), ("V", C.c_int), ("Hg", C.c_int), ("Wg", C.c_int), ("p", C.c_int), ("D", C.c_int),
                ("dtype", C.c_int)]


class orbit_agg_desc(C.Structure):
    _fields_ = [("B", C.c_int), ("L", C.c_int), ("V", C.c_int), ("D", C.c_int), ("heads", C.c_int),
                ("dtype", C.c_int), ("resid_dtype", C.c_int)]


_AGG_NAMES = ("q", "Wq", "bq", "Wk", "bk", "Wv", "bv", "Wo", "bo")


class orbit_agg_params(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in _AGG_NAMES]


class orbit_agg_grads(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in _AGG_NAMES]


class orbit_front_desc(C.Structure):
    _fields_ = [("B", C.c_int), ("V", C.c_int), ("Hg", C.c_int), ("Wg", C.c_int), ("p", C.c_int), ("D", C.c_int),
                ("heads", C.c_int), ("dtype", C.c_int), ("resid_dtype", C.c_int)]


class orbit_head_desc(C.Structure):
    _fields_ = [("B", C.c_int), ("V", C.c_int), ("Hg", C.c_int), ("Wg", C.c_int), ("p", C.c_int), ("D", C.c_int),
                ("ln_eps", C.c_float), ("dtype", C.c_int), ("resid_dtype", C.c_int)]


class orbit_block_desc(C.Structure):
    _fields_ = [("B", C.c_int), ("N", C.c_int), ("D", C.c_int), ("heads", C.c_int), ("F", C.c_int), ("T", C.c_int),
                ("ln_eps", C.c_float), ("dtype", C.c_int), ("resid_dtype", C.c_int), ("flags", C.c_uint)]


_SHARD_NAMES = ("Wqkv", "bqkv", "Wproj", "Wfc1", "bfc1", "Wfc2")
_COMMON_NAMES = ("ln1_g", "ln1_b", "ln2_g", "ln2_b", "bproj", "bfc2")
_QKN_NAMES = ("qn_g", "qn_b", "kn_g", "kn_b")      # QK-LayerNorm parameters [d_h], only with ORBIT_QK_NORM
ORBIT_QK_NORM, ORBIT_RECOMPUTE = 1, 2


class orbit_block_shard(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in _SHARD_NAMES]


class orbit_block_params(C.Structure):
    _fields_ = ([(n, C.c_void_p) for n in _COMMON_NAMES] + [("shards", C.POINTER(orbit_block_shard))] +
                [(n, C.c_void_p) for n in _QKN_NAMES])


class orbit_block_grads(C.Structure):
    _fields_ = ([(n, C.c_void_p) for n in _COMMON_NAMES] + [("shards", C.POINTER(orbit_block_shard))] +
                [(n, C.c_void_p) for n in _QKN_NAMES])


# ---- prototypes ---------------------------------------------------------------------------------------------
def _proto(name, restype, argtypes):
    f = getattr(lib, name)
    f.restype = restype
    f.argtypes = argtypes
    return f


_vp, _sz = C.c_void_p, C.c_size_t
_proto("orbit_last_error", C.c_char_p, [])
_proto("orbit_version", C.c_int, [])
_proto("orbit_launch_count", C.c_longlong, [])
_proto("orbit_reset_launch_count", None, [])
_bd, _bp, _bg = C.POINTER(orbit_block_desc), C.POINTER(orbit_block_params), C.POINTER(orbit_block_grads)
_proto("orbit_rank_fwd_attn", C.c_int, [_bd, _vp, _bp, _vp, _vp, _vp])
_proto("orbit_rank_fwd_mlp", C.c_int, [_bd, _bp, _vp, _vp, _vp])
_proto("orbit_rank_fwd_out", C.c_int, [_bd, _bp, _vp, _vp, _vp, _vp])
_proto("orbit_rank_bwd_mlp", C.c_int, [_bd, _vp, _bp, _vp, _bg, _vp, _vp, _sz, _vp])
_proto("orbit_rank_bwd_attn", C.c_int, [_bd, _vp, _bp, _vp, _bg, _vp, _vp, _sz, _vp])
_proto("orbit_rank_bwd_out", C.c_int, [_bd, _bp, _vp, _bg, _vp, _vp, _vp, _sz, _vp])
_proto("orbit_rank_saved_bytes", _sz, [_bd])
_proto("orbit_rank_bwd_workspace_bytes", _sz, [_bd])
_proto("orbit_grads_unscale_check", C.c_int, [C.c_int, C.POINTER(_vp), C.POINTER(_sz), C.c_int, _vp, _vp, _vp])
_proto("orbit_grads_accumulate", C.c_int, [C.c_int, C.POINTER(_vp), C.POINTER(_vp), C.POINTER(_sz), C.c_int, _vp, _vp, _vp])
_proto("orbit_grad_scale_update", C.c_int, [_vp, _vp, _vp, C.c_float, C.c_float, C.c_int, _vp])
HAS_DEBUG_SWITCH = hasattr(lib, "orbit_set_debug_force_simt")      # only the A/B build exports it (csrc/orbit_debug.h)
if HAS_DEBUG_SWITCH:
    _proto("orbit_set_debug_force_simt", None, [C.c_int])
_proto("orbit_tokenize", C.c_int, [C.POINTER(orbit_embed_desc), _vp, _vp, _vp, _vp, _vp])
_proto("orbit_tokenize_bwd", C.c_int, [C.POINTER(orbit_embed_desc), _vp, _vp, _vp, _vp, _vp, _sz, _vp])
_proto("orbit_tokenize_bwd_workspace_bytes", _sz, [C.POINTER(orbit_embed_desc)])
_proto("orbit_tokenize_bwd_noalloc", C.c_int, [C.POINTER(orbit_embed_desc), _vp, _vp, _vp, _vp, _vp])
_proto("orbit_tokenize_bwd_noalloc_max_bytes", _sz, [])
_proto("orbit_var_aggregate", C.c_int,
       [C.POINTER(orbit_agg_desc), _vp, C.POINTER(orbit_agg_params), _vp, _vp, _vp, _vp, _sz, _vp])
_proto("orbit_var_aggregate_bwd", C.c_int,
       [C.POINTER(orbit_agg_desc), _vp, C.POINTER(orbit_agg_params), _vp, _vp, _vp, C.POINTER(orbit_agg_grads), _vp,
        _vp, _sz, _vp])
for _n in ("orbit_var_aggregate_workspace_bytes", "orbit_var_aggregate_bwd_workspace_bytes",
           "orbit_var_aggregate_saved_bytes"):
    _proto(_n, _sz, [C.POINTER(orbit_agg_desc)])
_proto("orbit_embed_fused", C.c_int,
       [C.POINTER(orbit_front_desc), _vp, _vp, _vp, C.POINTER(orbit_agg_params), _vp, _vp, _vp, _vp, _sz, _vp])
_proto("orbit_embed_fused_bwd", C.c_int,
       [C.POINTER(orbit_front_desc), _vp, _vp, _vp, C.POINTER(orbit_agg_params), _vp, _vp, _vp, _vp,
        C.POINTER(orbit_agg_grads), _vp, _vp, _sz, _vp])
for _n in ("orbit_embed_fused_workspace_bytes", "orbit_embed_fused_bwd_workspace_bytes", "orbit_embed_fused_saved_bytes"):
    _proto(_n, _sz, [C.POINTER(orbit_front_desc)])
_proto("orbit_head_loss", C.c_int, [C.POINTER(orbit_head_desc)] + [_vp] * 11 + [_sz, _vp])
_proto("orbit_head_loss_bwd", C.c_int, [C.POINTER(orbit_head_desc)] + [_vp] * 10 + [_sz, _vp])
for _n in ("orbit_head_loss_workspace_bytes", "orbit_head_loss_bwd_workspace_bytes", "orbit_head_loss_saved_bytes"):
    _proto(_n, _sz, [C.POINTER(orbit_head_desc)])
_proto("orbit_block_fwd", C.c_int,
       [C.POINTER(orbit_block_desc), _vp, C.POINTER(orbit_block_params), _vp, _vp, _vp, _sz, _vp])
_proto("orbit_block_bwd", C.c_int,
       [C.POINTER(orbit_block_desc), _vp, C.POINTER(orbit_block_params), _vp, _vp, C.POINTER(orbit_block_grads), _vp,
        _sz, _vp])
for _n in ("orbit_block_fwd_workspace_bytes", "orbit_block_bwd_workspace_bytes", "orbit_block_saved_bytes"):
    _proto(_n, _sz, [C.POINTER(orbit_block_desc)])
_proto("orbit_chain_fwd", C.c_int, [C.c_int] * 5 + [C.c_int, _vp, C.POINTER(_vp), C.POINTER(_vp), _vp, _vp, _sz, _vp])
_proto("orbit_chain_bwd", C.c_int, [C.c_int] * 5 + [C.c_int, _vp, C.POINTER(_vp), C.POINTER(_vp), _vp, _vp, _sz, _vp])
_proto("orbit_chain_workspace_bytes", _sz, [C.c_int] * 5 + [C.c_int])
_proto("orbit_mse_loss_grad", C.c_int, [C.c_int, _sz, _vp, _vp, _vp, _vp, _vp])
_proto("orbit_profile_gemm", C.c_int, [C.c_int])
_proto("orbit_profile_gemm_collect", C.c_int, [C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_longlong)])
_proto("orbit_profile_collect", C.c_int, [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_longlong)])
_proto("orbit_debug_gemm", C.c_int, [C.c_int] * 4 + [_vp, C.c_longlong, C.c_longlong, _vp, C.c_longlong, C.c_longlong, _vp, _vp])
_ll = C.c_longlong
_proto("orbit_debug_gemm_batched", C.c_int, [C.c_int] * 5 + [_vp, _ll, _ll, _ll, _vp, _ll, _ll, _ll, _vp, _ll, _ll, _vp])
_proto("orbit_debug_gemm_out", C.c_int, [C.c_int] * 4 + [_vp, _ll, _ll, _vp, _ll, _ll, C.c_int, _vp, _ll, _vp, _vp])
_proto("orbit_debug_layernorm_fwd", C.c_int, [C.c_int] * 5 + [C.c_float] + [_vp] * 7)
_proto("orbit_debug_layernorm_bwd", C.c_int, [C.c_int] * 7 + [_vp] * 11)

EXPORTS = ["orbit_tokenize", "orbit_tokenize_bwd", "orbit_tokenize_bwd_workspace_bytes", "orbit_var_aggregate",
           "orbit_var_aggregate_bwd", "orbit_var_aggregate_workspace_bytes",
           "orbit_var_aggregate_bwd_workspace_bytes", "orbit_var_aggregate_saved_bytes", "orbit_block_fwd",
           "orbit_block_bwd", "orbit_block_fwd_workspace_bytes", "orbit_block_bwd_workspace_bytes",
           "orbit_block_saved_bytes", "orbit_mse_loss_grad", "orbit_chain_fwd", "orbit_chain_bwd", "orbit_chain_workspace_bytes",
           "orbit_last_error", "orbit_version", "orbit_launch_count", "orbit_reset_launch_count",
           "orbit_debug_gemm", "orbit_profile_gemm",
           "orbit_profile_gemm_collect", "orbit_profile_collect", "orbit_embed_fused", "orbit_embed_fused_bwd",
           "orbit_embed_fused_workspace_bytes", "orbit_embed_fused_bwd_workspace_bytes",
           "orbit_embed_fused_saved_bytes", "orbit_debug_gemm_batched", "orbit_head_loss", "orbit_head_loss_bwd",
           "orbit_head_loss_workspace_bytes", "orbit_head_loss_bwd_workspace_bytes", "orbit_head_loss_saved_bytes",
           "orbit_debug_layernorm_fwd", "orbit_debug_layernorm_bwd", "orbit_debug_gemm_out",
           "orbit_rank_fwd_attn", "orbit_rank_fwd_mlp", "orbit_rank_fwd_out", "orbit_rank_bwd_mlp", "orbit_rank_bwd_attn",
           "orbit_rank_bwd_out", "orbit_rank_saved_bytes", "orbit_rank_bwd_workspace_bytes",
           "orbit_grads_unscale_check", "orbit_grads_accumulate", "orbit_grad_scale_update",
           "orbit_tokenize_bwd_noalloc", "orbit_tokenize_bwd_noalloc_max_bytes"]


# ---- marshalling helpers --------------------------------------------------------------------------------------
def _ptr(t):
    if t is None:
        return None
    if isinstance(t, int):
        return t
    assert t.is_cuda and t.is_contiguous(), "device-resident contiguous tensor required"
    return t.data_ptr()


def _stream(stream=None):
    s = stream if stream is not None else torch.cuda.current_stream()
    return s.cuda_stream


def _check(status, where):
    if status != ORBIT_OK:
        raise OrbitError(status, where)


def embed_desc(B, V, Hg, Wg, p, D, dtype):
    return orbit_embed_desc(B, V, Hg, Wg, p, D, DTYPES[dtype])


def agg_desc(B, L, V, D, heads, dtype, resid_dtype):
    return orbit_agg_desc(B, L, V, D, heads, DTYPES[dtype], DTYPES[resid_dtype])


def front_desc(B, V, Hg, Wg, p, D, heads, dtype, resid_dtype):
    return orbit_front_desc(B, V, Hg, Wg, p, D, heads, DTYPES[dtype], DTYPES[resid_dtype])


def head_desc(B, V, Hg, Wg, p, D, ln_eps, dtype, resid_dtype):
    return orbit_head_desc(B, V, Hg, Wg, p, D, ln_eps, DTYPES[dtype], DTYPES[resid_dtype])


def block_desc(B, N, D, heads, F, T=1, ln_eps=1e-5, dtype="bf16", resid_dtype="bf16", flags=0):
    return orbit_block_desc(B, N, D, heads, F, T, ln_eps, DTYPES[dtype], DTYPES[resid_dtype], flags)


def _agg_struct(cls, P):
    return cls(*[_ptr(P[n]) for n in _AGG_NAMES])


def _block_struct(cls, common, shards):
    arr = (orbit_block_shard * len(shards))(*[orbit_block_shard(*[_ptr(S[n]) for n in _SHARD_NAMES]) for S in shards])
    st = cls(*[_ptr(common[n]) for n in _COMMON_NAMES], arr, *[_ptr(common.get(n)) for n in _QKN_NAMES])
    st._keep = arr
    return st


# ---- entry points (same names as the C-ABI) ------------------------------------------------------------------
def orbit_tokenize(d, x, Wp, bp, tok, stream=None):
    _check(lib.orbit_tokenize(C.byref(d), _ptr(x), _ptr(Wp), _ptr(bp), _ptr(tok), _stream(stream)), "orbit_tokenize")


def orbit_tokenize_bwd_workspace_bytes(d):
    return lib.orbit_tokenize_bwd_workspace_bytes(C.byref(d))


def orbit_tokenize_bwd(d, x, dtok, dWp, dbp, ws, stream=None):
    _check(lib.orbit_tokenize_bwd(C.byref(d), _ptr(x), _ptr(dtok), _ptr(dWp), _ptr(dbp), _ptr(ws), ws.numel() * ws.element_size(),
                                  _stream(stream)), "orbit_tokenize_bwd")


def orbit_tokenize_bwd_noalloc_max_bytes():
    return lib.orbit_tokenize_bwd_noalloc_max_bytes()


def orbit_tokenize_bwd_noalloc(d, x, dtok, dWp, dbp, stream=None):
    """orbit_tokenize_bwd with the workspace inside the library (include/orbit.h): no allocation on the path."""
    _check(lib.orbit_tokenize_bwd_noalloc(C.byref(d), _ptr(x), _ptr(dtok), _ptr(dWp), _ptr(dbp), _stream(stream)),
           "orbit_tokenize_bwd_noalloc")


def orbit_var_aggregate_saved_bytes(d):
    return lib.orbit_var_aggregate_saved_bytes(C.byref(d))


def orbit_var_aggregate_workspace_bytes(d):
    return lib.orbit_var_aggregate_workspace_bytes(C.byref(d))


def orbit_var_aggregate_bwd_workspace_bytes(d):
    return lib.orbit_var_aggregate_bwd_workspace_bytes(C.byref(d))


def orbit_var_aggregate(d, tok, P, pos, agg, saved, ws, stream=None):
    ps = _agg_struct(orbit_agg_params, P)
    _check(lib.orbit_var_aggregate(C.byref(d), _ptr(tok), C.byref(ps), _ptr(pos), _ptr(agg), _ptr(saved), _ptr(ws),
                                   ws.numel() * ws.element_size(), _stream(stream)), "orbit_var_aggregate")


def orbit_var_aggregate_bwd(d, tok, P, dagg, saved, dtok, G, dpos, ws, stream=None):
    ps = _agg_struct(orbit_agg_params, P)
    gs = _agg_struct(orbit_agg_grads, G)
    _check(lib.orbit_var_aggregate_bwd(C.byref(d), _ptr(tok), C.byref(ps), _ptr(dagg), _ptr(saved), _ptr(dtok),
                                       C.byref(gs), _ptr(dpos), _ptr(ws), ws.numel() * ws.element_size(),
                                       _stream(stream)), "orbit_var_aggregate_bwd")


def orbit_embed_fused_saved_bytes(d):
    return lib.orbit_embed_fused_saved_bytes(C.byref(d))


def orbit_embed_fused_workspace_bytes(d):
    return lib.orbit_embed_fused_workspace_bytes(C.byref(d))


def orbit_embed_fused_bwd_workspace_bytes(d):
    return lib.orbit_embed_fused_bwd_workspace_bytes(C.byref(d))


def orbit_embed_fused(d, x, Wp, bp, P, pos, agg, saved, ws, stream=None):
    ps = _agg_struct(orbit_agg_params, P)
    _check(lib.orbit_embed_fused(C.byref(d), _ptr(x), _ptr(Wp), _ptr(bp), C.byref(ps), _ptr(pos), _ptr(agg), _ptr(saved),
                                 _ptr(ws), ws.numel() * ws.element_size(), _stream(stream)), "orbit_embed_fused")


def orbit_embed_fused_bwd(d, x, Wp, bp, P, dagg, saved, dWp, dbp, G, dpos, ws, stream=None):
    ps = _agg_struct(orbit_agg_params, P)
    gs = _agg_struct(orbit_agg_grads, G)
    _check(lib.orbit_embed_fused_bwd(C.byref(d), _ptr(x), _ptr(Wp), _ptr(bp), C.byref(ps), _ptr(dagg), _ptr(saved),
                                     _ptr(dWp), _ptr(dbp), C.byref(gs), _ptr(dpos), _ptr(ws),
                                     ws.numel() * ws.element_size(), _stream(stream)), "orbit_embed_fused_bwd")


def orbit_head_loss_saved_bytes(d):
    return lib.orbit_head_loss_saved_bytes(C.byref(d))


def orbit_head_loss_workspace_bytes(d):
    return lib.orbit_head_loss_workspace_bytes(C.byref(d))


def orbit_head_loss_bwd_workspace_bytes(d):
    return lib.orbit_head_loss_bwd_workspace_bytes(C.byref(d))


def orbit_head_loss(d, z, lnf_g, lnf_b, Wh, bh, target, latw, pred, loss, saved, ws, stream=None):
    _check(lib.orbit_head_loss(C.byref(d), _ptr(z), _ptr(lnf_g), _ptr(lnf_b), _ptr(Wh), _ptr(bh), _ptr(target), _ptr(latw),
                               _ptr(pred), _ptr(loss), _ptr(saved), _ptr(ws), ws.numel() * ws.element_size(),
                               _stream(stream)), "orbit_head_loss")


def orbit_head_loss_bwd(d, z, lnf_g, Wh, saved, dz, dlnf_g, dlnf_b, dWh, dbh, ws, stream=None):
    _check(lib.orbit_head_loss_bwd(C.byref(d), _ptr(z), _ptr(lnf_g), _ptr(Wh), _ptr(saved), _ptr(dz), _ptr(dlnf_g),
                                   _ptr(dlnf_b), _ptr(dWh), _ptr(dbh), _ptr(ws), ws.numel() * ws.element_size(),
                                   _stream(stream)), "orbit_head_loss_bwd")


def orbit_block_saved_bytes(d):
    return lib.orbit_block_saved_bytes(C.byref(d))


def orbit_block_fwd_workspace_bytes(d):
    return lib.orbit_block_fwd_workspace_bytes(C.byref(d))


def orbit_block_bwd_workspace_bytes(d):
    return lib.orbit_block_bwd_workspace_bytes(C.byref(d))


def orbit_block_fwd(d, x, common, shards, y, saved, ws, stream=None):
    """common: dict ln1_g, ln1_b, ln2_g, ln2_b, bproj, bfc2; shards: list of T dicts Wqkv, bqkv, Wproj, Wfc1, bfc1, Wfc2."""
    ps = _block_struct(orbit_block_params, common, shards)
    _check(lib.orbit_block_fwd(C.byref(d), _ptr(x), C.byref(ps), _ptr(y), _ptr(saved), _ptr(ws),
                               ws.numel() * ws.element_size(), _stream(stream)), "orbit_block_fwd")


def orbit_block_bwd(d, dy, common, shards, saved, dx, gcommon, gshards, ws, stream=None):
    ps = _block_struct(orbit_block_params, common, shards)
    gs = _block_struct(orbit_block_grads, gcommon, gshards)
    _check(lib.orbit_block_bwd(C.byref(d), _ptr(dy), C.byref(ps), _ptr(saved), _ptr(dx), C.byref(gs), _ptr(ws),
                               ws.numel() * ws.element_size(), _stream(stream)), "orbit_block_bwd")


# ---- rank-local Hybrid-STOP program: `shard` / `gshard` are THIS rank's shard dicts, `part` the fp32 [B,N,D] partial the
# caller all-reduces between the calls (include/orbit.h)
def orbit_rank_saved_bytes(d):
    return lib.orbit_rank_saved_bytes(C.byref(d))


def orbit_rank_bwd_workspace_bytes(d):
    return lib.orbit_rank_bwd_workspace_bytes(C.byref(d))


def orbit_rank_fwd_attn(d, x, common, shard, part, saved, stream=None):
    ps = _block_struct(orbit_block_params, common, [shard])
    _check(lib.orbit_rank_fwd_attn(C.byref(d), _ptr(x), C.byref(ps), _ptr(part), _ptr(saved), _stream(stream)),
           "orbit_rank_fwd_attn")


def orbit_rank_fwd_mlp(d, common, shard, part, saved, stream=None):
    ps = _block_struct(orbit_block_params, common, [shard])
    _check(lib.orbit_rank_fwd_mlp(C.byref(d), C.byref(ps), _ptr(part), _ptr(saved), _stream(stream)), "orbit_rank_fwd_mlp")


def orbit_rank_fwd_out(d, common, shard, part, y, saved, stream=None):
    ps = _block_struct(orbit_block_params, common, [shard])
    _check(lib.orbit_rank_fwd_out(C.byref(d), C.byref(ps), _ptr(part), _ptr(y), _ptr(saved), _stream(stream)),
           "orbit_rank_fwd_out")


def orbit_rank_bwd_mlp(d, dy, common, shard, saved, gcommon, gshard, part, ws, stream=None):
    ps = _block_struct(orbit_block_params, common, [shard])
    gs = _block_struct(orbit_block_grads, gcommon, [gshard])
    _check(lib.orbit_rank_bwd_mlp(C.byref(d), _ptr(dy), C.byref(ps), _ptr(saved), C.byref(gs), _ptr(part), _ptr(ws),
                                  ws.numel() * ws.element_size(), _stream(stream)), "orbit_rank_bwd_mlp")


def orbit_rank_bwd_attn(d, dy, common, shard, saved, gcommon, gshard, part, ws, stream=None):
    ps = _block_struct(orbit_block_params, common, [shard])
    gs = _block_struct(orbit_block_grads, gcommon, [gshard])
    _check(lib.orbit_rank_bwd_attn(C.byref(d), _ptr(dy), C.byref(ps), _ptr(saved), C.byref(gs), _ptr(part), _ptr(ws),
                                   ws.numel() * ws.element_size(), _stream(stream)), "orbit_rank_bwd_attn")


def orbit_rank_bwd_out(d, common, shard, saved, gcommon, gshard, part, dx, ws, stream=None):
    ps = _block_struct(orbit_block_params, common, [shard])
    gs = _block_struct(orbit_block_grads, gcommon, [gshard])
    _check(lib.orbit_rank_bwd_out(C.byref(d), C.byref(ps), _ptr(saved), C.byref(gs), _ptr(part), _ptr(dx), _ptr(ws),
                                  ws.numel() * ws.element_size(), _stream(stream)), "orbit_rank_bwd_out")


# ---- dynamic gradient scaling / fp32 accumulation: lists of gradient tensors of one dtype
def _counts(ts):
    return (_sz * len(ts))(*[t.numel() for t in ts])


def orbit_grads_unscale_check(grads, dtype, scale, found_inf, stream=None):
    """grads: list of device tensors of `dtype`, unscaled in place by 1 / scale[0]; found_inf[0] <- 1.0 on Inf / NaN."""
    _check(lib.orbit_grads_unscale_check(len(grads), _ptr_array(grads), _counts(grads), DTYPES[dtype], _ptr(scale),
                                         _ptr(found_inf), _stream(stream)), "orbit_grads_unscale_check")


def orbit_grads_accumulate(grads, acc, dtype, scale=None, found_inf=None, stream=None):
    """acc[i] (fp32) += grads[i] / scale[0]."""
    _check(lib.orbit_grads_accumulate(len(grads), _ptr_array(grads), _ptr_array(acc), _counts(grads), DTYPES[dtype],
                                      _ptr(scale), _ptr(found_inf), _stream(stream)), "orbit_grads_accumulate")


def orbit_grad_scale_update(scale, growth_tracker, found_inf, growth_factor, backoff_factor, growth_interval, stream=None):
    _check(lib.orbit_grad_scale_update(_ptr(scale), _ptr(growth_tracker), _ptr(found_inf), growth_factor, backoff_factor,
                                       growth_interval, _stream(stream)), "orbit_grad_scale_update")


def _ptr_array(ts):
    return (_vp * len(ts))(*[_ptr(t) for t in ts])


def orbit_chain_workspace_bytes(m, d, n, e, T, dtype):
    return lib.orbit_chain_workspace_bytes(m, d, n, e, T, DTYPES[dtype])


def orbit_chain_fwd(m, d, n, e, T, dtype, x, A_cols, B_rows, y, ws, stream=None):
    _check(lib.orbit_chain_fwd(m, d, n, e, T, DTYPES[dtype], _ptr(x), _ptr_array(A_cols), _ptr_array(B_rows), _ptr(y),
                               _ptr(ws), ws.numel() * ws.element_size(), _stream(stream)), "orbit_chain_fwd")


def orbit_chain_bwd(m, d, n, e, T, dtype, dy, A_cols, B_rows, dx, ws, stream=None):
    _check(lib.orbit_chain_bwd(m, d, n, e, T, DTYPES[dtype], _ptr(dy), _ptr_array(A_cols), _ptr_array(B_rows), _ptr(dx),
                               _ptr(ws), ws.numel() * ws.element_size(), _stream(stream)), "orbit_chain_bwd")


def orbit_mse_loss_grad(dtype, y, t, dy, loss, stream=None):
    _check(lib.orbit_mse_loss_grad(DTYPES[dtype], y.numel(), _ptr(y), _ptr(t), _ptr(dy), _ptr(loss), _stream(stream)),
           "orbit_mse_loss_grad")


def orbit_debug_gemm(M, N, K, dtype, A, a_rs, a_cs, B, b_rs, b_cs, Cout, stream=None):
    _check(lib.orbit_debug_gemm(M, N, K, DTYPES[dtype], _ptr(A), a_rs, a_cs, _ptr(B), b_rs, b_cs, _ptr(Cout),
                                _stream(stream)), "orbit_debug_gemm")


def orbit_debug_gemm_batched(M, N, K, batch, dtype, A, a_rs, a_cs, a_bs, B, b_rs, b_cs, b_bs, Cout, ldc, c_bs, stream=None):
    _check(lib.orbit_debug_gemm_batched(M, N, K, batch, DTYPES[dtype], _ptr(A), a_rs, a_cs, a_bs, _ptr(B), b_rs, b_cs, b_bs,
                                        _ptr(Cout), ldc, c_bs, _stream(stream)), "orbit_debug_gemm_batched")


def orbit_debug_gemm_out(M, N, K, dtype, A, a_rs, a_cs, B, b_rs, b_cs, out_dtype, Cout, ldc, bias=None, stream=None):
    _check(lib.orbit_debug_gemm_out(M, N, K, DTYPES[dtype], _ptr(A), a_rs, a_cs, _ptr(B), b_rs, b_cs, DTYPES[out_dtype],
                                    _ptr(Cout), ldc, _ptr(bias), _stream(stream)), "orbit_debug_gemm_out")


def orbit_debug_layernorm_fwd(M, D, x_dt, p_dt, out_dt, eps, x, gamma, beta, out, mean, rstd, stream=None):
    _check(lib.orbit_debug_layernorm_fwd(M, D, DTYPES[x_dt], DTYPES[p_dt], DTYPES[out_dt], eps, _ptr(x), _ptr(gamma),
                                         _ptr(beta), _ptr(out), _ptr(mean), _ptr(rstd), _stream(stream)),
           "orbit_debug_layernorm_fwd")


def orbit_debug_layernorm_bwd(M, D, dout_dt, x_dt, p_dt, add_dt, out_dt, dout, x, mean, rstd, gamma, add, dx_f32, dx_out,
                              dgamma_acc, dbeta_acc, stream=None):
    _check(lib.orbit_debug_layernorm_bwd(M, D, DTYPES[dout_dt], DTYPES[x_dt], DTYPES[p_dt], DTYPES[add_dt], DTYPES[out_dt],
                                         _ptr(dout), _ptr(x), _ptr(mean), _ptr(rstd), _ptr(gamma), _ptr(add), _ptr(dx_f32),
                                         _ptr(dx_out), _ptr(dgamma_acc), _ptr(dbeta_acc), _stream(stream)),
           "orbit_debug_layernorm_bwd")


def orbit_profile_gemm(on: bool):
    _check(lib.orbit_profile_gemm(1 if on else 0), "orbit_profile_gemm")


PROF_GEMM, PROF_ATTN_FWD, PROF_ATTN_BWD, PROF_LN, PROF_FRONT = range(5)


def orbit_profile_collect(category):
    """(summed kernel ms, summed algorithmic work, launches) of one category of the per-launch event record."""
    ms, wk, n = C.c_double(), C.c_double(), C.c_longlong()
    _check(lib.orbit_profile_collect(category, C.byref(ms), C.byref(wk), C.byref(n)), "orbit_profile_collect")
    return ms.value, wk.value, n.value


def orbit_profile_gemm_collect():
    ms, fl, n = C.c_double(0), C.c_double(0), C.c_longlong(0)
    _check(lib.orbit_profile_gemm_collect(C.byref(ms), C.byref(fl), C.byref(n)), "orbit_profile_gemm_collect")
    return ms.value, fl.value, n.value


def orbit_version():
    return lib.orbit_version()


def orbit_launch_count():
    return lib.orbit_launch_count()


def orbit_reset_launch_count():
    lib.orbit_reset_launch_count()


def orbit_set_debug_force_simt(mode: int):
    """A/B switch of the debug build only (ORBIT_LIB=dbg); the product library has a single dispatch."""
    if not HAS_DEBUG_SWITCH:
        raise RuntimeError("orbit_set_debug_force_simt: not in this build; build with ORBIT_DEBUG_SWITCH=1 and run with "
                           "ORBIT_LIB=dbg (A/B comparisons only)")
    lib.orbit_set_debug_force_simt(int(mode))
