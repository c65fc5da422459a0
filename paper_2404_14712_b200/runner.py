"""Sequencing of the C-ABI calls for a whole ORBIT step (the public Python API a user calls).

No arithmetic lives here: tensors are allocated with torch (device memory only), parameters are copied to
the device, and the liborbit entry points are called in order on the current stream:
    orbit_tokenize -> orbit_var_aggregate -> depth x orbit_block_fwd -> orbit_mse_loss_grad
    -> depth x orbit_block_bwd -> orbit_var_aggregate_bwd -> orbit_tokenize_bwd
(SURVEY.md §3(ii)).
"""
from __future__ import annotations

import numpy as np
import torch

from . import binding as ob
from .inputs import Config

TD = ob.TORCH_DTYPES


def to_dev(a: np.ndarray, dtype: str, device="cuda") -> torch.Tensor:
    """numpy (float32 holding storage-exact values) -> device tensor of the storage dtype."""
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(device=device, dtype=TD[dtype]).contiguous()


def to_np(t: torch.Tensor) -> np.ndarray:
    return t.detach().to(torch.float32).cpu().numpy()


def _bytes(n, device="cuda"):
    return torch.empty(max(int(n), 256), dtype=torch.uint8, device=device)


class BlockRunner:
    """One ViT block (optionally Hybrid-STOP sharded) behind orbit_block_fwd / orbit_block_bwd."""

    COMMON = ob._COMMON_NAMES
    SHARD = ob._SHARD_NAMES

    def __init__(self, B, N, D, heads, F, T, dtype, resid_dtype, common: dict, shards: list, ln_eps=1e-5,
                 device="cuda", recompute=False):
        """QK-LayerNorm (ORBIT_QK_NORM) is switched on by the presence of qn_g, qn_b, kn_g, kn_b in `common`;
        recompute=True sets ORBIT_RECOMPUTE (activation checkpointing)."""
        self.qk_norm = "qn_g" in common
        flags = (ob.ORBIT_QK_NORM if self.qk_norm else 0) | (ob.ORBIT_RECOMPUTE if recompute else 0)
        self.desc = ob.block_desc(B, N, D, heads, F, T, ln_eps, dtype, resid_dtype, flags)
        self.B, self.N, self.D, self.heads, self.F, self.T = B, N, D, heads, F, T
        self.dtype, self.resid_dtype, self.device = dtype, resid_dtype, device
        names = self.COMMON + (ob._QKN_NAMES if self.qk_norm else ())
        self.common = {k: to_dev(common[k], dtype, device) for k in names}
        self.shards = [{k: to_dev(S[k], dtype, device) for k in self.SHARD} for S in shards]
        self.gcommon = {k: torch.empty_like(v) for k, v in self.common.items()}
        self.gshards = [{k: torch.empty_like(v) for k, v in S.items()} for S in self.shards]
        self.saved = _bytes(ob.orbit_block_saved_bytes(self.desc), device)
        self.ws_f = _bytes(ob.orbit_block_fwd_workspace_bytes(self.desc), device)
        self.ws_b = None
        self.y = torch.empty(B, N, D, dtype=TD[resid_dtype], device=device)
        self.dx = torch.empty(B, N, D, dtype=TD[resid_dtype], device=device)

    def share_bwd_ws(self, ws):
        self.ws_b = ws

    def fwd(self, x):
        ob.orbit_block_fwd(self.desc, x, self.common, self.shards, self.y, self.saved, self.ws_f)
        return self.y

    def bwd(self, dy):
        if self.ws_b is None:
            self.ws_b = _bytes(ob.orbit_block_bwd_workspace_bytes(self.desc), self.device)
        ob.orbit_block_bwd(self.desc, dy, self.common, self.shards, self.saved, self.dx, self.gcommon, self.gshards,
                           self.ws_b)
        return self.dx


class RankBlockRunner:
    """One rank of a tensor-parallel group running the rank-local Hybrid-STOP program (orbit_rank_*):
    six C-ABI calls with four all-reduce(sum) of the fp32 [B, N, D] partial in between.  `allreduce(t)` sums the tensor
    `t` in place over the group (default: torch.distributed.all_reduce on the default group -- NCCL over NVLink on a
    multi-GPU node, gloo in the tests).  `shard` is THIS rank's shard dict."""

    COMMON = ob._COMMON_NAMES
    SHARD = ob._SHARD_NAMES

    def __init__(self, B, N, D, heads, F, T, dtype, resid_dtype, common: dict, shard: dict, allreduce=None, ln_eps=1e-5,
                 device="cuda"):
        self.qk_norm = "qn_g" in common
        self.desc = ob.block_desc(B, N, D, heads, F, T, ln_eps, dtype, resid_dtype, ob.ORBIT_QK_NORM if self.qk_norm else 0)
        names = self.COMMON + (ob._QKN_NAMES if self.qk_norm else ())
        self.common = {k: to_dev(common[k], dtype, device) for k in names}
        self.shard = {k: to_dev(shard[k], dtype, device) for k in self.SHARD}
        self.gcommon = {k: torch.empty_like(v) for k, v in self.common.items()}
        self.gshard = {k: torch.empty_like(v) for k, v in self.shard.items()}
        self.saved = _bytes(ob.orbit_rank_saved_bytes(self.desc), device)
        self.ws = _bytes(ob.orbit_rank_bwd_workspace_bytes(self.desc), device)
        self.part = torch.empty(B, N, D, dtype=torch.float32, device=device)
        self.y = torch.empty(B, N, D, dtype=TD[resid_dtype], device=device)
        self.dx = torch.empty(B, N, D, dtype=TD[resid_dtype], device=device)
        if allreduce is None:
            import torch.distributed as dist
            allreduce = dist.all_reduce
        self.allreduce = allreduce
        self.partials = None          # optional dict: copies of this rank's pre-all-reduce partials (tests)

    def _reduce(self, name):
        if self.partials is not None:
            self.partials[name] = self.part.clone()
        self.allreduce(self.part)

    def fwd(self, x):
        ob.orbit_rank_fwd_attn(self.desc, x, self.common, self.shard, self.part, self.saved)
        self._reduce("proj")
        ob.orbit_rank_fwd_mlp(self.desc, self.common, self.shard, self.part, self.saved)
        self._reduce("fc2")
        ob.orbit_rank_fwd_out(self.desc, self.common, self.shard, self.part, self.y, self.saved)
        return self.y

    def bwd(self, dy):
        ob.orbit_rank_bwd_mlp(self.desc, dy, self.common, self.shard, self.saved, self.gcommon, self.gshard, self.part, self.ws)
        self._reduce("dm")
        ob.orbit_rank_bwd_attn(self.desc, dy, self.common, self.shard, self.saved, self.gcommon, self.gshard, self.part, self.ws)
        self._reduce("da")
        ob.orbit_rank_bwd_out(self.desc, self.common, self.shard, self.saved, self.gcommon, self.gshard, self.part, self.dx, self.ws)
        return self.dx


class FrontRunner:
    """orbit_tokenize + orbit_var_aggregate and their backward."""

    def __init__(self, B, V, Hg, Wg, p, D, heads, dtype, resid_dtype, emb: dict, agg: dict, pos=None, device="cuda"):
        self.L = (Hg // p) * (Wg // p)
        self.ed = ob.embed_desc(B, V, Hg, Wg, p, D, dtype)
        self.ad = ob.agg_desc(B, self.L, V, D, heads, dtype, resid_dtype)
        self.dtype, self.resid_dtype, self.device = dtype, resid_dtype, device
        self.Wp, self.bp = to_dev(emb["Wp"], dtype, device), to_dev(emb["bp"], dtype, device)
        self.agg = {k: to_dev(agg[k], dtype, device) for k in ob._AGG_NAMES}
        self.pos = None if pos is None else to_dev(pos, resid_dtype, device)
        self.tok = torch.empty(B, self.L, V, D, dtype=TD[dtype], device=device)
        self.out = torch.empty(B, self.L, D, dtype=TD[resid_dtype], device=device)
        self.saved = _bytes(ob.orbit_var_aggregate_saved_bytes(self.ad), device)
        self.ws_f = _bytes(ob.orbit_var_aggregate_workspace_bytes(self.ad), device)
        self.ws_b = None
        self.dtok = None
        self.gagg = {k: torch.empty_like(v) for k, v in self.agg.items()}
        self.dpos = None if pos is None else torch.empty_like(self.pos)
        self.dWp, self.dbp = torch.empty_like(self.Wp), torch.empty_like(self.bp)
        self.ws_t = _bytes(ob.orbit_tokenize_bwd_workspace_bytes(self.ed), device)

    def fwd(self, x):
        ob.orbit_tokenize(self.ed, x, self.Wp, self.bp, self.tok)
        ob.orbit_var_aggregate(self.ad, self.tok, self.agg, self.pos, self.out, self.saved, self.ws_f)
        return self.out

    def bwd(self, dagg):
        if self.ws_b is None:
            self.ws_b = _bytes(ob.orbit_var_aggregate_bwd_workspace_bytes(self.ad), self.device)
            self.dtok = torch.empty_like(self.tok)
        ob.orbit_var_aggregate_bwd(self.ad, self.tok, self.agg, dagg, self.saved, self.dtok, self.gagg, self.dpos,
                                   self.ws_b)
        ob.orbit_tokenize_bwd(self.ed, self.x_last, self.dtok, self.dWp, self.dbp, self.ws_t)

    def fwd_keep(self, x):
        self.x_last = x
        return self.fwd(x)


class FusedFrontRunner:
    """orbit_embed_fused and its backward: tokenise + aggregate in pixel space, tok never materialised."""

    def __init__(self, B, V, Hg, Wg, p, D, heads, dtype, resid_dtype, emb: dict, agg: dict, pos=None, device="cuda"):
        self.L = (Hg // p) * (Wg // p)
        self.fd = ob.front_desc(B, V, Hg, Wg, p, D, heads, dtype, resid_dtype)
        self.dtype, self.resid_dtype, self.device = dtype, resid_dtype, device
        self.Wp, self.bp = to_dev(emb["Wp"], dtype, device), to_dev(emb["bp"], dtype, device)
        self.agg = {k: to_dev(agg[k], dtype, device) for k in ob._AGG_NAMES}
        self.pos = None if pos is None else to_dev(pos, resid_dtype, device)
        self.out = torch.empty(B, self.L, D, dtype=TD[resid_dtype], device=device)
        self.saved = _bytes(ob.orbit_embed_fused_saved_bytes(self.fd), device)
        self.ws_f = _bytes(ob.orbit_embed_fused_workspace_bytes(self.fd), device)
        self.ws_b = None
        self.gagg = {k: torch.empty_like(v) for k, v in self.agg.items()}
        self.dpos = None if pos is None else torch.empty_like(self.pos)
        self.dWp, self.dbp = torch.empty_like(self.Wp), torch.empty_like(self.bp)

    def fwd_keep(self, x):
        self.x_last = x
        ob.orbit_embed_fused(self.fd, x, self.Wp, self.bp, self.agg, self.pos, self.out, self.saved, self.ws_f)
        return self.out

    def bwd(self, dagg):
        if self.ws_b is None:
            self.ws_b = _bytes(ob.orbit_embed_fused_bwd_workspace_bytes(self.fd), self.device)
        ob.orbit_embed_fused_bwd(self.fd, self.x_last, self.Wp, self.bp, self.agg, dagg, self.saved, self.dWp, self.dbp,
                                 self.gagg, self.dpos, self.ws_b)


class HeadRunner:
    """orbit_head_loss / orbit_head_loss_bwd: final LayerNorm, image-space head, latitude-weighted MSE."""

    NAMES = ("lnf_g", "lnf_b", "Wh", "bh")

    def __init__(self, B, V, Hg, Wg, p, D, dtype, resid_dtype, head: dict, ln_eps=1e-5, device="cuda", keep_pred=True):
        self.hd = ob.head_desc(B, V, Hg, Wg, p, D, ln_eps, dtype, resid_dtype)
        L = (Hg // p) * (Wg // p)
        self.P = {k: to_dev(head[k], dtype, device) for k in self.NAMES}
        self.G = {k: torch.empty_like(v) for k, v in self.P.items()}
        self.saved = _bytes(ob.orbit_head_loss_saved_bytes(self.hd), device)
        self.ws_f = _bytes(ob.orbit_head_loss_workspace_bytes(self.hd), device)
        self.ws_b = _bytes(ob.orbit_head_loss_bwd_workspace_bytes(self.hd), device)
        self.pred = torch.empty(B, V, Hg, Wg, dtype=torch.float32, device=device) if keep_pred else None
        self.loss = torch.zeros(1, dtype=torch.float32, device=device)
        self.dz = torch.empty(B, L, D, dtype=TD[resid_dtype], device=device)

    def loss_and_grad(self, z, target_img, latw=None):
        ob.orbit_head_loss(self.hd, z, self.P["lnf_g"], self.P["lnf_b"], self.P["Wh"], self.P["bh"], target_img, latw,
                           self.pred, self.loss, self.saved, self.ws_f)
        ob.orbit_head_loss_bwd(self.hd, z, self.P["lnf_g"], self.P["Wh"], self.saved, self.dz, self.G["lnf_g"],
                               self.G["lnf_b"], self.G["Wh"], self.G["bh"], self.ws_b)
        return self.loss, self.dz


class StepRunner:
    """Whole hot path for a Config: tokenise -> aggregate -> depth x block, forward + backward, MSE loss."""

    def __init__(self, cfg: Config, emb=None, agg=None, blocks=None, pos=None, device="cuda", fused_front=False,
                 head=None):
        self.cfg = cfg
        self.front = None
        self.head = None
        if head is not None:
            self.head = HeadRunner(cfg.B, cfg.V, cfg.Hg, cfg.Wg, cfg.p, cfg.D, cfg.dtype, cfg.resid_dtype, head, cfg.ln_eps,
                                   device)
        if cfg.V is not None:
            self.front = (FusedFrontRunner if fused_front else FrontRunner)(cfg.B, cfg.V, cfg.Hg, cfg.Wg, cfg.p, cfg.D, cfg.heads, cfg.dtype, cfg.resid_dtype,
                                     emb, agg, pos, device)
        self.blocks = []
        ws = None
        for common, shards in blocks:
            br = BlockRunner(cfg.B, cfg.L, cfg.D, cfg.heads, cfg.F, cfg.T, cfg.dtype, cfg.resid_dtype, common, shards,
                             cfg.ln_eps, device)
            if ws is None:
                ws = _bytes(ob.orbit_block_bwd_workspace_bytes(br.desc), device)
            br.share_bwd_ws(ws)
            self.blocks.append(br)
        self.loss = torch.zeros(1, dtype=torch.float32, device=device)
        self.dy = torch.empty(cfg.B, cfg.L, cfg.D, dtype=TD[cfg.resid_dtype], device=device)

    def forward(self, x):
        h = self.front.fwd_keep(x) if self.front is not None else x
        for b in self.blocks:
            h = b.fwd(h)
        return h

    def backward(self, dy):
        g = dy
        for b in reversed(self.blocks):
            g = b.bwd(g)
        if self.front is not None:
            self.front.bwd(g)
        return g

    def step_head(self, x, target_img):
        """The paper's training step: ... -> blocks -> final LN + head -> latitude-weighted MSE and
        backward.  x, target_img: [B,V,Hg,Wg] fp32."""
        y = self.forward(x)
        loss, dz = self.head.loss_and_grad(y, target_img)
        self.backward(dz)
        return loss

    def capture(self, fn):
        """Capture one invocation of `fn` (a closure over this runner's calls and FIXED device tensors) into a CUDA
        graph and return its replay function.  Every C-ABI entry point only enqueues kernels on the caller's stream
        (no allocation, no host synchronisation; tensor maps travel by value as kernel parameters), so a whole step is
        capturable; replay removes the per-launch host work and most of the inter-kernel gaps of launch-bound shapes
        (C2: 330 launches per step).  Not usable together with orbit_profile_gemm (event timing cannot be captured)."""
        torch.cuda.synchronize()
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            fn()                                   # warm-up on the capture stream (first-use attribute calls)
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            fn()
        torch.cuda.synchronize()
        self._graphs = getattr(self, "_graphs", []) + [g]
        return g.replay

    def step(self, x, target):
        """x: fields [B,V,Hg,Wg] fp32 (or block input [B,N,D] for block-only configs); target [B,L,D]."""
        y = self.forward(x)
        ob.orbit_mse_loss_grad(self.cfg.resid_dtype, y, target, self.dy, self.loss)
        self.backward(self.dy)
        return self.loss
