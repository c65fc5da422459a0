#!/usr/bin/env python
"""bench.py -- ORBIT hot path on B200: ViT block fwd+bwd bf16 TFLOP/s (BASELINE.json metric) on the 113B-class
block C5 (default), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C5|C4|C3|C2]

N > 1 (torchrun): replicas only -- the path does not shard across GPUs (north_star: no collectives); every rank
runs the same workload, timing is the max over ranks, value is the sum ("weak").
--impl reference: the fp64 CPU oracle, as it stands, on a bounded sample of the same workload (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2404_14712_b200 import inputs as syn  # noqa: E402

METRIC = "vit_block_fwd_bwd_bf16_tflops"
UNIT = "TFLOP/s"


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return dict(bf16=float(d["bf16_tflops"]), bf16_sustained=float(d.get("bf16_tflops_sustained", 0) or 0),
                        hbm=float(d["hbm_gbs"]), src="measured")
        except Exception:
            pass
    return dict(bf16=1590.0, bf16_sustained=1400.0, hbm=6650.0, src="fallback")


def workload_string(cfg):
    if cfg.V is None:
        return (f"{cfg.name}: one ViT block fwd+bwd, B={cfg.B} N={cfg.L} D={cfg.D} heads={cfg.heads} F={cfg.F} T={cfg.T} "
                f"{cfg.dtype}")
    return (f"{cfg.name}: tokenise+aggregate+{cfg.depth} blocks fwd+bwd, B={cfg.B} V={cfg.V} grid={cfg.Hg}x{cfg.Wg} p={cfg.p} "
            f"L={cfg.L} D={cfg.D} heads={cfg.heads} F={cfg.F} {cfg.dtype}")


def step_flops(cfg):
    """Model FLOPs of one step's blocks (2 per MAC; backward = 2x forward; no recompute) -- SURVEY.md §8(d)."""
    return 3.0 * cfg.block_flops_fwd() * cfg.depth


# ------------------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle on a bounded sample
# ------------------------------------------------------------------------------------------------------------
def oracle_sample(cfg, n_tokens, batch=1):
    """Block fwd+bwd of the oracle at cfg's widths on `batch` samples of n_tokens tokens.  Returns a closure running one
    sample step and the sample's model FLOPs.  Weights are widened to float64 outside the timed call (input
    preparation, not arithmetic of the method)."""
    from oracle import orbit_oracle as orc
    seed = syn.seed_of(cfg.name)
    P = syn.block_params(seed, cfg.D, cfg.F, cfg.dtype)
    P = {k: np.asarray(v, dtype=np.float64) for k, v in P.items()}
    x = np.asarray(syn.normal(seed, "blk.x", (batch, n_tokens, cfg.D), dtype=cfg.resid_dtype), dtype=np.float64)
    dy = np.asarray(syn.normal(seed, "blk.dy", (batch, n_tokens, cfg.D), dtype=cfg.resid_dtype), dtype=np.float64)
    flops = batch * 3.0 * (2.0 * n_tokens * cfg.D * (4 * cfg.D + 2 * cfg.F) + 4.0 * n_tokens * n_tokens * cfg.D)

    def run():
        y, cache = orc.block_fwd(x, P, cfg.heads, cfg.ln_eps)
        dx, G = orc.block_bwd(dy, P, cache)
        return float(y[0, 0, 0]) + float(dx[0, 0, 0])

    return run, flops


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [i.get("num_threads") for i in threadpool_info() if i.get("user_api") == "blas"]
        if n:
            return int(max(n))
    except Exception:
        pass
    return os.cpu_count() or 1


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # a step of the reference arm = the oracle on a bounded sample: 256 tokens at the 113B-class width (~4 s per step),
    # one whole sample (L tokens) at the smaller widths
    n_tok = 256 if cfg.D >= 8192 else (512 if cfg.D >= 4096 else cfg.L)
    run, flops = oracle_sample(cfg, n_tok)
    for _ in range(args.warmup):
        run()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        run()
    dt = (time.perf_counter() - t0) / args.steps
    val = flops / dt / 1e12
    sample = f"oracle block fwd+bwd at {cfg.name} widths on {n_tok} of {cfg.L} tokens (B=1), fp64 numpy/OpenBLAS"
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_string(cfg), "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": blas_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-i", str(gpu_index), "-lms", "20"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    # the sampler is started before the warm-up (nvidia-smi takes a few hundred ms to print its first line); only the
    # samples whose timestamp falls inside [begin, end] -- host times taken right after the barriers that bracket the
    # timed region -- are used (all samples if the region was shorter than the sampling period)
    def begin(self):
        import datetime
        self.t0 = datetime.datetime.now()

    def end(self):
        import datetime
        self.t1 = datetime.datetime.now()

    def stop(self):
        import datetime
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        rows = []
        for ln in self.f.read().splitlines():
            c = [t.strip() for t in ln.split(",")]
            if len(c) < 8:
                continue
            try:
                ts = datetime.datetime.strptime(c[0], "%Y/%m/%d %H:%M:%S.%f")
                rows.append((ts, float(c[1]), float(c[2]), float(c[3]), c[4:8]))
            except ValueError:
                continue
        t0, t1 = getattr(self, "t0", None), getattr(self, "t1", None)
        inside = [r for r in rows if t0 is not None and t1 is not None and t0 <= r[0] <= t1]
        if not inside:
            inside = rows
        sm, mx, reasons, pw = [], [], set(), []
        for _, a, b, c3, flags in inside:
            sm.append(a); mx.append(b); pw.append(c3)
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), flags):
                if v.lower().startswith("active"):
                    reasons.add(name)
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if sm:
            out = {"sm_mhz": float(np.median(sm)), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                   "power_w_max": max(pw), "samples": len(sm)}
        return out


class HostPipeline:
    """The end-to-end leg's input / output plumbing: every step copies its inputs from pinned host memory and its
    results back to pinned host memory, as a training loop with a prefetching loader does -- the copies run on their
    own streams and overlap the neighbouring steps' kernels.  Inputs are double buffered on the device (step i+1's
    batch lands while step i computes); results are snapshotted device-to-device on the compute stream (so the next
    step may overwrite them) and drained to the host on the read-back stream.  Every copy of every step is inside
    the timed region: finish() makes the compute stream wait for the last read-back before the closing event."""

    def __init__(self, host_in, host_out):
        import torch
        self.torch = torch
        self.host_in, self.host_out = host_in, host_out
        self.h2d, self.d2h = torch.cuda.Stream(), torch.cuda.Stream()
        self.slots = [[torch.empty(h.shape, dtype=h.dtype, device="cuda") for h in host_in] for _ in range(2)]
        self.stage = [torch.empty(h.shape, dtype=h.dtype, device="cuda") for h in host_out]
        self.slot_free = [None, None]
        self.drained = None
        self.i = 0

    def inputs(self):
        torch = self.torch
        cur = torch.cuda.current_stream()
        k = self.i % 2
        self.k = k
        with torch.cuda.stream(self.h2d):
            if self.slot_free[k] is not None:
                self.h2d.wait_event(self.slot_free[k])          # the step that last read this slot has finished
            for d, h in zip(self.slots[k], self.host_in):
                d.copy_(h, non_blocking=True)
            ready = torch.cuda.Event()
            ready.record(self.h2d)
        cur.wait_event(ready)
        return self.slots[k]

    def outputs(self, dev_out):
        torch = self.torch
        cur = torch.cuda.current_stream()
        if self.drained is not None:
            cur.wait_event(self.drained)                        # previous read-back has left the snapshot buffers
        for st, d in zip(self.stage, dev_out):
            st.copy_(d.view(st.shape), non_blocking=True)
        done = torch.cuda.Event()
        done.record(cur)
        self.slot_free[self.k] = done
        with torch.cuda.stream(self.d2h):
            self.d2h.wait_event(done)
            for h, st in zip(self.host_out, self.stage):
                h.copy_(st, non_blocking=True)
            self.drained = torch.cuda.Event()
            self.drained.record(self.d2h)
        self.i += 1

    def finish(self):
        if self.drained is not None:
            self.torch.cuda.current_stream().wait_event(self.drained)


def max_over_ranks(ms, world, device):
    """Replicas-only scaling: the step time of the job is the slowest rank's; every rank gets it."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(ms)], device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def run_ours(args, cfg):
    import torch
    import torch.distributed as dist
    from paper_2404_14712_b200 import binding as ob, runner as rn

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    seed = syn.seed_of(cfg.name)
    if args.debug_mode:
        ob.orbit_set_debug_force_simt(args.debug_mode)      # needs the A/B build: ORBIT_LIB=dbg

    # ---- build the workload (inputs resident in HBM) ----
    if cfg.V is None:
        P = syn.block_params(seed, cfg.D, cfg.F, cfg.dtype)
        sr = rn.StepRunner(cfg, blocks=[(P, syn.shard_block_params(P, cfg.heads, cfg.T))])
        del P
        x_h = syn.normal(seed, "blk.x", (cfg.B, cfg.L, cfg.D), dtype=cfg.resid_dtype)
        dy_h = syn.normal(seed, "blk.dy", (cfg.B, cfg.L, cfg.D), dtype=cfg.resid_dtype)
        x_d, dy_d = rn.to_dev(x_h, cfg.resid_dtype), rn.to_dev(dy_h, cfg.resid_dtype)

        def step():
            sr.forward(x_d)
            sr.backward(dy_d)
        tdt = ob.TORCH_DTYPES[cfg.resid_dtype]
        hx = torch.from_numpy(x_h).to(tdt).pin_memory()
        hdy = torch.from_numpy(dy_h).to(tdt).pin_memory()
        hy, hdx = torch.empty_like(hx).pin_memory(), torch.empty_like(hx).pin_memory()
        h2d = hx.numel() * hx.element_size() * 2
        d2h = h2d

        pipe = HostPipeline([hx, hdy], [hy, hdx])

        def step_e2e():
            xs, dys = pipe.inputs()
            sr.forward(xs)
            sr.backward(dys)
            pipe.outputs([sr.blocks[-1].y, sr.blocks[0].dx])
    else:
        emb = syn.embed_params(seed, cfg.V, cfg.p, cfg.D, cfg.dtype)
        agg = syn.agg_params(seed, cfg.D, cfg.dtype)
        blocks = []
        for i in range(cfg.depth):
            P = syn.block_params(seed, cfg.D, cfg.F, cfg.dtype, tag=f"blk{i}")
            blocks.append((P, syn.shard_block_params(P, cfg.heads, 1)))
        sr = rn.StepRunner(cfg, emb, agg, blocks, fused_front=args.front == "fused")
        del blocks
        x_h = syn.fields(seed, cfg.B, cfg.V, cfg.Hg, cfg.Wg, per_variable_scale=True)
        t_h = syn.normal(seed, "target", (cfg.B, cfg.L, cfg.D), dtype=cfg.resid_dtype)
        x_d, t_d = rn.to_dev(x_h, "f32"), rn.to_dev(t_h, cfg.resid_dtype)

        def step():
            sr.step(x_d, t_d)
        hx = torch.from_numpy(x_h).pin_memory()
        ht = torch.from_numpy(t_h).to(ob.TORCH_DTYPES[cfg.resid_dtype]).pin_memory()
        hloss = torch.zeros(1).pin_memory()
        h2d = hx.numel() * 4 + ht.numel() * ht.element_size()
        d2h = 4

        pipe = HostPipeline([hx, ht], [hloss])

        def step_e2e():
            xs, ts = pipe.inputs()
            sr.step(xs, ts)
            pipe.outputs([sr.loss])

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps, finish=None):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        for _ in range(steps):
            fn()
        if finish:
            finish()
        e1.record()
        barrier()
        return max_over_ranks(e0.elapsed_time(e1), world, "cuda")

    sampler = ClockSampler(local) if rank == 0 else None
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    # ---- timed region: device-resident inputs, EXACTLY args.steps steps, nothing but the product's own launches ----
    ob.orbit_reset_launch_count()
    if sampler:
        sampler.begin()
    ms = timed(step, args.steps)
    if sampler:
        sampler.end()
    launches = ob.orbit_launch_count()
    clocks = sampler.stop() if sampler else None
    # ---- roofline leg: the same args.steps steps again with a CUDA-event pair around every tensor-core GEMM launch (on the
    # launching stream).  Kept out of the headline region: ~200 event records per C2 step sit between dependent kernels and
    # switch off their programmatic-dependent-launch overlap (C2: 6.1 ms instrumented vs 5.3 ms plain).
    ob.orbit_profile_gemm(True)
    ms_instr = timed(step, args.steps)
    gemm_ms, gemm_flops, gemm_n = ob.orbit_profile_gemm_collect()
    secondary_raw = {name: ob.orbit_profile_collect(cat) for name, cat in
                     (("attention_fwd", ob.PROF_ATTN_FWD), ("attention_bwd", ob.PROF_ATTN_BWD), ("layernorm", ob.PROF_LN),
                      ("front_end", ob.PROF_FRONT))}
    ob.orbit_profile_gemm(False)
    # ---- optional: the same device-resident step replayed from a CUDA graph ----
    graph_ms = None
    if args.graph:
        replay = sr.capture(step)
        for _ in range(3):
            replay()
        graph_ms = timed(replay, args.steps) / args.steps
    # ---- end to end through the public API with host buffers ----
    for _ in range(2):
        step_e2e()
    ms_e2e = timed(step_e2e, args.steps, pipe.finish)

    flops = step_flops(cfg)
    ms_step = ms / args.steps
    tflops = flops / (ms_step * 1e-3) / 1e12 * world
    tflops_e2e = flops / (ms_e2e / args.steps * 1e-3) / 1e12 * world
    tokens_s = cfg.B * cfg.L / (ms_step * 1e-3) * world
    peaks = measured_peaks()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    achieved = gemm_flops / (gemm_ms * 1e-3) / 1e12 if gemm_ms > 0 else 0.0
    traffic = None
    tp = os.path.join(ROOT, "profiles", "roofline_traffic.csv")
    if os.path.exists(tp):
        try:
            import csv
            for row in csv.DictReader(open(tp)):
                if row["workload"] == cfg.name:
                    traffic = float(row["dram_bytes_per_launch"])
        except Exception:
            traffic = None
    roofline = {"bound": "tensor", "kernel": "gemm_tc2_kernel / gemm_tc_kernel (tcgen05 bf16 GEMM; every GEMM launch of the step)",
                # the GEMM launches are timed inside the long timed step (the power-capped regime), so the peak is the
                # SUSTAINED measured bf16 figure; the burst figure (a kernel timed alone) is given beside it
                "achieved": achieved, "peak": peaks["bf16_sustained"] or peaks["bf16"], "unit": "TFLOP/s",
                "frac": achieved / (peaks["bf16_sustained"] or peaks["bf16"]),
                "peak_source": f"{peaks['src']} sustained bf16 (MEASURED_PEAKS.json bf16_tflops_sustained: torch.matmul back to "
                               f"back for 4 s; kernels here are timed inside a long step)",
                "peak_burst": peaks["bf16"], "frac_of_burst": achieved / peaks["bf16"],
                "launches": gemm_n, "avg_launch_ms": gemm_ms / max(gemm_n, 1),
                "share_of_step": gemm_ms / ms_instr if ms_instr > 0 else None, "traffic": traffic,
                "measured_in": f"second timed pass of the same {args.steps} steps with a CUDA-event pair around every GEMM launch "
                               f"({ms_instr / args.steps:.3f} ms per instrumented step); share_of_step is relative to that pass",
                "timed_region_s": ms_instr * 1e-3}
    # secondary entries: the kernels that are NOT the dominant one, each against the roofline that bounds it (same
    # instrumented pass).  Tensor-bound: attention (4 B N^2 D FLOP forward, twice that backward); HBM-bound: LayerNorm
    # and the front-end streaming kernels (algorithmic bytes of DESIGN.md §5) against MEASURED_PEAKS.json hbm_gbs.
    secondary = []
    descr = {"attention_fwd": ("tensor", "attn_fwd_tc5_kernel (flash forward, tcgen05)"),
             "attention_bwd": ("tensor", "attn_delta5 + attn_bwd_dq_tc5 + attn_bwd_dkv_tc5 (flash backward, tcgen05; model FLOPs 8 B N^2 D)"),
             "layernorm": ("hbm", "ln_fwd_tma_* / ln_bwd_tma_* (TMA-staged LayerNorm forward and backward)"),
             "front_end": ("hbm", "front-end streaming kernels (tokenise / per-patch aggregation, or the pixel-space per-patch kernels)")}
    for name, (s_ms, s_work, s_n) in secondary_raw.items():
        if s_n == 0 or s_ms <= 0:
            continue
        bound, kern = descr[name]
        if bound == "tensor":
            ach, pk, unit = s_work / (s_ms * 1e-3) / 1e12, peaks["bf16"], "TFLOP/s"
            src = "measured burst bf16 (these kernels are short and not power capped)"
        else:
            ach, pk, unit = s_work / (s_ms * 1e-3) / 1e9, peaks["hbm"], "GB/s"
            src = "measured copy bandwidth (MEASURED_PEAKS.json hbm_gbs)"
        secondary.append({"name": name, "bound": bound, "kernel": kern, "achieved": ach, "peak": pk, "unit": unit,
                          "frac": ach / pk if pk else None, "peak_source": src, "launches": s_n,
                          "avg_launch_ms": s_ms / s_n, "share_of_step": s_ms / ms_instr if ms_instr > 0 else None})
    # ---- CPU baseline: the oracle on a bounded sample (rank 0, N = 1 only) ----
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        # about 10-30 s of CPU work: C5 1024 tokens, C4 one whole sample, C3 two samples, C2 the whole batch
        n_tok = 1024 if cfg.D >= 8192 else cfg.L
        nb = 1 if cfg.D >= 4096 else min(cfg.B, 2 if cfg.D >= 2048 else cfg.B)
        run, sflops = oracle_sample(cfg, n_tok, nb)
        t0 = time.perf_counter()
        run()
        dt = time.perf_counter() - t0
        cpu = {"value": sflops / dt / 1e12, "unit": UNIT, "cores": blas_threads(), "kind": "oracle",
               "sample": f"oracle block fwd+bwd at {cfg.name} widths on {nb} x {n_tok} of {cfg.B} x {cfg.L} tokens, fp64 "
                         f"numpy/OpenBLAS, {dt:.1f} s"}
    line = {
        "metric": METRIC, "value": tflops, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
        "data": "synthetic",
        "config": {"workload": workload_string(cfg), "l2": "inputs larger than L2 (weights + saved activations "
                   "streamed every step; no flush needed)", "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "front_end": (args.front if cfg.V is not None else None),
                   "model_flops_per_step": flops},
        "tokens_per_s": tokens_s,
        "frac_of_peak_measured_burst": tflops / world / peaks["bf16"],
        "frac_of_peak_measured_sustained": (tflops / world / peaks["bf16_sustained"]) if peaks["bf16_sustained"] else None,
        "frac_of_peak_nominal_2250": tflops / world / 2250.0,
        "clocks": clocks,
        "e2e": {"value": tflops_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": ms_e2e / args.steps,
                "overlap": "every step's H2D / D2H runs on copy streams (double-buffered inputs, snapshotted results) inside the timed region"},
        "gpu_launches": int(launches),
        **({"graph": {"ms_per_step": graph_ms, "value": flops / (graph_ms * 1e-3) / 1e12 * world, "unit": UNIT}} if graph_ms else {}),
        "roofline": roofline,
        "roofline_secondary": secondary,
        "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_hbm_probe():
    """Write-only, read-only and copy bandwidth of this GPU's HBM (torch fills / reductions / copies of 3 GiB buffers, best of
    10, CUDA events): the ceilings of kernels that only write (orbit_tokenize) or only read (orbit_tokenize_bwd) a large
    tensor.  MEASURED_PEAKS.json's hbm_gbs is the COPY figure (read + write bytes).  profiles/r2_hbm_probe.md."""
    import torch
    torch.cuda.set_device(0)
    n = 3 << 28                                               # 3 Gi bf16 elements... as int32: 3 GiB
    a = torch.empty(n, dtype=torch.int32, device="cuda")
    b = torch.empty(n, dtype=torch.int32, device="cuda")
    nbytes = n * 4

    def best(fn, moved):
        ts = []
        for _ in range(10):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fn(); e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        return moved / (min(ts) * 1e-3) / 1e9
    a.zero_(); b.zero_(); torch.cuda.synchronize()
    out = {"probe": "hbm", "buffer_bytes": nbytes,
           "write_only_gbs": best(lambda: a.zero_(), nbytes),
           "write_only_fill_gbs": best(lambda: a.fill_(7), nbytes),
           "read_only_gbs": best(lambda: a.sum(), nbytes),
           "copy_gbs": best(lambda: b.copy_(a), 2 * nbytes),
           "how": "torch zero_ / fill_ / sum / copy_ on 3 GiB int32 buffers, best of 10, CUDA events; copy counts read + write bytes"}
    pk = measured_peaks()
    out["measured_peaks_hbm_gbs"] = pk["hbm"]
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C5", choices=["C2", "C3", "C4", "C5", "P113", "P10B"],
                    help="C2..C5: BASELINE.json configs (default C5, the one the metric is quoted on); P113 / P10B: one block "
                         "of the paper's own 113B / 10B shapes (PAPER.md:140: d_h 192 / 256)")
    ap.add_argument("--front", default="fused", choices=["fused", "twocall"],
                    help="front end of C2/C3: orbit_embed_fused (pixel space, no tok tensor) or orbit_tokenize + "
                         "orbit_var_aggregate (tok materialised)")
    ap.add_argument("--graph", action="store_true",
                    help="additionally time the device-resident step replayed from a CUDA graph (reported as 'graph'; "
                         "the headline value and the roofline leg stay un-captured)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--debug-mode", type=int, default=0, help="kernel-variant switch of the A/B build (ORBIT_DEBUG_SWITCH=1 build, ORBIT_LIB=dbg); never set by the default run")
    ap.add_argument("--hbm-probe", action="store_true",
                    help="print the write-only / read-only / copy HBM bandwidth of cuda:0 (JSON) and exit")
    args = ap.parse_args()
    if args.hbm_probe:
        run_hbm_probe()
        return
    cfg = syn.CONFIGS[args.workload]
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
