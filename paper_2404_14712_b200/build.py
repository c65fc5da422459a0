"""In-tree build of liborbit.so (and nothing else) with nvcc for sm_100a.

    python -m paper_2404_14712_b200.build [--force]
    ORBIT_DEBUG_SWITCH=1 python -m paper_2404_14712_b200.build      # A/B build: liborbit_dbg.so (csrc/orbit_debug.h)

The library has no torch dependency: plain CUDA runtime, C-ABI (include/orbit.h).  nvcc cross-compiles
without a GPU.  Object files are cached under csrc/build/ keyed by source mtime.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "liborbit.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr", "-Xptxas", "-v"]


def _sources():
    return sorted(f for f in os.listdir(CSRC) if f.endswith(".cu"))


def _headers_mtime():
    hs = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    hs.append(os.path.join(HERE, "..", "include", "orbit.h"))
    return max(os.path.getmtime(h) for h in hs)


def _compile(src, obj, log, extra=()):
    cmd = [NVCC, *FLAGS, *extra, "-c", os.path.join(CSRC, src), "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    with open(log, "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed on {src}:\n{r.stdout}\n{r.stderr}")
    return src


def build(force: bool = False, verbose: bool = True, debug_switch: bool | None = None) -> str:
    """debug_switch (default: env ORBIT_DEBUG_SWITCH=1) builds liborbit_dbg.so with -DORBIT_DEBUG_SWITCH: the kernel-variant
    A/B switch of csrc/orbit_debug.h.  The product library has no such switch."""
    if debug_switch is None:
        debug_switch = os.environ.get("ORBIT_DEBUG_SWITCH") == "1"
    bdir = os.path.join(CSRC, "build_dbg" if debug_switch else "build")
    out = os.path.join(HERE, "liborbit_dbg.so") if debug_switch else OUT
    extra = ["-DORBIT_DEBUG_SWITCH"] if debug_switch else []
    if debug_switch:                               # measurement probes of the A/B build only, e.g. ORBIT_NVCC_EXTRA=-DORBIT_PROBE_NOEXP
        extra += os.environ.get("ORBIT_NVCC_EXTRA", "").split()
    os.makedirs(bdir, exist_ok=True)
    hm = _headers_mtime()
    todo, objs = [], []
    for src in _sources():
        obj = os.path.join(bdir, src[:-3] + ".o")
        objs.append(obj)
        sm = max(os.path.getmtime(os.path.join(CSRC, src)), hm)
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < sm:
            todo.append((src, obj, os.path.join(bdir, src[:-3] + ".log")))
    if todo:
        if verbose:
            print(f"[orbit build] nvcc sm_100a: {', '.join(t[0] for t in todo)}", file=sys.stderr)
        with ThreadPoolExecutor(max_workers=min(8, len(todo))) as ex:
            list(ex.map(lambda t: _compile(*t, extra=extra), todo))
    if todo or not os.path.exists(out) or any(os.path.getmtime(o) > os.path.getmtime(out) for o in objs):
        cmd = [NVCC, "-shared", "-o", out, *objs, "-gencode", "arch=compute_100a,code=sm_100a", "-lcudart"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
