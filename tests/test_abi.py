"""CPU checks of the boundary: liborbit.so builds for sm_100a, loads, and exports every symbol that
include/orbit.h declares; argument validation that needs no GPU returns the documented codes."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2404_14712_b200 import build
    path = build.build(verbose=False)
    return ctypes.CDLL(path)


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "orbit.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(orbit_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_exported(lib):
    syms = declared_symbols()
    assert len(syms) >= 20
    for s in syms:
        assert hasattr(lib, s), f"{s} declared in include/orbit.h but not exported"


def test_binding_lists_same_symbols():
    from paper_2404_14712_b200 import binding
    assert sorted(binding.EXPORTS) == declared_symbols()
    assert binding.orbit_version() == 100


def test_size_queries_and_validation_without_gpu(lib):
    from paper_2404_14712_b200 import binding as ob
    d = ob.block_desc(1, 2048, 12288, 96, 49152)
    sv = ob.orbit_block_saved_bytes(d)
    # x, a, O, x1, m (5 x M*D) + qkv (3 M*D) + u, g (2 x M*F) bf16 + stats
    assert sv >= 2 * 2048 * (8 * 12288 + 2 * 49152)
    assert ob.orbit_block_bwd_workspace_bytes(d) > 0
    # NULL pointers and bad shapes are rejected before any CUDA call
    bad = ob.block_desc(1, 16, 64, 3, 128)
    lib.orbit_block_fwd.restype = ctypes.c_int
    assert lib.orbit_block_fwd(ctypes.byref(bad), None, None, None, None, None, 0, None) == 2   # ERR_SHAPE
    ok = ob.block_desc(1, 16, 64, 2, 128)
    assert lib.orbit_block_fwd(ctypes.byref(ok), None, None, None, None, None, 0, None) == 1    # ERR_NULL
    lib.orbit_last_error.restype = ctypes.c_char_p
    assert b"NULL" in lib.orbit_last_error()
    ok.flags = 8                                     # unknown flag bit
    assert lib.orbit_block_fwd(ctypes.byref(ok), None, None, None, None, None, 0, None) == 6    # ERR_UNSUPPORTED
    # ORBIT_RECOMPUTE keeps only the block input in `saved` and moves the forward state into the workspaces
    rc = ob.block_desc(1, 2048, 12288, 96, 49152, 1, 1e-5, "bf16", "bf16", ob.ORBIT_RECOMPUTE)
    assert ob.orbit_block_saved_bytes(rc) == 2048 * 12288 * 2
    assert ob.orbit_block_fwd_workspace_bytes(rc) >= ob.orbit_block_fwd_workspace_bytes(d) + sv
    assert ob.orbit_block_bwd_workspace_bytes(rc) >= ob.orbit_block_bwd_workspace_bytes(d) + sv
    # ORBIT_QK_NORM widens the qkv buffer by the normalised Q', K' copies and rejects unsupported head widths
    qn = ob.block_desc(1, 2048, 12288, 96, 49152, 1, 1e-5, "bf16", "bf16", ob.ORBIT_QK_NORM)
    assert ob.orbit_block_saved_bytes(qn) >= sv + 2 * 2048 * 12288 * 2
    odd = ob.block_desc(1, 16, 96, 2, 192, 1, 1e-5, "bf16", "bf16", ob.ORBIT_QK_NORM)     # d_h = 48
    assert lib.orbit_block_fwd(ctypes.byref(odd), None, None, None, None, None, 0, None) == 2   # ERR_SHAPE


def test_sass_is_sm100a(lib):
    """The shipped library holds sm_100a code only (no multi-arch fatbin)."""
    import subprocess
    from paper_2404_14712_b200 import build
    out = subprocess.run(["/usr/local/cuda/bin/cuobjdump", "--list-elf", build.OUT], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs
