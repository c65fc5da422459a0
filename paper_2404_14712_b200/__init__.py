"""orbit-b200: B200-native per-GPU training step of ORBIT's ClimaX-style ViT (arxiv 2404.14712).

The package holds only what the hot path needs:
  csrc/       hand-written CUDA (sm_100a) kernels + the C-ABI of include/orbit.h
  binding.py  thin ctypes marshalling over liborbit.so (same names as the C entry points)
  inputs.py   seeded synthetic input recipes (no method arithmetic; shared with the tests)
  build.py    in-tree nvcc build of liborbit.so

Nothing here imports `oracle/` (test infrastructure) and there is no CPU fallback:
`binding` raises if liborbit.so is missing.
"""
__all__ = ["binding", "inputs", "build"]
