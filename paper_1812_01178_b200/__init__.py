"""tdx: B200-native batched tridiagonal line solves (PDD / PPT / cyclic) after Ha, Park & You,
arxiv 1812.01178 (Algorithm 1).

The package holds only what the hot path needs:
  inputs.py   seeded synthetic grids / right-hand sides (no method arithmetic; serves tests, oracle callers and bench)
  configs.py  the five BASELINE.json workloads as data
  binding.py  ctypes marshalling onto the C-ABI library csrc/libtdx.so (declared in include/tdx.h)
  build.py    nvcc build step for csrc/libtdx.so (sm_100a)
Nothing here imports `oracle/`; the product path fails loudly when libtdx.so is missing.
"""
__all__ = ["inputs", "configs", "binding", "build"]
