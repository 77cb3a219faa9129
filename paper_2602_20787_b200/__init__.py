"""B200-native direct-summation gravity for the StePS periodic-cylinder (S^1 x R^2) method.

The product is the C-ABI library `libsteps_cyl.so` (include/steps_cyl.h, csrc/) and the
thin ctypes binding in `binding.py`; `workloads.py` generates the seeded synthetic inputs.
Nothing here imports `oracle/`.
"""
__all__ = ["binding", "workloads", "build"]
