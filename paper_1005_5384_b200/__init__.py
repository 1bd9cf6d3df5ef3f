"""B200-native tree-code force calculation (hot path of arXiv 1005.5384).

Sub-modules: ``build`` (nvcc build of csrc/ -> libtc_b200.so), ``binding`` (ctypes
marshalling of include/tc.h), ``inputs`` (seeded synthetic workloads; shared with
the oracle, holds none of the method's arithmetic).  Nothing here imports
``oracle/``.
"""
__all__ = ["build", "binding", "inputs"]
