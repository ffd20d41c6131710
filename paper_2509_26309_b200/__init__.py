"""tbpm-b200: B200-native (sm_100a) hot path of TBPLaS 2.0's tight-binding propagation method.

The product is the C-ABI library `libtbpm.so` (include/tbpm.h, csrc/); `tbpm` is its thin Python binding
(argument marshalling only) and `workloads` the seeded input generators.  Nothing here imports `oracle/`.
"""
__all__ = ["tbpm", "workloads"]
