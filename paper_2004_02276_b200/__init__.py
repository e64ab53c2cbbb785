"""B200-native (sm_100a, fp64 CUDA) hot path of the STREAmS method (arXiv 2004.02276).

`paper_2004_02276_b200.binding` is the thin ctypes layer over the C-ABI library declared in
include/streams.h; the seeded synthetic inputs live outside the product, in the top-level `workloads` package.
"""
__all__ = ["binding", "build", "replicas"]
