"""B200-native hot path of the metadynamics-of-paths method (arxiv 2501.11962).

The product is the C-ABI library `libmop_b200.so` built from `csrc/` (see
include/mop.h); `binding` is a thin ctypes layer with the same names, and
`workloads` holds the seeded synthetic input generators.  Nothing here falls
back to a CPU implementation: using the binding without the built CUDA library
raises.
"""
__all__ = ["binding", "workloads"]
