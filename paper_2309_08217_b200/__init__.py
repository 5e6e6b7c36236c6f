"""B200-native (sm_100a) hot path of the GENGA hybrid symplectic N-body step (arXiv 2309.08217).

``binding``   -- ctypes binding of the C-ABI library ``libgenga_b200.so`` (include/genga.h)
``workloads`` -- seeded synthetic inputs for the BASELINE.json configs (no method arithmetic)
``build``     -- nvcc build of the CUDA library for sm_100a

Importing this package does not load the CUDA library; ``binding.load()`` does, and fails loudly
if it is missing.  There is no CPU fallback.
"""
__all__ = ["binding", "workloads", "build"]
