"""B200-native Cornerstone octree construction (arXiv 2307.06345, single-GPU hot path).

The product is ``libcornerstone_b200.so`` (hand-written CUDA for sm_100a behind the C ABI of
``include/cornerstone.h``); this package is the thin Python binding over it.  PyTorch is used
only for device memory and streams.  There is no CPU fallback: every call fails loudly if the
shared library is missing.

    from paper_2307_06345_b200 import binding as cs
    ctx = cs.Context(max_particles=n, max_leaves=n // 4)
    tree = cs.buildOctree(ctx, x, y, z, bucketSize=64)

``workloads`` holds the seeded synthetic particle sets (shared with the test oracle; it
contains none of the method's arithmetic).
"""
__all__ = ["binding", "workloads", "build"]
