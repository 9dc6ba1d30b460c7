"""B200-native per-cell implicit matter-radiation source update of arXiv 2407.18304.

The product is the C-ABI library built from csrc/ (declared in include/mgrhd.h); this
package is its thin Python binding plus the seeded workload generators.  There is no CPU
fallback: anything that computes goes through the CUDA library and fails loudly without it.
"""
__all__ = ["binding", "workloads"]
