"""paper_1608_00386_b200 -- B200-native optical forward model of the MAORY MCAO simulator.

The product is libao.so (hand-written CUDA for sm_100a behind the C ABI of include/ao.h);
`binding` marshals torch tensors into it, `inputs` builds the seeded synthetic workloads.
Nothing here falls back to the CPU: the oracle under oracle/ is test infrastructure only.
"""
from . import inputs  # noqa: F401  (descriptors + seeded generators; no arithmetic of the method)

__all__ = ["inputs", "binding", "build"]
