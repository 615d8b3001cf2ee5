"""B200-native recursive Green's function sweep for armchair graphene nanoribbons.

The product is the C-ABI library built from csrc/ (see include/rgf.h) and the thin ctypes
binding in .binding; `inputs` holds only the seeded synthetic workload generators.
Nothing is imported eagerly: `from paper_1107_5300_b200 import binding` loads the CUDA
library and fails loudly if it has not been built.
"""
__all__ = ["binding", "inputs"]
