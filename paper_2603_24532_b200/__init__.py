"""B200-native normal ordering of the chiral N2LO three-nucleon force (arxiv/paper_2603_24532).

The product is the C-ABI CUDA library libno3n.so (include/no.h); this package holds its sources
(csrc/), the build step (build.py), a ctypes binding with the same names (binding.py), a small
convenience wrapper over torch tensors (api.py) and the seeded synthetic workloads
(workloads.py).  The CPU oracle under /oracle is test infrastructure and is never imported here.
"""
from . import binding, workloads  # noqa: F401
from .api import NormalOrdering  # noqa: F401
