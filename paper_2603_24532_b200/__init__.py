"""B200-native normal ordering of the chiral N2LO three-nucleon force (arxiv/paper_2603_24532).

The product is the C-ABI CUDA library libno3n.so (include/no.h); this package holds its sources
(csrc/), the build step (build.py), a ctypes binding with the same names (binding.py), a small
convenience wrapper over torch tensors (api.py) and the seeded synthetic workloads
(workloads.py, trace_workloads.py); include/no_trace.h declares the second workload, the spin-isospin
trace of a closed diagram over the matrices the first one produces.  The CPU oracle under /oracle is test infrastructure and is never imported here.
"""
from . import binding, trace_workloads, workloads  # noqa: F401
from .api import NormalOrdering, SpinIsospinTrace  # noqa: F401
