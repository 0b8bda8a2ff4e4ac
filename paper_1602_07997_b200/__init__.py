"""B200-native nodal-DG hot path of arxiv 1602.07997 (acoustic + elastic RHS and
LSRK update on tetrahedra).  ``dg`` is the thin ctypes binding over the C-ABI
library ``libdg.so`` (include/dg.h); ``workloads`` holds the seeded input
generators.  Importing the package does not load the CUDA library; the first
use of ``dg`` does, and fails loudly if it is missing."""
__all__ = ["dg", "workloads"]
