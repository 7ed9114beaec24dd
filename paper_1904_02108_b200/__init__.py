"""B200-native LBM-IBM time-step hot path (Beny & Latt, arXiv 1904.02108).

The package holds the CUDA kernels + C-ABI library (``csrc/``), its thin Python binding
(``api``) and the seeded workload generators (``workloads``, shared with the tests' oracle,
contains none of the method's arithmetic).  Importing the package does not load the CUDA
library; ``paper_1904_02108_b200.api`` does, and fails loudly when it is missing.
"""

__all__ = ["api", "workloads"]
