"""B200-native SPH + shear-strength time step (arxiv/paper_2603_19764, section 2).

The package holds the CUDA kernels + C-ABI library (``csrc/``), a thin ctypes
binding with the same names (``binding.py``) and the seeded synthetic input
generators (``workloads.py``).  Importing the package does not load the CUDA
library; ``binding.load()`` does, and fails loudly if it is missing.
"""

__all__ = ["binding", "workloads"]
