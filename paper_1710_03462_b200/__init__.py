"""paper_1710_03462_b200 -- B200-native SoAx hot path (arXiv 1710.03462).

csrc/ + include/soax.h: the C-ABI CUDA library (libsoax.so);  binding.py: ctypes binding with the same names;
container.py: torch-owned device memory around it;  inputs.py: seeded synthetic particle sets (no method arithmetic).
Importing this package does not load CUDA; `binding.lib()` does, and fails loudly if the library is missing.
"""
from . import inputs  # noqa: F401

__all__ = ["inputs", "binding", "container", "build"]
