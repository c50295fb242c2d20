"""B200-native charge-blocked two-site update of a U(1)-symmetric MPS (arXiv:2303.11409).

The package holds the CUDA kernels + C-ABI library (``csrc/``), a thin ctypes binding
(``binding.py``) and the seeded input generators (``inputs.py``).  Nothing is imported
eagerly: ``inputs`` holds none of the method's arithmetic and is shared with the test
oracle; ``binding`` loads ``libu1mps.so`` and fails loudly if it is missing.
"""

__all__ = ["inputs", "binding"]
