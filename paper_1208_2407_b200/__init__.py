"""B200-native second-order Trotter-Suzuki lattice step (arxiv/paper_1208_2407 hot path).

``binding`` is the thin ctypes layer over the C-ABI CUDA library ``libts.so`` (include/ts.h);
``inputs`` holds the seeded synthetic workloads (no method arithmetic).  Importing the package
does not load the library; ``binding.lib()`` does and fails loudly when it is missing.
"""
__all__ = ["binding", "inputs", "build"]
