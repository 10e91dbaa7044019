"""B200-native forward/adjoint operator pair for transcranial PACT (arXiv 1709.02733).

`paper_1709_02733_b200.binding` is the thin ctypes layer over the C-ABI library
`libpact.so` (include/pact.h); `paper_1709_02733_b200.synth` builds seeded synthetic inputs.
Importing the package does not load the CUDA library; `binding.lib()` does, and raises if it is
missing (there is no CPU fallback).
"""

__all__ = ["binding", "synth"]
