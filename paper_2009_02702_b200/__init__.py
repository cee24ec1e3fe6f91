"""B200-native transfer-function propagation path of the Mixture Graph (arXiv 2009.02702).

The package is deliberately thin: ``mg`` is the ctypes binding of the C-ABI library
(``include/mg.h``), ``builder`` the binding of the host-side graph builder
(``include/mg_builder.h``) and ``synth`` the seeded input generators.  Nothing here
imports ``oracle/`` and nothing is imported implicitly, so that ``synth`` can be used by
the oracle's tests without touching the CUDA library.
"""

__all__ = ["mg", "builder", "synth"]
