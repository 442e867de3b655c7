"""plspec -- B200-native spectral integration of coded radar echoes (arXiv 2311.18737).

The product is the C-ABI library ``libplspec.so`` (``include/plspec.h``); this package holds
its CUDA sources (``csrc/``), a thin ctypes binding with the same names (``binding``) and
the seeded synthetic-input generators (``synth``).  The binding loads the CUDA library on
first use and fails loudly if it is missing -- there is no CPU fallback.
"""
__all__ = ["binding", "synth"]
