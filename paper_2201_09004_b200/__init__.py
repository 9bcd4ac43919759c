"""B200-native twisted-mass Wilson(-clover) Dslash + even-odd mixed-precision BiCGStab (arXiv:2201.09004 Eqs. 1-3).

The product is the C-ABI library ``libtmw.so`` (include/tmw.h, sources in csrc/); ``tmw`` is its thin ctypes
binding. ``synth`` holds the seeded input generators (no method arithmetic). There is no CPU fallback: every call
of ``tmw`` fails loudly when the CUDA library is missing.
"""
