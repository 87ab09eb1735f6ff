"""B200-native spin spherical harmonic and Wigner transforms (hot path of arXiv 2311.14670).

The transforms run only through the CUDA library (csrc/ -> libb200sht.so, C ABI in include/b200sht.h); there is
no CPU fallback.  Importing the package does not load the library; the first transform call does and raises
if it is missing.
"""
from . import synth  # noqa: F401
