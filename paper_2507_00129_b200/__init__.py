"""B200-native Lyman-alpha forest pixel-pair correlator (xi and distortion matrix).

The product is the C-ABI library `liblya.so` (include/lya.h, csrc/*.cu); this
package is the thin ctypes binding over it plus the seeded input generator.
Importing the package does not load the library; `paper_2507_00129_b200.binding`
does, and fails loudly if it has not been built (there is no CPU fallback).
"""
__all__ = ["gen", "binding", "build", "shard"]
