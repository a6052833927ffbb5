"""B200-native Wilson-Dirac matvec D*psi (eq. (2.2) of arXiv:0912.2186).

The product is the C-ABI library built from csrc/ (declared in include/wd.h); `binding`
is a thin ctypes layer with the same names, `fields` holds the seeded input generators.
Importing the package does not load the CUDA library; the first call does, and fails loudly
if the library has not been built (there is no CPU fallback).
"""
from . import fields  # noqa: F401
from . import binding  # noqa: F401
