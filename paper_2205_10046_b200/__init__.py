"""B200-native NEP3 hot path (arxiv 2205.10046): thin Python binding over the C-ABI CUDA library.

Every step of the path runs in the library's sm_100a kernels (csrc/); this package only marshals
arguments (torch tensors -> device pointers).  There is no CPU fallback: importing `binding` raises if
the shared library is missing.
"""
from .binding import (  # noqa: F401
    NEP, NepError, NepHyper, lib_path, lib_overridden, load_library, exported_symbols,
)
