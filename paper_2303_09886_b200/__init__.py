"""B200-native F-engine (channelizer) data path of arxiv 2303.09886.

Thin ctypes binding over the C ABI of include/fengine.h (argument marshalling only: every step of
the path runs in the CUDA kernels under csrc/).  There is no CPU fallback: importing works without
a GPU (so the symbol table can be checked), but creating an engine fails loudly without a device or
without the built library.
"""
from .binding import (  # noqa: F401
    FEngine,
    FEngineError,
    lib,
    library_path,
    EXPORTED_SYMBOLS,
    fp32_rate,
    process_noalloc,
    NOALLOC_MAX_FLOATS,
)
