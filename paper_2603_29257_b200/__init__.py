"""B200-native TDA-risp sigma-build (arxiv/paper_2603_29257): thin Python binding of librisp.so.

All arithmetic of the method runs in the CUDA kernels of `csrc/` behind the C ABI of `include/risp.h`;
this package only marshals arguments (ctypes) and uses PyTorch for device memory and streams.
There is no CPU fallback: every call raises if the CUDA library is missing or fails.
"""
from .binding import (RispContext, RispError, load_library, setup, library_path, EXPORTED_SYMBOLS)  # noqa: F401
