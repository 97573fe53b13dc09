"""B200-native recursively executed hash-grid renderer (arXiv 2409.10327) -- thin Python binding over the
C-ABI CUDA library `libhashrender.so` (include/hashrender.h).  Argument marshalling only."""
from .binding import (HR_DIRECT, HR_SHADOW, HR_INDIRECT, HR_DENSE, HR_TERM_DIRECT, HR_TERM_INDIRECT, HashRenderError,
                      HashRenderer, DirSet, GBufferNet, load_library)

__all__ = ["HR_DIRECT", "HR_SHADOW", "HR_INDIRECT", "HR_DENSE", "HR_TERM_DIRECT", "HR_TERM_INDIRECT", "HashRenderError",
           "HashRenderer", "DirSet", "GBufferNet", "load_library"]
