"""B200-native prefix-cached prefill path of CacheWeaver (arxiv/paper_2606_19667).

The product is the C-ABI library `libcacheweaver.so` (include/cacheweaver.h, csrc/); this package is its thin
Python binding plus a trace driver.  There is no CPU fallback: device calls need a CUDA device and the built
library.  Nothing here imports oracle/.
"""
from .binding import (ARMS, BLOCK_SIZE, CW_ERR_BAD_HANDLE, CW_ERR_CUDA, CW_ERR_INVALID, CW_ERR_NO_SPACE, CW_OK, EXPORTS,
                      LIB_PATH, Context, CwError, NoSpace, load_library)

__all__ = ["ARMS", "BLOCK_SIZE", "CW_OK", "CW_ERR_INVALID", "CW_ERR_NO_SPACE", "CW_ERR_BAD_HANDLE", "CW_ERR_CUDA", "EXPORTS",
           "LIB_PATH", "Context", "CwError", "NoSpace", "load_library"]
