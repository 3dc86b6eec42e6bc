"""B200-native line-segment tracking (LST) hot path of arXiv:2403.13166.

Thin Python binding over the C-ABI library `liblst_b200.so` (include/lst.h).  Argument marshalling
only: every step of the path runs in the CUDA kernels.  There is no CPU fallback -- importing the
binding fails loudly when the library is missing, and it never touches `oracle/`.
"""
from .binding import (LST, Caps, load_library, library_path, OBJ, CNT, STATUS_BITS, LstError,
                      default_caps, pack_batch, lst_sort_hits_static)

__all__ = ["LST", "Caps", "load_library", "library_path", "OBJ", "CNT", "STATUS_BITS", "LstError",
           "default_caps", "pack_batch", "lst_sort_hits_static"]
