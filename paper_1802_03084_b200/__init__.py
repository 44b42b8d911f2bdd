"""B200-native realfast search hot path (arXiv 1802.03084): thin Python binding over the
C-ABI library ``librealfast_b200.so`` (see include/realfast.h).  No CPU fallback."""
from .binding import (  # noqa: F401
    CAND_DTYPE,
    Plan,
    RealfastError,
    lib_path,
    load_library,
    meansub_static,
)
