"""tj -- B200-native pseudo-C_ell mode-coupling matrices (arxiv/paper_2602_15605).

The product is the C-ABI library `libtj.so` (include/tj.h, csrc/); `binding` is the thin Python
front-end with the same names.  Importing the package does not load the library; calling any
entry point does, and fails loudly if it is missing -- there is no CPU fallback.
"""
from . import windows  # noqa: F401
from .binding import (  # noqa: F401
    TJError,
    Tables,
    build_tables,
    coupling_tt,
    coupling_pol,
    coupling_band,
    l3_range,
    load_library,
    library_path,
)
