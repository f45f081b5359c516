"""B200-native CloakLM cloaked-layout hot path: ctypes binding of the C-ABI CUDA library libcloak.so.

See include/cloak.h for the boundary and DESIGN.md for the design.  Importing `binding` requires the
built library (`python -m paper_2606_18400_b200.build`); there is no CPU fallback.
"""
from .binding import *  # noqa: F401,F403
from .binding import (SYMBOLS, LIB_PATH, CloakError, cloak_block_shape, cloak_tensor, lib)  # noqa: F401
