"""Nekbone CG hot path on one B200 (sm_100a), fp64: hand-written CUDA behind the C-ABI of include/nk.h.

`Nekbone` is the thin binding (argument marshalling only).  The package never imports `oracle`
and has no CPU fallback: without libnk.so, `load()` raises.
"""
from .binding import (Nekbone, NkError, load, workspace_bytes, SIGNATURES, LIB_PATH,
                      NK_OK, NK_ERR_ARG, NK_ERR_WORKSPACE, NK_ERR_ID, NK_ERR_MASK, NK_ERR_GEOM,
                      NK_ERR_CUDA, NK_ERR_ALLOC, NK_ERR_MULT)

__all__ = ["Nekbone", "NkError", "load", "workspace_bytes", "SIGNATURES", "LIB_PATH"]
