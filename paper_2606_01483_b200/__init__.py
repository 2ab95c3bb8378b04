"""B200-native (sm_100a) MURMUR intra-chunk hot path: paged KV append, sliding-window eviction
and batched GQA decode attention behind the C ABI of include/murmur.h.

``binding.MurmurCache`` is the thin Python face of that ABI (argument marshalling only).
"""
from .binding import (MURMUR_ATTN_AUTO, MURMUR_ATTN_GENERIC, MURMUR_ATTN_MMA, MURMUR_OPT_ATTN_GRID, MURMUR_OPT_FUSE_STEP, MURMUR_OPT_PDL,
                      MURMUR_OPT_ATTN_VARIANT, MURMUR_WINDOW_OFF, MurmurCache, MurmurError, lib, version)

__all__ = ["MurmurCache", "MurmurError", "lib", "version", "MURMUR_WINDOW_OFF", "MURMUR_OPT_ATTN_VARIANT",
           "MURMUR_OPT_ATTN_GRID", "MURMUR_OPT_PDL", "MURMUR_OPT_FUSE_STEP", "MURMUR_ATTN_AUTO", "MURMUR_ATTN_GENERIC", "MURMUR_ATTN_MMA"]
