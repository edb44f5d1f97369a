"""B200-native SPH density + hydro-force hot path (after arxiv 2003.10850).

`inputs` holds the seeded synthetic particle sets; `binding` is the thin ctypes layer over
the C-ABI library `libsph.so` (include/sph.h).  Nothing here falls back to a CPU path.
"""
__all__ = ["inputs", "binding"]
