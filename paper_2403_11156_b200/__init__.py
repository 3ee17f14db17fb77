"""B200-native DFSPH particle pipeline (arxiv 2403.11156 hot path).

`scenes` holds the seeded synthetic inputs; `binding` is the thin ctypes layer
over the C-ABI library `libsph_b200.so` (include/sph.h).  Nothing here falls
back to a CPU implementation: using `binding` without the built CUDA library
raises.
"""

__all__ = ["scenes", "binding", "build"]
