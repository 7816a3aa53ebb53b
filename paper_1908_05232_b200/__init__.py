"""B200-native coupled flood-pedestrian timestep (arXiv 1908.05232).

`scenarios` holds the seeded synthetic inputs; `binding` is the thin ctypes layer over the
C-ABI CUDA library `libfloodped.so` (include/floodped.h).  Importing the package is cheap and
does not load the CUDA library; the first `Sim(...)` does, and fails loudly if it is missing.
"""
__all__ = ["scenarios", "binding"]
