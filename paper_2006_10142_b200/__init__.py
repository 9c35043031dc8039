"""B200-native ADI time stepping for the 2D acoustic wave equation (arxiv 2006.10142 hot path).

`Wave2D` is a thin ctypes binding over the C ABI in include/wave2d.h (libwave2d.so, hand-written CUDA
for sm_100a).  Importing this package does not load the shared library; constructing a `Wave2D` does,
and fails loudly if the library or a CUDA device is missing -- there is no CPU fallback.
"""
from .binding import Wave2D, Wave2DError, library_path, load_library  # noqa: F401
