"""B200-native null-geodesic tracer (arXiv 2310.15183 hot path): ctypes binding of libgp.so.

Importing the package loads (building in-tree with nvcc if needed) the CUDA library; there is
no fallback path.
"""
from .api import *  # noqa: F401,F403
from . import api  # noqa: F401
