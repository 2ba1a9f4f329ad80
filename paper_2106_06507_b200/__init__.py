"""B200-native Berends-Giele engine for all-gluon tree-level |M|^2 (arxiv 2106.06507).

``binding`` is the thin ctypes layer over the C-ABI in ``include/bg.h`` (CUDA kernels in ``csrc/``);
``workload`` holds the seeded synthetic input generators; ``build`` compiles ``libbg.so`` in-tree.
"""
from . import binding  # noqa: F401
from .binding import *  # noqa: F401,F403
