"""Sketch&Walk Attention hot path for NVIDIA B200 (sm_100a): hand-written CUDA kernels behind the
C ABI of ``include/sw.h`` (``libsw.so``), a ctypes binding with the same names, and a thin per-layer
driver.  Importing the package loads ``libsw.so``; there is no CPU or PyTorch fallback."""
from .binding import *  # noqa: F401,F403
from .binding import Layout, SwError, make_layout, EXPORTS, LIB_PATH  # noqa: F401
from .pipeline import DecodePipeline, PrefillPipeline  # noqa: F401
