"""B200-native batched per-agent perspective renderer (Gigapixel hot path, arxiv/paper_2606_19641).

`gp` is the thin ctypes binding of the C-ABI library declared in include/gp.h; every step of the
path runs in the library's sm_100a kernels.  There is no CPU fallback.
"""
from . import gp  # noqa: F401
from .gp import Renderer, GpError  # noqa: F401
