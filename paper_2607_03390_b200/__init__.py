"""B200-native TemporalGS hot path (arxiv/paper_2607_03390): thin Python binding of libtgs.so.

The binding only marshals arguments; every step of the path runs in the CUDA kernels of csrc/.
Importing this package does not load the library; `tgs.lib()` does and fails loudly when it is missing.
"""
from . import binding as tgs  # noqa: F401
from .binding import Context, TgsParams, TgsStats, TgsError  # noqa: F401
