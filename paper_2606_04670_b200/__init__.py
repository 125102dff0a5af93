"""paper_2606_04670_b200 -- B200-native (sm_100a) hot path of LipFit (arxiv/paper_2606_04670).

The product is the C-ABI library `liblipfit.so` (include/lipfit.h, sources in csrc/); this package
is its thin ctypes binding with the same entry-point names.
"""
from . import binding  # noqa: F401
from .binding import *  # noqa: F401,F403
from .binding import (LipfitError, bounds_variant, get_timing, knn_variant, launch_count, load,  # noqa: F401
                      pipe_throughput, release_workspace, set_timing, status_string, version)
