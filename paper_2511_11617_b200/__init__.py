"""B200-native Elastic-TP state resharding (AnchorTP's CMM hot path, arxiv 2511.11617).

The product is the C-ABI library ``libetp.so`` (``include/etp.h``, sources in ``csrc/``); this package is its thin
ctypes binding.  Nothing here falls back to the CPU, and nothing here imports ``oracle/``.
"""
from .binding import *  # noqa: F401,F403
from .binding import lib, EXPORTS  # noqa: F401
