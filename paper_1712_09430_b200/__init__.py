"""B200-native Phase-I TPC sector tracker (arxiv 1712.09430): CUDA kernels behind a C ABI (include/tpctrk.h).

``binding`` mirrors the C calls one-to-one; ``build`` compiles ``csrc/`` into ``libtpctrk.so`` for sm_100a.
Importing this package does not load the library; the first ``binding.lib()`` / ``Tracker`` does, and fails
loudly if it cannot (no CPU fallback exists).
"""
from . import build  # noqa: F401
from .binding import Tracker, TpcError, default_params, tpc_params  # noqa: F401
