"""moto-b200: B200-native hot path of arxiv 2509.26269.

The product is the C-ABI library ``libmoto.so`` (include/moto.h); this package is the thin
ctypes binding around it plus the seeded workload generators.  The library is loaded lazily
and loudly: there is no CPU fallback.
"""
from .binding import *  # noqa: F401,F403
from .binding import load_library  # noqa: F401
