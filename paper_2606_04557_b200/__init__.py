"""paper_2606_04557_b200: B200-native (sm_100a) hot path of "Cartridges at Scale" multi-cartridge
training behind a C ABI (include/cas.h).  `from paper_2606_04557_b200 import cas` gives the ctypes
binding; the library is loaded lazily on first call and there is no CPU fallback."""
from . import cas  # noqa: F401

__all__ = ["cas"]
