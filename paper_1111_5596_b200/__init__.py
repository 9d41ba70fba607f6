"""paper_1111_5596_b200 -- B200-native site-parallel evaluation of QDP++-style lattice
expressions (arXiv:1111.5596).  Thin ctypes binding over ``libqdp_b200.so``
(C ABI: ``include/qdp_b200.h``).  PyTorch is used only for device memory and streams.

There is no CPU fallback: importing this package needs the built library
(``python -m paper_1111_5596_b200.build``), and every call needs a CUDA device.
"""
from .binding import *  # noqa: F401,F403
from .binding import __all__  # noqa: F401
