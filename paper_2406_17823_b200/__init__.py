"""paper_2406_17823_b200 -- B200-native QTT/MPS time-step algebra (arxiv 2406.17823).

The product is the C-ABI library ``libqtt_b200.so`` (include/qtt.h); this package holds its CUDA
sources (``csrc/``), the in-tree build step (``build.py``) and a thin ctypes binding
(``binding.py``) with the same call names.  Importing the binding without the built library, or
without a CUDA device, fails loudly -- there is no CPU fallback.
"""
from .binding import *  # noqa: F401,F403
from .binding import Context, Mps, Mpo, QttError  # noqa: F401
