"""B200-native Landau-de Gennes / FIRE hot path (arXiv:1911.07045), sm_100a only.

``lq`` (binding.py) is a thin ctypes layer over ``csrc/liblq.so``'s C ABI
(include/lq.h); ``workloads`` builds the seeded synthetic inputs.  There is no
CPU fallback: every ``lq_*`` call fails loudly if the CUDA library is missing.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "binding", "build"]
