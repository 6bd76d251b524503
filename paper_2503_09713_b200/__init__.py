"""B200-native SPH hot path of arXiv:2503.09713 (Shamrock/Phantom SPH): hand-written CUDA for sm_100a behind the
C ABI of ``include/sph_b200.h``; ``binding`` is the ctypes front-end, ``workloads`` the seeded input generators,
``build`` compiles ``libsph_b200.so`` in-tree. No CPU fallback exists: using ``binding.Sim`` without the built
library or without a CUDA device raises."""
from . import workloads  # noqa: F401  (NumPy only)

__all__ = ["workloads", "binding", "build"]
