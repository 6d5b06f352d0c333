"""B200-native hot path of arXiv:1005.3276: CG on M^dag M with the overlap fermion
matrix applied through hand-written sm_100a 4D FFT kernels (C ABI: include/wz.h)."""
from . import inputs  # noqa: F401

__all__ = ["inputs", "wz", "build"]
