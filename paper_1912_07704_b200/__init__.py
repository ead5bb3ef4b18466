"""B200-native dedispersion + single-pulse search: thin Python binding of the C-ABI library (include/aa.h).

Argument marshalling only — every step of the hot path runs in the CUDA kernels of ``libaa.so``. There is no CPU
fallback: importing :mod:`paper_1912_07704_b200.api` raises if the library has not been built
(``python -m paper_1912_07704_b200.build``). PyTorch is used by callers for device memory and streams only.
"""
from .api import *  # noqa: F401,F403
from .api import __all__  # noqa: F401
