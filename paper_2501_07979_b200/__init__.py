"""B200-native differentiable cylindrical FDTD for one ZDA zone (arxiv 2501.07979).

``paper_2501_07979_b200.zda`` is the ctypes binding of ``libzda.so`` (C ABI: ``include/zda.h``).
"""
from . import zda  # noqa: F401
