"""B200-native batched Monte-Carlo solar-radiation-pressure force estimator (arxiv 2602.10712 hot path).

``workloads`` (numpy only) is importable anywhere.  The CUDA path is reached through
``paper_2602_10712_b200.binding`` (ctypes over the C-ABI library ``libsrp_b200.so``); it
raises if the library is not built -- there is no CPU fallback.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads"]
