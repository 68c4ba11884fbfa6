"""paper_2010_09341_b200 -- B200-native Vegas iteration + grid refinement (the VegasFlow hot path).

The product is the C-ABI shared library ``libvegas_b200.so`` (include/vegas_b200.h, sources under
``csrc/``); ``vegas`` is a thin ctypes binding with the same names, ``workloads`` the seeded
configuration tables, ``build`` the nvcc build step.  PyTorch only supplies device memory and the
stream.  There is no CPU fallback: without the built library or without a CUDA device every call fails.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "build", "vegas"]
