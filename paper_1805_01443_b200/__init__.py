"""B200 (sm_100a) discontinuous-Galerkin Euler hot path of arXiv:1805.01443.

``DG`` is a thin ctypes binding of the C-ABI library ``libdg.so`` (``include/dg.h``): argument
marshalling only.  PyTorch provides device memory and the CUDA stream; every step of the path
runs in the library's hand-written kernels.  There is no CPU fallback.
"""
from .dg import DG, DGError, load_library  # noqa: F401
from . import workloads  # noqa: F401
