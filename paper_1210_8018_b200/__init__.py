"""paper_1210_8018_b200 -- B200-native SU(3) Landau gauge fixing (arXiv 1210.8018, Algorithm 1).

The product is the C-ABI library ``liblgf.so`` (include/lgf.h; hand-written sm_100a CUDA
kernels under csrc/).  ``lgf`` is its ctypes binding: argument marshalling only.  PyTorch is
used for the device workspace and the stream, nothing else.  There is no CPU fallback.
"""
from . import lgf  # noqa: F401
from .lgf import GaugeFixer, LgfError  # noqa: F401
