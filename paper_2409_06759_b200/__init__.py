"""paper_2409_06759_b200 -- B200-native tensor-contraction backend for generated coupled-cluster code.

The product is libtcb200.so (C ABI in include/tcb200.h, hand-written sm_100a kernels in csrc/).  This package is
the thin Python binding over it (argument marshalling only) plus the seeded input generator `synth`.
There is no CPU fallback: if the shared library is missing or no CUDA device is present, calls raise.
"""
from .binding import (Context, Tensor, TcbError, load_library, library_path, TCB_OK, TCB_EINVAL_EXPR, TCB_ESHAPE,
                      TCB_ERANK, TCB_EALIAS, TCB_ENOMEM, TCB_ECUDA, TCB_EUNSUPPORTED, TCB_EINVAL)

__all__ = ["Context", "Tensor", "TcbError", "load_library", "library_path"]
