"""B200-native overlap Dirac operator hot path of arXiv 1510.06897 (Cundy & Lee, "Overlap fermions on GPUs").

Layout of the package:
  csrc/        hand-written sm_100a CUDA kernels + the extern "C" boundary (include/ovl.h)  -> libovl.so
  build.py     nvcc build of libovl.so (in-tree)
  binding.py   ctypes binding, same names as the C-ABI, argument marshalling only
  api.py       small convenience class over the binding for torch / numpy users
  inputs.py    seeded synthetic input generators (no method arithmetic; shared with the tests' oracle side)

Nothing in this package imports oracle/; there is no CPU fallback.
"""
from .binding import (  # noqa: F401
    OVL_F32, OVL_F64, OVL_RECON12, OVL_RECON18, OVL_OK, OVL_EINVAL, OVL_ENOMEM, OVL_ECUDA, OVL_ESTATE, OVL_ENOTCONV,
    OvlError,
)

__all__ = ["binding", "api", "inputs", "build"]
