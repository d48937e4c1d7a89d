"""B200-native even-odd twisted-mass Wilson D-slash and CG (arxiv 1209.5942 hot path).

The product is the C-ABI library ``liblqcd.so`` (include/lqcd.h, csrc/*.cu).
``binding`` is a thin ctypes layer with the same function names: argument
marshalling only, every step of the path runs in the CUDA kernels.  There is no
CPU fallback: if the library is missing or was not built, importing
``binding`` raises.
"""
from . import build as _build  # noqa: F401

__all__ = ["binding", "build"]
