"""hepk — B200-native (sm_100a) columnar HEP analysis kernels behind a C ABI (include/hepk.h).

The product is csrc/libhepk.so; `binding` is a thin ctypes layer over it (torch for device memory and
streams only).  There is no CPU fallback: importing works without a GPU, calling anything does not.
"""
from . import binding  # noqa: F401

__all__ = ["binding"]
