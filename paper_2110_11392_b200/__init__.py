"""B200-native Abacus near-field force (arXiv 2110.11392, sections 3.2 + 3.4).

``NearField`` (in ``.binding``) is a thin ctypes wrapper over the C-ABI library
``libnearfield_b200.so`` declared in ``include/nearfield.h``; every step of the path runs in
the CUDA kernels under ``csrc/``.  There is no CPU fallback: touching ``NearField`` (or any
other name re-exported from ``.binding``) raises if the library has not been built.
``.workloads`` (seeded input generators, none of the method's arithmetic) imports without it.
"""
import importlib

__all__ = ["NearField", "NearFieldError", "lib_path", "load_library"]


def __getattr__(name):
    if name in __all__:
        return getattr(importlib.import_module(__name__ + ".binding"), name)
    raise AttributeError(f"module {__name__!r} has no attribute {name!r}")
