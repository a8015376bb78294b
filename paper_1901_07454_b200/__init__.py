"""arbb200 - B200-native cable-equation stepping for many multi-compartment neurons
(the data-parallel hot path of arXiv 1901.07454, "Arbor").

`workloads`  seeded synthetic inputs (no method arithmetic),
`binding`    thin ctypes layer over the C-ABI library `libarbb200.so` (include/arbb200.h).

The binding is imported lazily so that the input generators can be used without the CUDA library;
any attempt to *compute* without the built library raises.
"""
import importlib

__all__ = ["workloads", "binding"]


def __getattr__(name):
    if name in __all__:
        return importlib.import_module("." + name, __name__)
    raise AttributeError(name)
