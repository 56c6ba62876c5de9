"""paper_1204_4779_b200 — B200-native hot path of the Euler solver Paraiso generates (arXiv 1204.4779 §4.1).

The product is the C-ABI library `libparaiso_hydro.so` (include/paraiso_hydro.h, csrc/*.cu, sm_100a);
`binding` is a thin ctypes marshalling layer with the same names.  There is no CPU fallback: creating
a solver without the compiled library or without a CUDA device raises.

`inputs` (seeded synthetic workloads) needs neither the library nor a GPU.
"""
from . import inputs  # noqa: F401

_LAZY = ("binding", "build")


def __getattr__(name):
    if name in _LAZY:
        import importlib

        return importlib.import_module(f"{__name__}.{name}")
    if name in ("ParaisoHydro", "load_library"):
        from . import binding

        return getattr(binding, name)
    raise AttributeError(name)
