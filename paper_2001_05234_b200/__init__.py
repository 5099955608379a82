"""B200-native FP64 pressure-projection hot path of CaNS (arXiv 2001.05234).

The product is the C-ABI library ``libcans_poisson.so`` (see ``include/cans_poisson.h``);
``binding`` is its thin ctypes wrapper and ``workloads`` the seeded input generators.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "binding"]


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
