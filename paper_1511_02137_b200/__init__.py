"""B200-native hot path of the (3+1)-D ideal relativistic hydro solver of arxiv 1511.02137.

`hydro`     -- thin ctypes binding of the C-ABI CUDA library (include/hydro.h, csrc/).
`slab`      -- z-slab decomposition over several ranks (host-side plumbing around the same library).
`synthetic` -- seeded input generators shared by the CUDA path and the CPU oracle (no method arithmetic).
"""
from . import synthetic  # noqa: F401

__all__ = ["synthetic", "hydro", "slab"]


def __getattr__(name):
    if name in ("hydro", "slab"):
        import importlib
        return importlib.import_module("." + name, __name__)
    raise AttributeError(name)
