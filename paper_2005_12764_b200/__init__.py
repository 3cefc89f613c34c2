"""B200-native two-component colour-gradient D3Q19 lattice Boltzmann hot path (arxiv 2005.12764).

`lb`        thin ctypes binding of the C-ABI library (include/lb.h); every step runs in CUDA kernels.
`workloads` seeded synthetic inputs (no LB arithmetic).
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "lb"]


def __getattr__(name):
    if name == "lb":
        import importlib
        return importlib.import_module(__name__ + ".lb")
    raise AttributeError(name)
