"""B200-native nodal finite-difference LLG right-hand side (arxiv 2411.11725 hot path).

The product is the C-ABI library `libnm.so` (sources in `csrc/`, header `include/nm.h`);
`binding` is the thin ctypes layer with the same names.  `workloads` holds the seeded input
generators and is importable without the CUDA library.
"""

__all__ = ["binding", "workloads"]


def __getattr__(name):
    if name in __all__:
        import importlib
        return importlib.import_module("." + name, __name__)
    raise AttributeError(name)
