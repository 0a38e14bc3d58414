"""B200-native modified-Born-series solver with domain decomposition (arxiv 2410.02395).

The product is the C-ABI library `libmbs_b200.so` (include/mbs.h) built from csrc/; `binding`
is the thin ctypes layer over it and `workloads` the seeded synthetic inputs.  Nothing here
falls back to a CPU implementation: importing `binding` fails loudly if the library is missing.
"""

__all__ = ["binding", "workloads"]


def __getattr__(name):
    if name in __all__:
        import importlib
        return importlib.import_module("." + name, __name__)
    raise AttributeError(name)
