"""pfc — B200-native energy/force/integrate hot path for an ANI-style ML
potential (the hot path behind arxiv 2412.18271's Python-force callback).

`workloads` (seeded inputs) imports without CUDA; `pfc` (the ctypes binding
of the C-ABI library built from csrc/) is imported lazily and fails loudly if
libpfc.so is missing.
"""
__all__ = ["workloads", "pfc"]


def __getattr__(name):
    if name in ("pfc", "workloads"):
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
