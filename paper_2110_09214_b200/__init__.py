"""paper_2110_09214_b200 -- B200-native (sm_100a) field-evaluation hot path of OuroborosBEM (arXiv 2110.09214).

`workloads` (seeded input generators) imports without the CUDA library.  Everything that computes
lives in libobem.so (csrc/, C-ABI in include/obem.h) and is reached through `api`; `api` raises
loudly when the library is missing -- there is no CPU fallback.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "api"]


def __getattr__(name):
    if name == "api":
        import importlib
        return importlib.import_module(".api", __name__)
    raise AttributeError(name)
