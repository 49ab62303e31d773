"""Fast-mode sea-surface radar raw-data synthesis (arxiv 2408.11472) for B200 (sm_100a).

`workloads` (seeded synthetic inputs) imports without the CUDA library; everything in `sim`
needs `csrc/libsim.so` and raises loudly if it is missing -- there is no CPU fallback.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "sim"]


def __getattr__(name):
    if name == "sim":
        import importlib
        return importlib.import_module(".sim", __name__)
    raise AttributeError(name)
