"""B200-native GMMNLSE / MPA hot path (arXiv 1708.05324, §III.D).

``workloads`` (numpy-only input generators) imports nothing heavy; the CUDA
binding lives in :mod:`paper_1708_05324_b200.binding` and is imported lazily so
that the input generators stay usable on machines without the built library.
"""

__all__ = ["workloads", "binding"]


def __getattr__(name):
    if name in ("Plan", "load_library", "GmmnlseError", "plan_from_workload"):
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)
