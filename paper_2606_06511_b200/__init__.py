"""B200-native (sm_100a) triangle-triangle intersection energy hot path (arXiv 2606.06511).

`inputs` (seeded synthetic workloads) is importable without the CUDA extension; the binding
(`tt`) loads `libtt.so` lazily and fails loudly when it is missing -- there is no CPU fallback.
"""
from . import inputs  # noqa: F401

__all__ = ["inputs", "tt"]


def __getattr__(name):
    if name == "tt":
        import importlib
        return importlib.import_module(".tt", __name__)
    raise AttributeError(name)
