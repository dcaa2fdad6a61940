"""paper_1307_0288_b200 — B200-native Chebyshev hot path of arXiv 1307.0288.

``workloads`` (seeded synthetic inputs, numpy only) imports without a GPU; the ``kg_*``
calls live in ``binding`` and need the in-tree CUDA library ``libkg.so`` (built by
``__graft_entry__.build()``); they raise if it is missing — there is no CPU fallback.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "binding"]


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
