"""zmc-b200: B200-native (sm_100a) hot path of ZMCintegral (arXiv:1902.07916).

Stratified Monte-Carlo over a grid of cells with the heuristic tree search of the paper's
section 2.1, as hand-written CUDA behind the C ABI declared in include/zmc.h. The Python layer
(`binding`) only marshals arguments; `workloads` holds the seeded synthetic problem definitions.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "binding"]


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
