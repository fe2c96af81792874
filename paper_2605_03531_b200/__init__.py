"""B200-native brute-force incoherent dedispersion (the hot path of arxiv/paper_2605_03531).

`binding` is the thin ctypes layer over the C-ABI library libdd.so (include/dd.h);
`workloads` holds the seeded synthetic inputs; `build` compiles the CUDA sources in-tree.
"""
from . import workloads  # noqa: F401
from .build import build  # noqa: F401


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
