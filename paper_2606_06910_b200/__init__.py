"""B200-native 3-D acoustic FDTD + CPML time step (arxiv/paper_2606_06910 hot path).

`binding` is the thin ctypes layer over the C-ABI library (include/fdtd_b200.h);
`inputs` holds the seeded synthetic workloads.  Nothing here falls back to a CPU
path: importing `binding` without the built CUDA library raises.
"""
from . import inputs  # noqa: F401

__all__ = ["inputs", "binding"]


def __getattr__(name):
    if name == "binding":
        import importlib

        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
