"""B200-native fused multi-table embedding lookup (DPIFrame, arxiv 2606.21101, §IV-B/§IV-C).

Only the hot path lives here: the device workload planner and the fused gather-and-pool kernel, behind
the C ABI declared in ``include/dpi.h`` (built from ``csrc/``), plus a thin ctypes binding (``binding``)
and the seeded synthetic input recipe (``workloads``, no method arithmetic).

Submodules are imported lazily so that ``workloads`` can be used without the CUDA library
(the CPU oracle's tests do that); anything on the product path fails loudly if ``libdpi.so`` is absent.
"""

__all__ = ["binding", "workloads", "build"]
__version__ = "0.1.0"


def __getattr__(name):
    if name in __all__:
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
