"""ikv -- IntentKV pruning + paged decode hot path, B200-native (sm_100a).

Sub-modules are imported lazily so that the seeded workload generators
(`paper_2606_09916_b200.workloads`) can be used without the CUDA library:

    from paper_2606_09916_b200 import ikv         # ctypes binding of libikv.so (fails loudly if missing)
    from paper_2606_09916_b200 import workloads   # seeded synthetic inputs
"""
import importlib

__all__ = ["ikv", "workloads", "build"]


def __getattr__(name):
    if name in __all__:
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
