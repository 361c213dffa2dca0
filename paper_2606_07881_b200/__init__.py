"""paper_2606_07881_b200 -- B200-native PACI stage-step library (hand-written CUDA for sm_100a).

`binding` (loaded lazily so that `python -m paper_2606_07881_b200.build` can run before the shared
library exists) is the thin ctypes layer over libpaci.so; see include/paci.h for the C ABI.
"""
import importlib

__all__ = ["binding", "build"]


def __getattr__(name):
    if name in ("binding", "build"):
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
