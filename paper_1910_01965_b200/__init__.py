"""zmc_scan -- B200-native batched direct Monte-Carlo parameter-grid integration.

The hot path of ZMCintegral-v5 (arXiv 1910.01965): f(x) = int g(y; x) dy at every point of a
Cartesian parameter grid, as hand-written sm_100a CUDA behind a C ABI
(include/zmc.h).  `workloads` holds the seeded synthetic input generators; `binding` is the thin
ctypes face of the C ABI (imported lazily: it fails loudly when the CUDA library is missing).
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "binding"]


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
