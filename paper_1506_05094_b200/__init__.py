"""B200-native (sm_100a) implementation of the RUMD short-range pair-interaction hot path
(arxiv 1506.05094): Verlet neighbour lists with a skin, shifted-force LJ / Coulomb pair forces with several
threads per particle, fused leap-frog NVE / Nose-Hoover NVT integration, behind the C-ABI library
``librumd_b200.so`` (``include/rumd_b200.h``).

``workloads`` (seeded synthetic inputs) is importable without the CUDA library; ``rumd`` (the ctypes binding)
loads the library on first use and fails loudly if it is missing -- there is no CPU fallback.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "rumd"]


def __getattr__(name):
    if name == "rumd":
        import importlib

        return importlib.import_module(".rumd", __name__)
    raise AttributeError(name)
