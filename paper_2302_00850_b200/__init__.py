"""B200-native hot path of the COLA inverter (arxiv 2302.00850): Wilson-clover fermion matrix,
even-odd Schur complement and the CGNR solver it drives, as hand-written sm_100a CUDA kernels behind
a C ABI (include/cola.h).  `inputs` (seeded synthetic fields) is importable without the CUDA
library; everything else loads libcola.so and fails loudly if it is missing.
"""
import importlib

_LAZY = {"binding", "build"}


def __getattr__(name):
    if name in _LAZY:
        return importlib.import_module(f"{__name__}.{name}")
    if name in ("Cola", "ColaError", "lib_path"):
        return getattr(importlib.import_module(f"{__name__}.binding"), name)
    raise AttributeError(name)
