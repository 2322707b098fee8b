"""kratos-hydro-b200: B200-native hot path of the Kratos hydrodynamics module (arXiv 2501.02317).

The product is the C-ABI library ``libkratos_hydro.so`` (see ``include/kratos_hydro.h``)
built from ``csrc/``; ``binding`` is the thin ctypes front end with the same names.
Sub-modules are imported lazily: ``inputs`` (seeded synthetic states) needs neither the
CUDA library nor a GPU.
"""
from __future__ import annotations

import importlib

__all__ = ["binding", "build", "inputs", "KratosHydro"]


def __getattr__(name):
    if name in ("binding", "build", "inputs"):
        return importlib.import_module(f"{__name__}.{name}")
    if name == "KratosHydro":
        return importlib.import_module(f"{__name__}.binding").KratosHydro
    raise AttributeError(name)
