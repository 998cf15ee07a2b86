"""paper_1908_02219_b200 — B200-native gyro-averaged charge/current deposition.

The product is the C-ABI library ``liborb_b200.so`` (``include/orb.h``, sources
under ``csrc/``); ``binding`` is the thin ctypes layer with the same names.
Importing the package does not load the library; the first call does and fails
loudly if it has not been built (there is no CPU fallback).
"""
from . import workloads  # noqa: F401  (host-side seeded inputs; no method arithmetic)

__all__ = ["workloads", "binding", "build"]


def __getattr__(name):
    if name in ("binding", "build"):
        import importlib
        return importlib.import_module("." + name, __name__)
    raise AttributeError(name)
