"""B200-native hot path of CLOSURE (arXiv 2403.09990): boundary walks, compaction, MEGB.

`instances` draws the seeded synthetic inputs; `binding` is the thin wrapper over the C ABI
(include/closure.h, libclosure_b200.so built by `build`).  Importing the package does not load
the library; the first use of `binding` does, and raises if it is missing (no CPU fallback).
"""
from . import instances  # noqa: F401

__all__ = ["instances", "binding", "build"]
