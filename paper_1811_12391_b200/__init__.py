"""dos -- discrete-ordinates CT dose hot path on one B200 (arXiv 1811.12391), C-ABI CUDA library + binding.

`inputs` holds the seeded synthetic workload generators (no transport arithmetic) and is the only thing imported
eagerly, so that the oracle-side tests and bench.py's reference arm never map (or build) the CUDA library.
`dos` is the ctypes binding of csrc/libdos.so (built in-tree with nvcc for sm_100a) and `scan` the axial-scan host
logic on top of it; both load on first attribute access. There is no CPU fallback: without libdos.so, touching
`dos` raises.
"""
import importlib

from . import inputs  # noqa: F401

_LAZY = ("dos", "scan")


def __getattr__(name):
    if name in _LAZY:
        return importlib.import_module("." + name, __name__)
    raise AttributeError(f"module {__name__!r} has no attribute {name!r}")
