"""dos -- discrete-ordinates CT dose hot path on one B200 (arXiv 1811.12391), C-ABI CUDA library + binding.

`inputs` holds the seeded synthetic workload generators (no transport arithmetic); `dos` is the ctypes
binding of csrc/libdos.so (built in-tree with nvcc for sm_100a). There is no CPU fallback.
"""
from . import inputs  # noqa: F401
from . import dos  # noqa: F401
from . import scan  # noqa: F401
