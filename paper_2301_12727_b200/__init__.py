"""B200-native 3-D staggered-grid viscoelastic FDTD time step (arXiv 2301.12727, section 2.3).

The product is the C-ABI library ``libbvfdtd.so`` (``include/bvfdtd.h``; CUDA kernels for sm_100a
under ``csrc/``); ``binding`` is its thin ctypes front end and ``workloads`` the seeded synthetic
input generator (inputs only, none of the method's arithmetic).  There is no CPU fallback.
"""
from . import workloads  # noqa: F401
from . import binding  # noqa: F401  (loads the shared library lazily, on first use)
from .binding import Simulation  # noqa: F401
