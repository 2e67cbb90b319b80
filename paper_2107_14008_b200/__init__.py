"""photons-b200: the truncated short-range gravity P2P operator of PhotoNs-GPU (arxiv 2107.14008) for one B200.

The product is the C-ABI CUDA library ``libphotons.so`` (``include/photons.h``); this package holds its
sources (``csrc/``), the build step (``build.py``), the ctypes binding (``binding.py``) and the seeded input
generators (``workloads.py``).  Importing the package does not load the library; ``binding.load()`` does and
raises if it has not been built.
"""
from . import workloads  # noqa: F401
