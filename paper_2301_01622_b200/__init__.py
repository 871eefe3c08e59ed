"""B200-native "lattice Boltzmann without populations" (arxiv 2301.01622): the fused
moments-only lattice update as hand-written sm_100a CUDA behind a C ABI (include/lbwp.h).

``lbwp``      -- ctypes binding (Lbwp, make_params, state_bytes)
``build``     -- nvcc build of liblbwp.so (in-tree)
``workloads`` -- seeded synthetic inputs of the BASELINE.json configs (no step arithmetic)
"""
from . import workloads  # noqa: F401
from .lbwp import Lbwp, LbwpError, make_params, state_bytes  # noqa: F401
