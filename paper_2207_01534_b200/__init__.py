"""B200-native two-component pseudopotential D3Q19 lattice Boltzmann step (arXiv 2207.01534).

The product is the C-ABI library `liblbm_b200.so` (include/lbm.h, csrc/); `Lbm` is its thin
ctypes binding.  Nothing in this package imports `oracle/`.
"""
from .lbm import Lbm, LbmError, lbm_build_index, lbm_build_slab_halo, lbm_comm_unique_id, lbm_params, lbm_options, make_options, load, make_params, SYMBOLS  # noqa: F401
