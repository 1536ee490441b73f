"""Seeded synthetic inputs for the two-component D3Q19 step (test/bench harness).

This module holds NO arithmetic of the method (no lattice tables, no collision,
no forces): it only produces geometry masks, initial density fields and the
parameter dictionaries of the five BASELINE.json configs. Both the oracle tests
and the CUDA path receive these arrays as plain inputs.
"""
from .generators import (  # noqa: F401
    sphere_pack_mask,
    grf_mask,
    clear_end_layers,
    tanh_profile,
    make_config,
    default_params,
    CONFIG_NAMES,
)
