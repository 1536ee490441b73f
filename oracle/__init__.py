"""CPU oracle of the two-component D3Q19 pseudopotential LBM step. TEST INFRASTRUCTURE ONLY:
importable from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference legs."""
from .lbmref import LbmRef, lattice, threads  # noqa: F401
