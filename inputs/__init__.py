"""Seeded synthetic inputs shared by the oracle, the tests and bench.py.

This package holds NONE of the method's arithmetic (no basis, no hops, no
Lanczos): only the lattices' bond lists, the named workload configurations of
BASELINE.json and the counter-based start-vector generator.  Both the CPU
oracle (`oracle/`) and the CUDA path (`paper_1204_3425_b200/`) are driven with
the bits produced here; neither imports the other.
"""
from .lattices import ring_bonds, torus_bonds, chain_bonds, ladder_bonds
from .vectors import g_uniform, start_vector_np, start_vector_torch, sample_indices
from .configs import CONFIGS, Config, get_config

__all__ = [
    "ring_bonds", "torus_bonds", "chain_bonds", "ladder_bonds",
    "g_uniform", "start_vector_np", "start_vector_torch", "sample_indices",
    "CONFIGS", "Config", "get_config",
]
