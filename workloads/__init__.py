"""Seeded synthetic inputs shared by tests, bench.py, the oracle and the CUDA path.

This package holds NO arithmetic of the SNAPS method (no distances, joins or
scores): only random feature tables, subspace-mask lists and the five
BASELINE.json configurations.  Recipe: DESIGN.md "Input recipe".
"""
from .tables import make_table, hypercube_table, duplicate_block_table, lattice_table, COLUMN_NAMES
from .masks import all_masks, pair_masks_plus_full, sample_masks, popcount
from .configs import CONFIGS, get_config, config_eps

__all__ = [
    "make_table", "hypercube_table", "duplicate_block_table", "lattice_table",
    "COLUMN_NAMES", "all_masks", "pair_masks_plus_full", "sample_masks",
    "popcount", "CONFIGS", "get_config", "config_eps",
]
