"""The five BASELINE.json configurations as seeded generators."""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Callable

import numpy as np

from .masks import all_masks, pair_masks_plus_full, sample_masks
from .tables import make_table


@dataclass
class Config:
    name: str
    n: int
    n_feat: int
    k: int
    seed: int
    join: str                      # "knn", "range" or "knn+range"
    target_neighbours: float = 0.0  # DSSJ mean neighbour count the eps_d aim for
    table: Callable[[], np.ndarray] = field(repr=False, default=None)
    masks: Callable[[], np.ndarray] = field(repr=False, default=None)


CONFIGS = {
    "c1_tiny": Config("c1_tiny", 2000, 4, 10, 0, "knn",
                      table=lambda: make_table(2000, 0, cols=[0, 1, 3, 4], outlier_frac=0.01),
                      masks=lambda: all_masks(4)),
    "c2_snapshot1_knn": Config("c2_snapshot1_knn", 31693, 15, 10, 1, "knn",
                               table=lambda: make_table(31693, 1, outlier_frac=0.01),
                               masks=lambda: all_masks(15)),
    "c3_snapshot1_dssj": Config("c3_snapshot1_dssj", 31693, 15, 0, 2, "range", 50.0,
                                table=lambda: make_table(31693, 2, outlier_frac=0.01),
                                masks=lambda: all_masks(15)),
    "c4_lsst_pairs": Config("c4_lsst_pairs", 1_000_000, 15, 10, 3, "knn",
                            table=lambda: make_table(1_000_000, 3, outlier_frac=0.001),
                            masks=lambda: pair_masks_plus_full(15)),
    "c5_lsst_oversub": Config("c5_lsst_oversub", 5_000_000, 15, 16, 4, "knn+range", 100.0,
                              table=lambda: make_table(5_000_000, 4, outlier_frac=0.001),
                              masks=lambda: sample_masks(256, 4)),
}


def get_config(name: str) -> Config:
    return CONFIGS[name]


def config_eps(name: str, masks) -> np.ndarray:
    """Per-mask radii of a DSSJ configuration from workloads/config_eps.json (written by
    `python -m oracle.write_config_eps`; inputs, like the tables): eps_d by mask dimension."""
    import json
    import os
    from .masks import popcount
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "config_eps.json")) as f:
        by_d = json.load(f)[name]["eps_by_dimension"]
    return np.array([by_d[str(int(d))] for d in popcount(masks)], dtype=np.float32)
